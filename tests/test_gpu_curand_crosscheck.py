"""-m gpu: pins of the ORACLE against cuRAND's own device code (toolkit headers), for the two recurrences whose
constants PAPER.md does not print (XORWOW: Ref.[30], reading R-B1; Philox4x32-10: Ref.[20], reading R-C1).
The helper tests/curand_crosscheck.cu is compiled here with nvcc; it is test infrastructure, never on the hot
path, and shares nothing with the product or the oracle."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def cc():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    src, so = os.path.join(HERE, "curand_crosscheck.cu"), os.path.join(HERE, "_curand_crosscheck.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "--shared", "-Xcompiler", "-fPIC",
                        "--extended-lambda", "-o", so, src], check=True)
    L = C.CDLL(so)
    L.cc_xorwow.restype = C.c_int
    L.cc_xorwow.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]
    L.cc_philox.restype = C.c_int
    L.cc_philox.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p]
    return L


def test_oracle_xorwow_is_curands_xorwow(cc):
    rng = np.random.default_rng(1)
    n, draws = 300, 40
    st = rng.integers(0, 2**32, size=(n, 6), dtype=np.uint32)
    st[0] = (123456789, 362436069, 521288629, 88675123, 5783321, 6615241)   # Marsaglia's default state
    st[1] = (1, 0, 0, 0, 0, 0)
    out = np.empty((n, draws), dtype=np.uint32)
    assert cc.cc_xorwow(st.ctypes.data, n, draws, out.ctypes.data) == 0
    for i in range(n):
        s = st[i].copy()
        assert [oracle.xorwow_next(s) for _ in range(draws)] == [int(v) for v in out[i]], i


def test_oracle_philox_is_curands_philox4x32_10(cc):
    rng = np.random.default_rng(2)
    n = 2000
    ck = rng.integers(0, 2**32, size=(n, 6), dtype=np.uint32)
    ck[0] = 0
    ck[1] = 0xFFFFFFFF
    ck[2] = (5, 1, 0, 0, 9, 0)                    # the stream mapping's counter shape (lo, hi, 0, 0)
    out = np.empty((n, 4), dtype=np.uint32)
    assert cc.cc_philox(ck.ctypes.data, n, out.ctypes.data) == 0
    for i in range(n):
        o = oracle.philox4x32([int(v) for v in ck[i, :4]], [int(v) for v in ck[i, 4:]])
        assert [int(v) for v in o] == [int(v) for v in out[i]], i
