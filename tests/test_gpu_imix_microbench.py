"""-m gpu: the issue rate of the instruction mix of the Philox K = 4 Ising half-sweep, measured.

DESIGN 6.6 bounds that kernel at about 1320 flips/ns from a model of the SM's issue slots.  This test runs
tests/imix_microbench.cu -- the same mix per 32 sites (137 IMAD.WIDE, 160 LOP3, 64 two-instruction carry chains,
72 additions) with no loads, stores or update logic -- and prints the rate the hardware sustains for it, so that
the bound is a measurement.  Test infrastructure only: nothing here is on the product path."""
import ctypes as C
import os
import subprocess

import pytest

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))


def test_issue_rate_of_the_philox_ising_instruction_mix():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    src, so = os.path.join(HERE, "imix_microbench.cu"), os.path.join(HERE, "_imix_microbench.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "--shared", "-Xcompiler", "-fPIC",
                        "-o", so, src], check=True)
    L = C.CDLL(so)
    L.imix_run.restype = C.c_float
    L.imix_run.argtypes = [C.c_uint32, C.c_uint32, C.c_int]
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    best = {}
    for ctas_per_sm in (4, 8, 16):
        blocks, iters = sms * ctas_per_sm, 1000
        ms = L.imix_run(blocks, iters, 5)
        assert ms > 0, "micro-benchmark kernel failed"
        sites = blocks * 128 * iters * 32
        best[ctas_per_sm] = sites / (ms * 1e6)  # sites per ns = the 'flips/ns' this mix could feed
    print("\nimix micro-benchmark (sites/ns by CTAs of 128 threads per SM): " +
          ", ".join(f"{k}: {v:.0f}" for k, v in best.items()))
    assert 300 < max(best.values()) < 10000
