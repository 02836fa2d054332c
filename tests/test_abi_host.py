"""-m "not gpu": the C-ABI library builds, loads, and exports every symbol
include/rng_b200.h declares; host-side logic (argument checks, the acceptance
table, state sizes); and the product path FAILS LOUDLY without a CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1204_6193_b200 as pkg
from paper_1204_6193_b200 import build as pkg_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    pkg_build.build()
    return pkg.lib()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "rng_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)  # strip comments
    names = re.findall(r"\b((?:rng|ising)_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_boundary_of_north_star():
    names = _declared_functions()
    for must in ("rng_create", "rng_fill_u32", "rng_fill_f32", "rng_draw_reduce", "ising_sweep"):
        assert must in names


def test_library_exports_every_declared_symbol(L):
    names = _declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/rng_b200.h but not exported"
    # and the binding covers exactly the header
    assert sorted(pkg.EXPORTS) == names


def test_no_torch_types_or_cpp_in_header():
    src = open(os.path.join(ROOT, "include", "rng_b200.h")).read()
    assert 'extern "C"' in src
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    assert "torch" not in code.lower() and "at::" not in code and "std::" not in code
    assert "#include <stdint.h>" in code and code.count("#include") == 1


def test_version_and_counters(L):
    assert pkg.rng_version().startswith("rng_b200") and "sm_100a" in pkg.rng_version()
    assert pkg.rng_kernel_launches() >= 0


def test_state_bytes(L):
    assert pkg.rng_state_bytes(pkg.RNG_LCG64, 1024) == 8 * 1024
    assert pkg.rng_state_bytes(pkg.RNG_LCG64_LEAPFROG, 7) == 56
    assert pkg.rng_state_bytes(pkg.RNG_XORWOW, 1 << 22) == 24 << 22  # "192 bits" PAPER.md:266
    assert pkg.rng_state_bytes(pkg.RNG_PHILOX4X32_10, 1 << 20) == 0   # no stored state
    assert pkg.rng_state_bytes(pkg.RNG_XS1024W, 1 << 24) == 4 << 24   # "32 bits/thread" PAPER.md:268
    assert pkg.rng_state_bytes(pkg.RNG_PHILOX4X32_7, 1 << 20) == 0
    assert pkg.rng_state_bytes(pkg.RNG_LCG32, 1000) == 4000            # "32 bits" PAPER.md:262 (Table 2)
    assert pkg.rng_state_bytes(pkg.RNG_XS1024W_SKIP, 64) == 256
    assert pkg.rng_state_bytes(pkg.RNG_LCG64_BOTH, 3) == 24
    assert pkg.rng_state_bytes(pkg.RNG_LFIB521, 512) == 2 * 521 * 4    # one ring of r words per 256 streams
    assert pkg.rng_state_bytes(pkg.RNG_LFIB1279, 256) == 1279 * 4
    assert pkg.rng_state_bytes(pkg.RNG_LCG32_LEAPFROG, 10) == 40
    assert pkg.rng_state_bytes(pkg.RNG_MWC, 10) == 80                  # 64 bits: (x, c)
    assert pkg.rng_state_bytes(pkg.RNG_MWC_MULTI, 10) == 120           # "64+32 = 96 bits"
    assert pkg.rng_state_bytes(99, 5) == 0


def test_invalid_arguments_are_rejected_before_any_cuda_call(L):
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_create(99, 16, 1)
    assert e.value.code == pkg.RNG_E_INVAL
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_create(pkg.RNG_LCG64, 0, 1)
    assert e.value.code == pkg.RNG_E_INVAL
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_create(pkg.RNG_XS1024W, 100, 1)  # not whole 32-lane instances
    assert e.value.code == pkg.RNG_E_INVAL and "32" in str(e.value)
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_create_shard(pkg.RNG_XORWOW, 10, 8, 4, 1)  # [8,12) not inside [0,10)
    assert e.value.code == pkg.RNG_E_INVAL
    assert L.rng_create(pkg.RNG_LCG64, 4, 1, None) == pkg.RNG_E_INVAL
    # NULL handles
    assert L.rng_fill_u32(None, None, 4, None) == pkg.RNG_E_INVAL
    assert L.rng_draw_reduce(None, None, 4, None) == pkg.RNG_E_INVAL
    assert L.ising_sweep(None, None, 4, 0.3, 1, None, None) == pkg.RNG_E_INVAL
    assert L.rng_get_state(None, None, 0) == pkg.RNG_E_INVAL
    assert L.rng_destroy(None) == pkg.RNG_OK
    assert pkg.rng_draws_done(None) == 0


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


@pytest.mark.skipif(_has_gpu(), reason="only meaningful on a box without a CUDA device")
def test_no_cpu_fallback_without_a_device(L):
    """north_star: 'no CPU fallback'.  On the CPU-only box a valid create must fail
    with RNG_E_CUDA, not silently compute somewhere else."""
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_create(pkg.RNG_PHILOX4X32_10, 1024, 1)
    assert e.value.code == pkg.RNG_E_CUDA
    assert "no CUDA device" in str(e.value) or "CUDA" in str(e.value)


def test_product_never_imports_the_oracle():
    """The oracle is test infrastructure: nothing under paper_1204_6193_b200/ or include/
    may import, include or link it (and vice versa)."""
    bad = []
    for base in ("paper_1204_6193_b200", "include"):
        for dp, _, fs in os.walk(os.path.join(ROOT, base)):
            if os.path.basename(dp) in ("build", "__pycache__"):
                continue
            for f in fs:
                if not f.endswith((".py", ".cu", ".cuh", ".h", ".cpp", ".c")):
                    continue
                txt = open(os.path.join(dp, f)).read()
                if re.search(r"^\s*(import|from)\s+oracle\b", txt, re.M) or re.search(r'#include\s*[<"].*oracle', txt) \
                        or "liboracle" in txt or "orc_" in txt:
                    bad.append(os.path.join(dp, f))
    assert not bad, bad
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1204_6193_b200", txt, re.M)
            assert "rng_b200.h" not in txt and "librng_b200" not in txt


def test_accept_table_integer_form_is_exactly_the_float_compare(L):
    """ising_accept_table: T[i] = min(2^24, ceil(P[i] 2^24)) makes (r>>8) < T[i] the same
    decision as (float)(r>>8)*2^-24 < P[i] (R-E3, both sides decide in f32).  Exhaustive
    around every threshold, random elsewhere; P itself must equal the oracle's table bit
    for bit (R-E4: both evaluate exp() in double on the same host)."""
    import oracle
    rs = np.random.RandomState(5)
    for beta in (0.0, 0.1, 0.3, 0.4, 0.44068679350977147, 1.0, 5.0, -0.2):
        P, T = pkg.ising_accept_table(beta)
        P = np.array(P, dtype=np.float32)
        Po = oracle.ising_accept_table(beta)
        assert P.tobytes() == Po.tobytes()
        for i in range(5):
            t = T[i]
            assert 0 <= t <= 1 << 24
            cand = np.unique(np.clip(np.concatenate([
                np.arange(t - 3, t + 4), [0, 1, (1 << 24) - 1], rs.randint(0, 1 << 24, 2000)]), 0, (1 << 24) - 1))
            u = cand.astype(np.float32) * np.float32(2.0 ** -24)
            assert np.array_equal(u < P[i], cand < t), (beta, i)
