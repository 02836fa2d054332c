"""ising_sweep_philox_static: the Ising sweep for callers that cannot allocate device memory.

Who needs it: a program that shares the GPU with a framework whose caching allocator already owns the memory, a
loop that cannot afford the device-wide synchronisation of cudaMalloc/cudaFree, a process with a memory budget
fixed at start-up.  `ising_sweep` shuts them out (its handle and its bit planes come from cudaMalloc), so the
library keeps 2 MiB of bit planes inside its own image and offers this one handle-free entry point on top of it
(include/rng_b200.h; L <= RNG_ISING_STATIC_MAX_L = 4096).

What is checked here: the new entry point leaves the same lattice and the same energy trace, bit for bit, as the
existing `ising_sweep` on an RNG_PHILOX4X32_10 handle -- on two calls in a row, the second continuing the first,
with lattices of different sizes sharing the one scratch array one after the other (so each call meets whatever
the previous one left there).  The existing path is itself compared with the CPU oracle in test_gpu_parity.py;
the small cases repeat that comparison directly.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

import paper_1204_6193_b200 as pkg

BETA_C = 0.44068679350977147


def test_static_sweep_refuses_what_its_scratch_cannot_hold():
    """Argument checks come before any CUDA call, so they run without a GPU: a lattice beyond the built-in scratch
    is refused with a message that names the limit -- it is never served by allocating."""
    from paper_1204_6193_b200 import build
    build.build()
    assert pkg.RNG_ISING_STATIC_MAX_L == 4096
    fake = 1 << 20  # an aligned non-NULL address; the call must fail before it could touch it
    for L, S, draws, beta, code, word in [
        (8192, 8192 * 8192 // 8, 0, BETA_C, pkg.RNG_E_INVAL, "4096"),      # beyond the maximum
        (4160, 4160 * 4160 // 8, 0, BETA_C, pkg.RNG_E_INVAL, "4096"),      # just beyond it
        (96, 96 * 96 // 8, 0, BETA_C, pkg.RNG_E_INVAL, "multiple of 64"),
        (128, 1000, 0, BETA_C, pkg.RNG_E_INVAL, "divide"),
        (128, 128 * 128 // 4, 0, BETA_C, pkg.RNG_E_INVAL, "K ="),          # K = 2 has no multi-spin kernel
        (128, 128 * 128 // 8, 2, BETA_C, pkg.RNG_E_INVAL, "multiple of 4"),
        (128, 128 * 128 // 8, 0, -0.1, pkg.RNG_E_INVAL, "beta"),
        (128, 128 * 128 // 8, 0, float("nan"), pkg.RNG_E_INVAL, "beta"),
    ]:
        with pytest.raises(pkg.RngError) as e:
            pkg.ising_sweep_philox_static(S, 1, draws, fake, L, beta, 1)
        assert e.value.code == code and word in str(e.value), (L, S, str(e.value))
    with pytest.raises(pkg.RngError):
        pkg.ising_sweep_philox_static(128 * 128 // 8, 1, 0, None, 128, BETA_C, 1)  # NULL lattice
    with pytest.raises(pkg.RngError):
        pkg.ising_sweep_philox_static(128 * 128 // 8, 1, 0, fake + 4, 128, BETA_C, 1)  # misaligned lattice


@pytest.mark.gpu
def test_static_sweep_equals_ising_sweep_on_two_calls_in_a_row():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_1204_6193_b200 import build
    build.build()
    import oracle  # test infrastructure: the direct comparison of the small cases

    torch.cuda.set_device(0)
    # (L, n_streams, seed): the largest lattice the scratch holds comes first, so that the smaller ones that follow
    # find the array full of another lattice's planes; K = 4 and 16 take the word kernels, K = 32 and 64 the stream kernel
    cases = [(4096, 4096 * 4096 // 8, 5), (256, 256 * 256 // 8, 1), (128, 128 * 128 // 64, 7), (64, 64 * 64 // 32, 3),
             (192, 192 * 192 // 128, 11)]
    for L, S, seed in cases:
        K = L * L // 2 // S
        g = pkg.Rng(pkg.RNG_PHILOX4X32_10, S, seed)           # the existing path
        sp_a = torch.empty(L * L, dtype=torch.int8, device="cuda")
        pkg.ising_init_random(sp_a, L, seed + 100)
        sp_b = sp_a.clone()
        tr_a = torch.zeros(5, dtype=torch.int64, device="cuda")
        tr_b = torch.full((5,), -1, dtype=torch.int64, device="cuda")
        small = L <= 256
        if small:
            o = oracle.Rng(pkg.RNG_PHILOX4X32_10, S, seed)
            ref = oracle.ising_init_random(L, seed + 100)

        # call 1: three sweeps from fresh streams
        g.ising_sweep(sp_a, L, BETA_C, 3, tr_a[:3])
        pkg.ising_sweep_philox_static(S, seed, 0, sp_b, L, BETA_C, 3, tr_b[:3])
        torch.cuda.synchronize()
        assert torch.equal(sp_a, sp_b), f"L={L} K={K}: lattices differ after the first call"
        assert torch.equal(tr_a[:3], tr_b[:3])
        d = 3 * 2 * K
        assert g.draws_done == d

        # call 2: two more sweeps, the caller carrying the stream position; device memory in use must not move
        free_before = torch.cuda.mem_get_info()[0]
        pkg.ising_sweep_philox_static(S, seed, d, sp_b, L, BETA_C, 2, tr_b[3:])
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info()[0]
        g.ising_sweep(sp_a, L, BETA_C, 2, tr_a[3:])
        torch.cuda.synchronize()
        assert free_after == free_before, "the static entry point changed the amount of free device memory"
        assert torch.equal(sp_a, sp_b), f"L={L} K={K}: lattices differ after the second call"
        assert torch.equal(tr_a, tr_b)
        assert abs(int(tr_b[-1].item())) <= 2 * L * L and int(sp_b.abs().min().item()) == 1

        if small:
            tr_o = o.ising_sweep(ref, L, BETA_C, 5, trace=True)
            assert np.array_equal(sp_b.cpu().numpy(), ref)
            assert np.array_equal(tr_b.cpu().numpy(), tr_o)
        g.close()

    # the trace is optional, and a call with nothing to do is a no-op that touches nothing
    L, S = 128, 128 * 128 // 8
    g = pkg.Rng(pkg.RNG_PHILOX4X32_10, S, 9)
    sp_a = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp_a, L, 4)
    sp_b = sp_a.clone()
    pkg.ising_sweep_philox_static(S, 9, 0, sp_b, L, 0.3, 0)
    assert torch.equal(sp_a, sp_b)
    g.ising_sweep(sp_a, L, 0.3, 4)
    pkg.ising_sweep_philox_static(S, 9, 0, sp_b, L, 0.3, 4)
    torch.cuda.synchronize()
    assert torch.equal(sp_a, sp_b)
    g.close()
