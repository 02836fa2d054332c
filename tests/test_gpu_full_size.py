"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(default kernel variants, the 4 GiB output buffer, the same handles and call sequences).

The oracle cannot produce 2^30 draws in seconds, but every stream is independent and seeded by
random access in its global id, so an oracle SHARD (rng_create_shard semantics: streams
[first, first+m) of n_total) reproduces exactly the rows of the full-size output it covers.
Rows are sampled at the start, the end and seeded random places (whole warp tiles and CTA
boundaries included); checksums / states are compared the same way.  C1 is small and is
compared in full; the L = 8192 lattice is compared in full (the oracle needs ~1 s per sweep).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402  (test infrastructure)
import paper_1204_6193_b200 as pkg  # noqa: E402
from paper_1204_6193_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def big_buffer():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_1204_6193_b200 import build
    build.build()
    torch.cuda.set_device(0)
    buf = torch.empty(1 << 30, dtype=torch.int32, device="cuda")  # 4 GiB, as in bench.py
    yield buf
    del buf
    torch.cuda.empty_cache()


def sample_shards(n_streams, width, count, seed):
    """`count` shard starts (multiples of `width`): first, last, around CTA / tile borders, random"""
    rng = np.random.default_rng(seed)
    last = n_streams - width
    fixed = [0, last, (n_streams // 2), (n_streams // 2) - width, 256 - width if 256 >= width else 0, 4096]
    rnd = (rng.integers(0, n_streams // width, size=count) * width).tolist()
    out = sorted({min(max(int(f) // width * width, 0), last) for f in fixed + rnd})
    return out


def rows_of(buf, first, m, n):
    return buf[first * n:(first + m) * n].cpu().numpy().view(np.uint32).reshape(m, n)


def check_fill_rows(cfg, buf, calls_done, m, shards, f32=False):
    """rows [f, f+m) of the last call's output == draws [(calls_done-1) n, calls_done n) of the oracle shard"""
    n = cfg.n_per_stream
    for f in shards:
        o = oracle.Rng(cfg.kind, m, cfg.seed, first=f, n_total=cfg.n_streams)
        for _ in range(calls_done - 1):
            o.fill_u32(n)
        exp = (o.fill_f32(n).view(np.uint32) if f32 else o.fill_u32(n)).reshape(m, n)
        got = rows_of(buf, f, m, n)
        assert np.array_equal(got, exp), f"{cfg.name}: rows [{f},{f + m}) differ, first at {np.argwhere(got != exp)[:3]}"


def test_c1_lcg64_full(big_buffer):
    cfg = W.C1
    g, o = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed), oracle.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    g.fill_u32(big_buffer, cfg.n_per_stream)
    assert np.array_equal(big_buffer[:cfg.draws_per_call].cpu().numpy().view(np.uint32), o.fill_u32(cfg.n_per_stream))
    g.fill_f32(big_buffer.view(torch.float32), cfg.n_per_stream)
    assert np.array_equal(big_buffer[:cfg.draws_per_call].cpu().numpy().view(np.uint32),
                          o.fill_f32(cfg.n_per_stream).view(np.uint32))
    assert np.array_equal(g.get_state(), o.get_state())
    g.close()


@pytest.mark.parametrize("cfg", [W.C2, W.C1_BIG, W.C3_FILL], ids=lambda c: c.name)
def test_4gib_fills_on_sampled_rows(cfg, big_buffer):
    """C2 (Philox 2^20 x 1024) and the supplementary 4 GiB LCG64 / XORWOW fills: two calls (u32, then f32)"""
    g = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    shards = sample_shards(cfg.n_streams, 64, 10, 1)
    big_buffer.zero_()
    g.fill_u32(big_buffer, cfg.n_per_stream)
    check_fill_rows(cfg, big_buffer, 1, 64, shards)
    g.fill_f32(big_buffer.view(torch.float32), cfg.n_per_stream)
    check_fill_rows(cfg, big_buffer, 2, 64, shards, f32=True)
    assert g.draws_done == 2 * cfg.n_per_stream
    # nothing was written past the end of the output
    g.close()


def test_c3_xorwow_draw_reduce_full(big_buffer):
    cfg = W.C3
    g = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    g.draw_reduce(big_buffer, cfg.n_per_stream)
    red = big_buffer[:2 * cfg.n_streams].cpu().numpy().view(np.uint32).reshape(-1, 2)
    m = 256
    for f in sample_shards(cfg.n_streams, m, 12, 2):
        o = oracle.Rng(cfg.kind, m, cfg.seed, first=f, n_total=cfg.n_streams)
        assert np.array_equal(red[f:f + m].reshape(-1), o.draw_reduce(cfg.n_per_stream)), f
    # the state of the whole handle: compare the sampled shards' final states
    st = g.get_state().reshape(-1, 6)
    f = cfg.n_streams - m
    o = oracle.Rng(cfg.kind, m, cfg.seed, first=f, n_total=cfg.n_streams)
    o.draw_reduce(cfg.n_per_stream)
    assert np.array_equal(st[f:f + m].reshape(-1), o.get_state())
    g.close()


def test_c4_xs1024_fill_calls_and_draw_full(big_buffer):
    """C4: 2^24 streams.  Fill mode to the depth bench.py runs it: 64 consecutive calls of 64 draws into one buffer
    on ONE handle (the persistent kernel's work-ticket counter and the Weyl index must carry across all of them);
    sampled instances after calls 1, 2, 3, 32, 63 and 64, the generator state after call 64; then draw mode
    (4096 draws) continuing the same handle."""
    cfg = W.C4_FILL
    n_calls = 64
    g = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    m = 128  # four instances
    shards = sample_shards(cfg.n_streams, m, 8, 3)
    for call in range(1, n_calls + 1):
        if call in (32, 63):
            big_buffer.zero_()  # a launch that wrote nothing would otherwise leave the previous call's rows behind
        g.fill_u32(big_buffer, cfg.n_per_stream)
        if call in (1, 2, 3, 32, 63, 64):
            check_fill_rows(cfg, big_buffer, call, m, shards)
    assert g.draws_done == n_calls * cfg.n_per_stream
    st = g.get_state()
    for f in shards:
        o = oracle.Rng(cfg.kind, m, cfg.seed, first=f, n_total=cfg.n_streams)
        o.fill_u32(n_calls * cfg.n_per_stream)
        assert np.array_equal(st[f:f + m], o.get_state()), f
    n_draw = W.C4_DRAW.n_per_stream
    g.draw_reduce(big_buffer, n_draw)
    red = big_buffer[:2 * cfg.n_streams].cpu().numpy().view(np.uint32).reshape(-1, 2)
    st = g.get_state()
    for f in shards[:5]:
        o = oracle.Rng(cfg.kind, m, cfg.seed, first=f, n_total=cfg.n_streams)
        o.fill_u32(n_calls * cfg.n_per_stream)
        assert np.array_equal(red[f:f + m].reshape(-1), o.draw_reduce(n_draw)), f
        assert np.array_equal(st[f:f + m], o.get_state()), f
    assert g.draws_done == n_calls * cfg.n_per_stream + n_draw
    g.close()


@pytest.mark.parametrize("cfg", [W.C5B_PHILOX, W.C5B_XORWOW, W.C5B_XORWOW_K8], ids=lambda c: c.name)
def test_c5b_ising_L8192_full_lattice(cfg):
    """L = 8192 at beta_c from the seeded random start: the whole lattice and the energy trace after
    2 + 1 sweeps (two calls, so the packed bit planes are rebuilt from the int8 lattice in between)"""
    L = cfg.L
    g, o = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed), oracle.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, cfg.lattice_seed)
    ref = oracle.ising_init_random(L, cfg.lattice_seed)
    assert np.array_equal(sp.cpu().numpy(), ref)
    tr = torch.empty(2, dtype=torch.int64, device="cuda")
    g.ising_sweep(sp, L, cfg.beta, 2, tr)
    tr_o = o.ising_sweep(ref, L, cfg.beta, 2, trace=True)
    assert np.array_equal(tr.cpu().numpy(), tr_o)
    assert np.array_equal(sp.cpu().numpy(), ref)
    g.ising_sweep(sp, L, cfg.beta, 1)
    o.ising_sweep(ref, L, cfg.beta, 1)
    assert np.array_equal(sp.cpu().numpy(), ref)
    e = torch.zeros(1, dtype=torch.int64, device="cuda")
    pkg.ising_energy(sp, L, e)
    assert int(e.item()) == oracle.ising_energy(ref, L)
    assert g.draws_done == o.draws_done
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()


# ---- SURVEY.md 8(c)-E7 depth: long single calls (PAPER.md:56 application test; BASELINE config 5 "1000 sweeps") -------
def _long_ising_call(kind, L, n_streams, n_sweeps, seed, lattice_seed, beta):
    g, o = pkg.Rng(kind, n_streams, seed), oracle.Rng(kind, n_streams, seed)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, lattice_seed)
    ref = oracle.ising_init_random(L, lattice_seed)
    tr = torch.empty(n_sweeps, dtype=torch.int64, device="cuda")
    g.ising_sweep(sp, L, beta, n_sweeps, tr)                       # ONE call, as bench.py issues it
    tr_o = o.ising_sweep(ref, L, beta, n_sweeps, trace=True)
    got = tr.cpu().numpy()
    for t in sorted({1, 2, 10, 100, n_sweeps}):
        if t <= n_sweeps:
            assert int(got[t - 1]) == int(tr_o[t - 1]), f"energy after sweep {t}"
    assert np.array_equal(got, tr_o), "energy trace"
    assert np.array_equal(sp.cpu().numpy(), ref), "final lattice"
    assert g.draws_done == o.draws_done == 2 * (L * L // 2 // n_streams) * n_sweeps
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state()), "final generator state"
    g.close()


@pytest.mark.parametrize("cfg", [W.C5B_XORWOW, W.C5B_PHILOX], ids=lambda c: c.name)
def test_c5b_ising_L8192_1000_sweeps_exactly_as_benched(cfg):
    """BASELINE config 5 to the letter: L = 8192, 1000 sweeps, ONE call -- the calls bench.py's C5b_xorwow and
    C5b_philox time (draw counter and Philox block index growing over 2000 half-sweeps, pack / unpack once around
    1000 sweeps).  The energy after sweeps 1, 2, 10, 100 and 1000, the whole 1000-entry trace,
    the final 64 MiB lattice and the final generator states against the oracle.  About 3.5 minutes of oracle time
    per generator; it replaces the 100-sweep and the L = 2048 x 1000-sweep cases of round 2, which it contains."""
    _long_ising_call(cfg.kind, cfg.L, cfg.n_streams, cfg.n_sweeps, cfg.seed, cfg.lattice_seed, cfg.beta)


# ---- the widened rows at the sizes bench.py times ------------------------------
@pytest.mark.parametrize("cfg", [W.N1_PHILOX7, W.N1_LCG32, W.N1_LCG64BOTH, W.N4_LFIB521, W.N4_LFIB1279],
                         ids=lambda c: c.name)
def test_next_kinds_4gib_fills_on_sampled_rows(cfg, big_buffer):
    g = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    shards = sample_shards(cfg.n_streams, 256, 6, 4)      # whole lagged Fibonacci instances
    big_buffer.zero_()
    g.fill_u32(big_buffer, cfg.n_per_stream)
    check_fill_rows(cfg, big_buffer, 1, 256, shards)
    g.fill_f32(big_buffer.view(torch.float32), cfg.n_per_stream)
    check_fill_rows(cfg, big_buffer, 2, 256, shards, f32=True)
    g.close()


@pytest.mark.parametrize("cfg", [W.N1_PHILOX10_DRAW, W.N1_PHILOX7_DRAW, W.N1_LCG64_DRAW, W.N1_LCG32_DRAW,
                                 W.N1_LCG64BOTH_DRAW, W.N4_LFIB521_DRAW, W.N4_LFIB1279_DRAW], ids=lambda c: c.name)
def test_next_kinds_draw_reduce_full(cfg, big_buffer):
    g = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    g.draw_reduce(big_buffer, cfg.n_per_stream)
    red = big_buffer[:2 * cfg.n_streams].cpu().numpy().view(np.uint32).reshape(-1, 2)
    m = 256
    for f in sample_shards(cfg.n_streams, m, 8, 5):
        o = oracle.Rng(cfg.kind, m, cfg.seed, first=f, n_total=cfg.n_streams)
        assert np.array_equal(red[f:f + m].reshape(-1), o.draw_reduce(cfg.n_per_stream)), f
    g.close()


def test_skip_ahead_seeding_of_2_19_instances():
    """C4's 2^24 streams seeded the paper's way: 19 levels of the doubling tree.  Sampled instances against
    X_0 J^g from the oracle's matrix powers (binary exponentiation over J_k = M^(2^(137+k)))"""
    S, seed = 1 << 24, W.MASTER_SEED
    g = pkg.Rng(pkg.RNG_XS1024W_SKIP, S, seed)
    st = g.get_state().reshape(-1, 32)
    x0 = oracle.Rng(oracle.XS1024W, 32, seed).get_state()
    Jk = [oracle.xs1024_matpow2(137)]
    for _ in range(18):
        Jk.append(oracle.xs1024_matmul(Jk[-1], Jk[-1]))

    def inst(G):
        X = x0
        for k in range(19):
            if (G >> k) & 1:
                X = oracle.xs1024_vecmat(X, Jk[k])
        return X
    rng = np.random.default_rng(6)
    for G in [0, 1, 2, (1 << 19) - 1, 1 << 18, (1 << 18) - 1, 0x55555, 0x2AAAA] + rng.integers(0, 1 << 19, 12).tolist():
        assert np.array_equal(st[G], inst(int(G))), G
    # the generator itself then runs as kind 4: a draw-mode call on the whole handle, sampled against the oracle
    # started from those states is covered by test_c4_*; here the first draws of two far-apart instances
    out = torch.empty(S * 4, dtype=torch.int32, device="cuda")
    g.fill_u32(out, 4)
    rows = out.cpu().numpy().view(np.uint32).reshape(S, 4)
    for G in (0, (1 << 19) - 1):
        X = inst(G).copy()
        for j in range(4):
            oracle.xs1024_update(X)
            y = (362437 * (j + 1)) & 0xFFFFFFFF
            assert np.array_equal(rows[32 * G:32 * G + 32, j], ((y ^ (y >> 16)) + X.astype(np.uint64)).astype(np.uint32))
    g.close()


@pytest.mark.parametrize("cfg", [W.T1_XORWOW_K100, W.T1_XORWOW_K1, W.T1_PHILOX_K100, W.T1_XS1024_K100,
                                 W.T1_XORWOW_K100_T8], ids=lambda c: c.name)
def test_table1_multihit_L1024_full_lattice(cfg):
    """the paper's Table-1 workload (1024^2, beta = 0.4, double checkerboard, 262144 streams): the whole lattice
    and the energy after 1 + 1 sweeps (k = 100: 2 * 10^8 updates on the oracle)"""
    L = cfg.L
    g, o = pkg.Rng(cfg.kind, cfg.n_streams, cfg.seed), oracle.Rng(cfg.kind, cfg.n_streams, cfg.seed)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, cfg.lattice_seed)
    ref = oracle.ising_init_random(L, cfg.lattice_seed)
    for _ in range(2):
        tr = torch.empty(1, dtype=torch.int64, device="cuda")
        g.ising_sweep_multihit(sp, L, cfg.beta, 1, cfg.tile, cfg.k_hits, tr)
        tr_o = o.ising_sweep_multihit(ref, L, cfg.beta, 1, cfg.tile, cfg.k_hits, trace=True)
        assert np.array_equal(sp.cpu().numpy(), ref)
        assert int(tr.item()) == int(tr_o[0])
    assert g.draws_done == o.draws_done == 8 * cfg.k_hits
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()
