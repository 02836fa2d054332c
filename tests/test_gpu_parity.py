"""-m gpu: parity tests proper.  The CUDA path, called through the C-ABI, against the
CPU oracle, element by element, on the same seeds.  Bar: BIT-EXACT for every integer
stream, every float conversion (compared as bit patterns), every checksum, every
generator state and every spin configuration (north_star)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402  (test infrastructure)
import paper_1204_6193_b200 as pkg  # noqa: E402

KINDS = list(pkg.KIND_NAMES)
IDS = [pkg.KIND_NAMES[k] for k in KINDS]
XS_KINDS = (pkg.RNG_XS1024W, pkg.RNG_XS1024W_SKIP)
LFIB_KINDS = (pkg.RNG_LFIB521, pkg.RNG_LFIB1279)  # one ring buffer per 256 streams


@pytest.fixture(scope="module", autouse=True)
def _device():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_1204_6193_b200 import build
    build.build()
    torch.cuda.set_device(0)
    yield
    torch.cuda.synchronize()


def dev_u32(n):
    return torch.empty(max(n, 4), dtype=torch.int32, device="cuda")


def host(t, n, dtype=np.uint32):
    return t.cpu().numpy().view(dtype)[:n]


def n_streams_for(kind, S):
    if kind in LFIB_KINDS:
        return max(256, S - S % 256)
    return S - S % 32 if kind in XS_KINDS else S


# ---------------------------------------------------------------------------------
# bounds: compute-sanitizer is closed on the GPU pool (profiles/r03_sanitizer.txt), so out-of-bounds
# stores are looked for with guard bands of our own around every buffer a kernel writes
# ---------------------------------------------------------------------------------
GUARD = 4096  # words on either side
PATTERN = 0x5A5A5A5A


def guarded(n_words):
    """a device buffer of n_words int32 with GUARD pattern words before and after it -> (whole, view)"""
    whole = torch.full((n_words + 2 * GUARD,), PATTERN, dtype=torch.int32, device="cuda")
    return whole, whole[GUARD:GUARD + n_words]


def assert_guards_intact(whole, n_words, what):
    lo, hi = whole[:GUARD], whole[GUARD + n_words:]
    assert bool((lo == PATTERN).all()) and bool((hi == PATTERN).all()), f"{what}: a store landed outside the output"


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_no_store_outside_the_output_buffers(kind):
    """fill (u32 and f32), draw_reduce and the Ising sweeps write only inside the caller's buffers: guard bands
    of 16 KiB on both sides of each output stay untouched, for stream counts and row lengths that end inside a
    warp tile, inside a 128-bit store and inside a TMA box"""
    for S0, n in ((1000, 7), (4136, 64), (2080, 100), (992, 257), (33, 1028)):
        S = n_streams_for(kind, S0)
        g, o = pkg.Rng(kind, S, 5), oracle.Rng(kind, S, 5)
        whole, out = guarded(S * n)
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n))
        assert_guards_intact(whole, S * n, f"fill_u32 S={S} n={n}")
        whole, out = guarded(S * n)
        g.fill_f32(out.view(torch.float32), n)
        assert np.array_equal(host(out, S * n), o.fill_f32(n).view(np.uint32))
        assert_guards_intact(whole, S * n, f"fill_f32 S={S} n={n}")
        whole, red = guarded(2 * S)
        g.draw_reduce(red, n)
        assert np.array_equal(host(red, 2 * S), o.draw_reduce(n))
        assert_guards_intact(whole, 2 * S, f"draw_reduce S={S} n={n}")
        g.close()
    # the consumer: lattice (int8, viewed inside an int32 guard buffer) and the energy trace (int64)
    for L, Sx, sweeps in ((64, 256, 3), (128, 2048, 2), (48, 96, 2)):
        S = n_streams_for(kind, Sx)
        if (L * L // 2) % S:
            continue
        g, o = pkg.Rng(kind, S, 5), oracle.Rng(kind, S, 5)
        whole, w = guarded(L * L // 4)
        sp = w.view(torch.int8)
        pkg.ising_init_random(sp, L, 3)
        ref = oracle.ising_init_random(L, 3)
        twhole, tw = guarded(2 * sweeps)
        tr = tw.view(torch.int64)
        g.ising_sweep(sp, L, 0.44, sweeps, tr)
        tr_o = o.ising_sweep(ref, L, 0.44, sweeps, trace=True)
        assert np.array_equal(sp.cpu().numpy(), ref) and np.array_equal(tr.cpu().numpy(), tr_o)
        assert_guards_intact(whole, L * L // 4, f"ising_sweep L={L}")
        assert_guards_intact(twhole, 2 * sweeps, f"ising_sweep trace L={L}")
        g.close()


# ---------------------------------------------------------------------------------
# fill: several warp tiles + ragged tail in both directions (S not a multiple of 32 /
# of the CTA size, n not a multiple of 4 / of the 32-draw tile), continuation.
# ---------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("S,ns", [(1000, (100, 37, 4, 1, 0, 64)), (33, (3, 129)), (1, (17, 16)), (4096 + 40, (32,))])
def test_fill_u32_and_continuation(kind, S, ns):
    S = n_streams_for(kind, S)
    if S == 0:
        S = 32
    g, o = pkg.Rng(kind, S, 1), oracle.Rng(kind, S, 1)
    for n in ns:
        out = dev_u32(S * n)
        g.fill_u32(out, n)
        exp = o.fill_u32(n)
        got = host(out, S * n)
        assert np.array_equal(got, exp), f"{pkg.KIND_NAMES[kind]} S={S} n={n}: first diff at {np.flatnonzero(got != exp)[:5]}"
        assert g.draws_done == o.draws_done
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_fill_f32_bit_patterns(kind):
    S = n_streams_for(kind, 777)
    g, o = pkg.Rng(kind, S, 12345), oracle.Rng(kind, S, 12345)
    for n in (64, 13):
        out = torch.empty(S * n, dtype=torch.float32, device="cuda")
        g.fill_f32(out, n)
        exp = o.fill_f32(n)
        got = out.cpu().numpy()
        assert np.array_equal(got.view(np.uint32), exp.view(np.uint32))
        assert got.min() >= 0.0 and got.max() <= 1.0 - 2.0 ** -24
    g.close()


def test_f32_map_exact_for_every_24_bit_value():
    """The library evaluates (u >> 8) 2^-24 by reading u >> 8 as a (denormal) float and multiplying by 2^125
    (generators.cuh).  Every one of the 2^24 values of u >> 8, each with a different low byte, goes through the
    fill kernel: an LCG32 stream's first draw is its state word, and rng_set_state chooses the states.  Compared
    with the oracle's map applied to the same words and with the definition evaluated by numpy."""
    S = 1 << 24
    u = (np.arange(S, dtype=np.uint32) << np.uint32(8)) | ((np.arange(S, dtype=np.uint32) * np.uint32(167)) & np.uint32(255))
    g = pkg.Rng(pkg.RNG_LCG32, S, 1)
    g.set_state(u)
    out = torch.empty(S, dtype=torch.float32, device="cuda")
    g.fill_f32(out, 1)
    got = out.cpu().numpy()
    g.close()
    exp = (u >> np.uint32(8)).astype(np.float32) * np.float32(2.0 ** -24)  # exact: 24-bit integer, power of two
    assert np.array_equal(got.view(np.uint32), exp.view(np.uint32)), np.flatnonzero(got != exp)[:8]
    for i in (0, 1, 255, 256, (1 << 23) - 1, 1 << 23, (1 << 23) + 1, S - 1, 0x5A5A5A, 0x123456):
        assert float(got[i]) == oracle.u32_to_f32(int(u[i])), i


@pytest.mark.parametrize("kind", [pkg.RNG_PHILOX4X32_10, pkg.RNG_PHILOX4X32_7], ids=["philox10", "philox7"])
@pytest.mark.parametrize("cvt", [0, 1, 2, 3], ids=["denormal_scale", "i2fp", "prmt_ffma", "i2f_xu"])
def test_philox_f32_conversion_forms_are_the_same_map(kind, cvt):
    """variant "cvt": four exact evaluations of (u >> 8) 2^-24 in the Philox fill kernel; every one against the
    oracle, on full tiles (the lean all-full path), on a ragged last tile and across a continuation"""
    S = 67
    g, o = pkg.Rng(kind, S, 2024), oracle.Rng(kind, S, 2024)
    g.set_variant("cvt", cvt)
    for n in (1024, 2048 + 512, 36):
        out = torch.empty(S * n, dtype=torch.float32, device="cuda")
        g.fill_f32(out, n)
        exp = o.fill_f32(n)
        assert np.array_equal(out.cpu().numpy().view(np.uint32), exp.view(np.uint32)), (cvt, n)
    g.close()


@pytest.mark.parametrize("kind", [pkg.RNG_PHILOX4X32_10, pkg.RNG_PHILOX4X32_7], ids=["philox10", "philox7"])
@pytest.mark.parametrize("store", [1, 2, 3, 4], ids=["U4T2", "U2T4", "one_shot_ctas", "persistent_grid"])
def test_philox_fill_grid_and_tile_variants(kind, store):
    """variant "store" of the Philox fill: blocks per lane x groups per tile, and who hands out the tiles (a
    persistent grid striding over them, or one short-lived CTA per 8 tiles); full tiles, more tiles than one wave
    of CTAs, a ragged last tile, continuation, u32 and f32 -- all against the oracle"""
    S = 3000  # x 3 tiles per row for n = 3072: 9000 tiles = 1125 one-shot CTAs
    g, o = pkg.Rng(kind, S, 31), oracle.Rng(kind, S, 31)
    g.set_variant("store", store)
    for n in (3072, 1024, 520):
        out = dev_u32(S * n)
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n)), (store, n)
        outf = torch.empty(S * n, dtype=torch.float32, device="cuda")
        g.fill_f32(outf, n)
        assert np.array_equal(outf.cpu().numpy().view(np.uint32), o.fill_f32(n).view(np.uint32)), (store, n)
    g.close()


@pytest.mark.parametrize("kind", LFIB_KINDS, ids=["lfib521", "lfib1279"])
@pytest.mark.parametrize("store", [1, 2], ids=["tile32", "tile64"])
def test_lfib_fill_tiles_ring_is_the_staging_buffer(kind, store):
    """the lagged Fibonacci fill keeps 32 or 64 batches in its ring and writes rows out of it (lfib.cu): whole
    tiles, several tiles, a ragged last tile, rows that are not 16-byte aligned, continuation across calls (the
    state is reloaded into the last slots), u32 and f32, and the state at the end -- all against the oracle"""
    S = 512
    g, o = pkg.Rng(kind, S, 77), oracle.Rng(kind, S, 77)
    g.set_variant("store", store)
    for n in (64, 200, 32, 7, 1, 130, 3):
        out = dev_u32(S * n)
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n)), (store, n)
        outf = torch.empty(max(S * n, 4), dtype=torch.float32, device="cuda")
        g.fill_f32(outf, n)
        assert np.array_equal(outf.cpu().numpy().view(np.uint32)[:S * n], o.fill_f32(n).view(np.uint32)), (store, n)
        assert np.array_equal(g.get_state(), o.get_state()), (store, n)
    g.close()


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_mixed_call_sequence_is_one_stream(kind):
    """fill_u32(n1), draw_reduce(n2), fill_f32(n3) continue the same streams (state
    persists in the handle): compare against one oracle fill of n1+n2+n3."""
    S = n_streams_for(kind, 300)
    n1, n2, n3 = 7, 50, 9
    g, o = pkg.Rng(kind, S, 99), oracle.Rng(kind, S, 99)
    ref = o.fill_u32(n1 + n2 + n3).reshape(S, -1)
    a = dev_u32(S * n1)
    g.fill_u32(a, n1)
    r = dev_u32(2 * S)
    g.draw_reduce(r, n2)
    f = torch.empty(S * n3, dtype=torch.float32, device="cuda")
    g.fill_f32(f, n3)
    assert np.array_equal(host(a, S * n1).reshape(S, n1), ref[:, :n1])
    mid = ref[:, n1:n1 + n2]
    red = host(r, 2 * S).reshape(S, 2)
    assert np.array_equal(red[:, 0], np.bitwise_xor.reduce(mid, axis=1))
    assert np.array_equal(red[:, 1], mid.sum(axis=1, dtype=np.uint64).astype(np.uint32))
    expf = (ref[:, n1 + n2:] >> 8).astype(np.float32) * np.float32(2.0 ** -24)
    assert np.array_equal(f.cpu().numpy().reshape(S, n3), expf)
    g.close()


# ---------------------------------------------------------------------------------
# draw_reduce
# ---------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("S,ns", [(2048 + 96, (256, 1, 0, 3, 1001)), (32, (5,))])
def test_draw_reduce(kind, S, ns):
    S = n_streams_for(kind, S)
    g, o = pkg.Rng(kind, S, 7), oracle.Rng(kind, S, 7)
    for n in ns:
        out = dev_u32(2 * S)
        g.draw_reduce(out, n)
        assert np.array_equal(host(out, 2 * S), o.draw_reduce(n)), (pkg.KIND_NAMES[kind], S, n)
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()


@pytest.mark.parametrize("kind", [pkg.RNG_LCG64, pkg.RNG_LCG64_LEAPFROG], ids=["lcg64", "lcg64_leapfrog"])
@pytest.mark.parametrize("variant", [1, 2], ids=["thread_per_stream", "cta_per_stream"])
def test_lcg_intra_stream_skip_ahead_is_the_same_stream(kind, variant):
    """eq.(2) applied inside a stream (one CTA per stream, lanes leap by step^1024) gives the bits of
    the sequential walk: u32, f32, ragged and unaligned n, continuation, final state"""
    S = 37
    g, o = pkg.Rng(kind, S, 5), oracle.Rng(kind, S, 5)
    g.set_variant("lcg", variant)
    for n in (4096, 1024, 1, 3, 1030, 2047, 0, 512):
        out = dev_u32(S * n)
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n)), (variant, n)
        assert np.array_equal(g.get_state(), o.get_state()), (variant, n)
    outf = torch.empty(S * 1500, dtype=torch.float32, device="cuda")
    g.fill_f32(outf, 1500)
    assert np.array_equal(outf.cpu().numpy().view(np.uint32), o.fill_f32(1500).view(np.uint32))
    assert np.array_equal(g.get_state(), o.get_state())
    g.close()


@pytest.mark.parametrize("store", [0, 1], ids=["tma_tensor_store", "lds_stg"])
@pytest.mark.parametrize("K", [1, 2, 4, 8, 16, 32, 64])
def test_xs1024_lane_layouts_are_one_generator(K, store):
    """the paper's generator with K words per lane (K = 1: Listing 1's one word per thread, shuffles;
    K = 32: whole instance in one thread; 64: the generic row-tile / per-stream kernels): identical
    fill (u32, f32, ragged n, unaligned rows), draw_reduce and final state"""
    for S in (32, 32 * 37, 32 * 256 + 32 * 5):
        g, o = pkg.Rng(pkg.RNG_XS1024W, S, 11), oracle.Rng(pkg.RNG_XS1024W, S, 11)
        g.set_variant("xs1024", K)
        g.set_variant("store", store)
        for n in (64, 32, 5, 100, 1, 36, 128):
            out = dev_u32(S * n)
            g.fill_u32(out, n)
            assert np.array_equal(host(out, S * n), o.fill_u32(n)), (K, S, n)
        outf = torch.empty(S * 40, dtype=torch.float32, device="cuda")
        g.fill_f32(outf, 40)
        assert np.array_equal(outf.cpu().numpy().view(np.uint32), o.fill_f32(40).view(np.uint32))
        for n in (257, 3, 0):
            red = dev_u32(2 * S + 4)
            g.draw_reduce(red, n)
            assert np.array_equal(host(red, 2 * S), o.draw_reduce(n)), (K, S, n)
        # 8-byte (not 16-byte) aligned checksum buffer is allowed by the API
        pkg.rng_draw_reduce(g.handle, red.data_ptr() + 8, 9)
        assert np.array_equal(host(red, 2 * S + 2)[2:], o.draw_reduce(9))
        assert g.draws_done == o.draws_done
        assert np.array_equal(g.get_state(), o.get_state())
        g.close()


def test_xs1024_shared_memory_exchange_is_the_same_generator():
    """the paper's Listing 1 with __syncwarp (variant "xs1024" = 33, draw mode): same checksums and final state as the
    oracle, i.e. as the shuffle layouts; several CTAs, a ragged last CTA, continuation across calls and variants"""
    for kind in XS_KINDS:
        S = 32 * 37
        g, o = pkg.Rng(kind, S, 4), oracle.Rng(kind, S, 4)
        g.set_variant("xs1024", 33)
        red = dev_u32(2 * S)
        for n in (1, 100, 257):
            g.draw_reduce(red, n)
            assert np.array_equal(host(red, 2 * S), o.draw_reduce(n)), n
        assert np.array_equal(g.get_state(), o.get_state())
        g.set_variant("xs1024", 1)          # the shuffle form of the same layout continues the same streams
        g.draw_reduce(red, 64)
        assert np.array_equal(host(red, 2 * S), o.draw_reduce(64))
        g.close()


@pytest.mark.parametrize("xsfill", [0, 1, 2, 3], ids=["by_row_length", "one_shot_ctas", "tickets_1_tile", "tickets_2_tiles"])
@pytest.mark.parametrize("K", [1, 2, 4, 8, 16])
def test_xs1024_fill_schedules_are_one_generator(K, xsfill):
    """the TMA fill path of the paper's generator under every work distribution (one short-lived CTA per item;
    persistent warps drawing items from the handle's ticket counter, one or two tiles per warp): more items than
    resident warps (so that warps loop and prefetch the next item's state), a ragged last item, several calls on
    one handle (the ticket base carries over), rows of 32 k and of 4 k' draws, u32 and f32"""
    resident_warps = 148 * {1: 32, 2: 28, 4: 14, 8: 7, 16: 3}[K]  # the most any variant keeps on a B200
    S = 32 * K * (2 * resident_warps + 3) + 32 * (K // 2 + 1)      # a warp hosts K instances; last item ragged
    g, o = pkg.Rng(pkg.RNG_XS1024W, S, 21), oracle.Rng(pkg.RNG_XS1024W, S, 21)
    g.set_variant("xs1024", K)
    g.set_variant("xsfill", xsfill)
    out = dev_u32(S * 64)
    for n in (64, 36, 64, 4):
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n)), (K, xsfill, n)
    outf = out.view(torch.float32)
    g.fill_f32(outf, 32)
    assert np.array_equal(host(out, S * 32), o.fill_f32(32).view(np.uint32))
    assert g.draws_done == o.draws_done
    assert np.array_equal(g.get_state(), o.get_state())
    g.close()


def test_xs1024_fill_long_rows_take_the_ping_pong_tiles():
    """n >= 2048 selects two tiles per warp; a few instances, long ragged rows"""
    S, n = 32 * 9, 2048 + 36
    g, o = pkg.Rng(pkg.RNG_XS1024W, S, 5), oracle.Rng(pkg.RNG_XS1024W, S, 5)
    out = dev_u32(S * n)
    for _ in range(2):
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n))
    assert np.array_equal(g.get_state(), o.get_state())
    g.close()


# ---------------------------------------------------------------------------------
# seeding / sharding: a shard [first, first+n_local) of n_total reproduces those rows
# ---------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_shard_equals_rows_of_the_whole(kind):
    n_total, first, n_local, n = (1280, 256, 512, 20) if kind in LFIB_KINDS else (640, 256, 160, 20)
    whole = oracle.Rng(kind, n_total, 3).fill_u32(n).reshape(n_total, n)
    g = pkg.Rng(kind, n_local, 3, first=first, n_total=n_total)
    if g.state_bytes():
        o = oracle.Rng(kind, n_local, 3, first=first, n_total=n_total)
        assert np.array_equal(g.get_state(), o.get_state()), "seed kernel state != oracle seeding"
    out = dev_u32(n_local * n)
    g.fill_u32(out, n)
    assert np.array_equal(host(out, n_local * n).reshape(n_local, n), whole[first:first + n_local])
    g.close()


def test_lcg_leapfrog_is_one_global_sequence():
    """all streams generate numbers out of the same global sequence (1)."""
    S, n = 96, 50
    g = pkg.Rng(pkg.RNG_LCG64_LEAPFROG, S, 1)
    out = dev_u32(S * n)
    g.fill_u32(out, n)
    got = host(out, S * n).reshape(S, n)
    x = oracle.splitmix64(1, 0)
    seq = []
    for _ in range(S * n):
        seq.append(x >> 32)
        x = oracle.lcg64_step(x)
    assert np.array_equal(got.T.reshape(-1), np.array(seq, dtype=np.uint32))
    g.close()


def test_set_state_roundtrip_and_hand_traced_states():
    """rng_set_state with the hand-traceable states of tests/golden: XORWOW from
    (1,0,0,0,0,0) gives 0x587c8 first (R-B1); xs1024 from X0 = 1 (word 31) gives lane
    31 = 0x587c1, lane 0 = 0x587c0 (R-D5/D6)."""
    g = pkg.Rng(pkg.RNG_XORWOW, 2, 1)
    st = np.array([1, 0, 0, 0, 0, 0, 123456789, 362436069, 521288629, 88675123, 5783321, 6615241], dtype=np.uint32)
    g.set_state(st)
    assert np.array_equal(g.get_state(), st)
    out = dev_u32(2 * 8)
    g.fill_u32(out, 8)
    got = host(out, 16).reshape(2, 8)
    assert list(got[0]) == [0x587c8, 0xb0fbd, 0x109a52, 0x165247, 0x1ea6dc, 0x542ed4, 0x329b97a, 0x335f744a]
    assert list(got[1][:5]) == [246875399, 3690007200, 1264581005, 3906711041, 1866187943]
    g.close()
    g = pkg.Rng(pkg.RNG_XS1024W, 32, 1)
    X = np.zeros(32, dtype=np.uint32)
    X[31] = 1
    g.set_state(X)
    out = dev_u32(32 * 2)
    g.fill_u32(out, 2)
    got = host(out, 64).reshape(32, 2)
    assert got[31, 0] == 0x587c1 and got[0, 0] == 0x587c0
    assert got[31, 1] == 0xb0f82 and got[0, 1] == 0xb1001
    g.close()


# ---------------------------------------------------------------------------------
# error behaviour on a live handle
# ---------------------------------------------------------------------------------
def test_argument_errors_on_a_live_handle():
    g = pkg.Rng(pkg.RNG_PHILOX4X32_10, 64, 1)
    buf = dev_u32(64 * 8 + 4)
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_fill_u32(g.handle, buf.data_ptr() + 4, 8)  # misaligned
    assert e.value.code == pkg.RNG_E_INVAL
    with pytest.raises(pkg.RngError) as e:
        pkg.rng_fill_u32(g.handle, None, 8)
    assert e.value.code == pkg.RNG_E_INVAL
    sp = torch.zeros(36, dtype=torch.int8, device="cuda")
    with pytest.raises(pkg.RngError):  # 64 streams do not divide 6*6/2
        g.ising_sweep(sp, 6, 0.3, 1)
    with pytest.raises(pkg.RngError):  # odd L
        g.ising_sweep(sp, 5, 0.3, 1)
    assert g.draws_done == 0
    g.close()


# ---------------------------------------------------------------------------------
# Ising consumer
# ---------------------------------------------------------------------------------
def test_ising_init_and_energy():
    for L in (4, 6, 64, 130):
        sp = torch.empty(L * L + 16, dtype=torch.int8, device="cuda")
        pkg.ising_init_random(sp, L, 2)
        ref = oracle.ising_init_random(L, 2)
        assert np.array_equal(sp.cpu().numpy()[:L * L], ref)
        e = torch.zeros(1, dtype=torch.int64, device="cuda")
        pkg.ising_energy(sp, L, e)
        assert int(e.item()) == oracle.ising_energy(ref, L)


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("L,S,sweeps", [(4, 8, 50), (4, 1, 20), (6, 6, 10), (64, 256, 12), (64, 2048, 6),
                                        (128, 32, 4), (256, 4096, 5), (512, 16384, 3), (48, 96, 5), (64, 512, 4),
                                        (1024, 1024, 2)])
def test_ising_sweep_bit_exact(kind, L, S, sweeps):
    if (kind in XS_KINDS and S % 32) or (kind in LFIB_KINDS and S % 256):
        pytest.skip("xs1024 needs whole 32-stream instances")
    beta = 0.3 if L == 4 else 0.44068679350977147
    g, o = pkg.Rng(kind, S, 1), oracle.Rng(kind, S, 1)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 2)
    ref = oracle.ising_init_random(L, 2)
    tr = torch.empty(sweeps, dtype=torch.int64, device="cuda")
    g.ising_sweep(sp, L, beta, sweeps, tr)
    tr_o = o.ising_sweep(ref, L, beta, sweeps, trace=True)
    assert np.array_equal(sp.cpu().numpy(), ref), f"lattice differs at {np.flatnonzero(sp.cpu().numpy() != ref)[:8]}"
    assert np.array_equal(tr.cpu().numpy(), tr_o)
    assert g.draws_done == o.draws_done == sweeps * L * L // S
    # a second call continues both the lattice and the streams
    g.ising_sweep(sp, L, beta, 3)
    o.ising_sweep(ref, L, beta, 3)
    assert np.array_equal(sp.cpu().numpy(), ref)
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()


@pytest.mark.parametrize("variant", [0, 1, 2, 3], ids=["auto", "generic", "bytes", "multispin"])
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("L,S,sweeps", [(64, 64, 5), (128, 32, 4), (256, 4096, 4), (64, 512, 4), (128, 512, 3),
                                        (192, 576, 3), (512, 16384, 2), (1024, 1024, 2)])
def test_ising_kernel_variants_share_one_trajectory(kind, L, S, sweeps, variant):
    """every kernel variant (generic byte kernel, 16-byte chunk kernel, multi-spin bit planes in
    STREAM and WORD mode) reproduces the oracle's lattice, energy trace and generator state"""
    if (kind in XS_KINDS and S % 32) or (kind in LFIB_KINDS and S % 256):
        pytest.skip("xs1024 needs whole 32-stream instances")
    beta = 0.44068679350977147
    g, o = pkg.Rng(kind, S, 1), oracle.Rng(kind, S, 1)
    g.set_variant("ising", variant)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 2)
    ref = oracle.ising_init_random(L, 2)
    tr = torch.empty(sweeps, dtype=torch.int64, device="cuda")
    g.ising_sweep(sp, L, beta, sweeps, tr)
    tr_o = o.ising_sweep(ref, L, beta, sweeps, trace=True)
    assert np.array_equal(sp.cpu().numpy(), ref), f"lattice differs at {np.flatnonzero(sp.cpu().numpy() != ref)[:8]}"
    assert np.array_equal(tr.cpu().numpy(), tr_o)
    # misalign the draw counter (Philox must leave its whole-block fast paths), then continue without a trace
    red = dev_u32(2 * S)
    g.draw_reduce(red, 3)
    o.draw_reduce(3)
    g.ising_sweep(sp, L, beta, 2)
    o.ising_sweep(ref, L, beta, 2)
    assert np.array_equal(sp.cpu().numpy(), ref)
    assert g.draws_done == o.draws_done
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()


@pytest.mark.parametrize("beta", [0.0, 0.3, 1.5, 20.0, -0.2])
def test_ising_variants_at_other_temperatures(beta):
    """beta = 0 (every move accepted), large beta (thresholds down to T = 0 ... never accepted) and
    beta < 0 (table shape the fast paths do not cover): all fall back correctly"""
    L, S, sweeps = 128, 1024, 3
    for kind in (pkg.RNG_PHILOX4X32_10, pkg.RNG_XORWOW):
        for variant in (0, 2, 3):
            g, o = pkg.Rng(kind, S, 7), oracle.Rng(kind, S, 7)
            g.set_variant("ising", variant)
            sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
            pkg.ising_init_random(sp, L, 3)
            ref = oracle.ising_init_random(L, 3)
            g.ising_sweep(sp, L, beta, sweeps)
            o.ising_sweep(ref, L, beta, sweeps)
            assert np.array_equal(sp.cpu().numpy(), ref), (beta, kind, variant)
            g.close()


def test_ising_equals_fill_then_apply():
    """ising_sweep consumes exactly the draws rng_fill_u32 would have produced
    (include/rng_b200.h: 'fill K draws per stream, then apply')."""
    L, S = 32, 64
    K = L * L // 2 // S
    g1, g2 = pkg.Rng(pkg.RNG_XORWOW, S, 5), pkg.Rng(pkg.RNG_XORWOW, S, 5)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 9)
    g1.ising_sweep(sp, L, 0.4, 2)
    buf = dev_u32(S * 4 * K)
    g2.fill_u32(buf, 4 * K)
    assert np.array_equal(g1.get_state(), g2.get_state())
    g1.close()
    g2.close()


@pytest.mark.slow
def test_ising_L4_monte_carlo_energy_within_3_sigma(golden):
    """C5a: L=4, beta=0.3; <E>/N from the GPU trajectory agrees with the exact
    enumeration of all 2^16 states (tests/golden/ising_L4.txt) within 3 sigma
    (binning error), for Philox and XORWOW."""
    exact = float(golden("ising_L4.txt")["e"][0])
    L, S, therm, sweeps = 4, 8, 1000, 200000
    for kind in (pkg.RNG_PHILOX4X32_10, pkg.RNG_XORWOW):
        g = pkg.Rng(kind, S, 1)
        sp = torch.empty(16, dtype=torch.int8, device="cuda")
        pkg.ising_init_random(sp, L, 2)
        g.ising_sweep(sp, L, 0.3, therm)
        tr = torch.empty(sweeps, dtype=torch.int64, device="cuda")
        g.ising_sweep(sp, L, 0.3, sweeps, tr)
        e = tr.cpu().numpy().astype(np.float64) / 16.0
        nb = 100
        bins = e[: (len(e) // nb) * nb].reshape(nb, -1).mean(axis=1)
        sigma = bins.std(ddof=1) / np.sqrt(nb)
        assert abs(e.mean() - exact) < 3 * sigma, (pkg.KIND_NAMES[kind], e.mean(), exact, sigma)
        assert sigma < 5e-3
        g.close()


# ---------------------------------------------------------------------------------
# host-buffer entry points (the e2e path bench.py times)
# ---------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
def test_host_entry_points(kind):
    S, n = 512, 40
    g, o = pkg.Rng(kind, S, 1), oracle.Rng(kind, S, 1)
    a = np.empty(S * n, dtype=np.uint32)
    g.fill_u32_host(a, n)
    assert np.array_equal(a, o.fill_u32(n))
    f = np.empty(S * n, dtype=np.float32)
    g.fill_f32_host(f, n)
    assert np.array_equal(f.view(np.uint32), o.fill_f32(n).view(np.uint32))
    r = np.empty(2 * S, dtype=np.uint32)
    g.draw_reduce_host(r, 33)
    assert np.array_equal(r, o.draw_reduce(33))
    g.close()
    L, S = 64, (256 if kind in LFIB_KINDS else 128)
    g, o = pkg.Rng(kind, S, 1), oracle.Rng(kind, S, 1)
    sp = oracle.ising_init_random(L, 2)
    ref = sp.copy()
    tr = np.empty(4, dtype=np.int64)
    g.ising_sweep_host(sp, L, 0.4, 4, tr)
    tr_o = o.ising_sweep(ref, L, 0.4, 4, trace=True)
    assert np.array_equal(sp, ref) and np.array_equal(tr, tr_o)
    g.close()


# ---------------------------------------------------------------------------------
# the paper's application test (Table 1), scaled down: 1024 x 1024, beta = 0.4,
# internal energy and specific heat against the exact finite-lattice result
# ---------------------------------------------------------------------------------
def _table1_run(kind, S, seed=1, L=1024, beta=0.4, therm=3000, sweeps=200000, nb=100):
    """-> (e, err_e, C_V, err_CV) from `sweeps` sweeps after `therm` discarded; e = -E/N; errors from nb bins
    (e: spread of bin means; C_V = beta^2 N (<e^2> - <e>^2): jackknife over bins)"""
    g = pkg.Rng(kind, S, seed)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, seed + 100)
    g.ising_sweep(sp, L, beta, therm)
    tr = torch.empty(sweeps, dtype=torch.int64, device="cuda")
    g.ising_sweep(sp, L, beta, sweeps, tr)
    g.close()
    N = L * L
    e = -tr.cpu().numpy().astype(np.float64) / N
    bins = e.reshape(nb, -1)
    e_err = bins.mean(axis=1).std(ddof=1) / np.sqrt(nb)
    tot1, tot2 = e.sum(), (e * e).sum()
    b1, b2, m = bins.sum(axis=1), (bins * bins).sum(axis=1), sweeps - bins.shape[1]
    jk = beta * beta * N * ((tot2 - b2) / m - ((tot1 - b1) / m) ** 2)
    cv = beta * beta * N * (tot2 / sweeps - (tot1 / sweeps) ** 2)
    cv_err = np.sqrt((nb - 1) / nb * ((jk - jk.mean()) ** 2).sum())
    return e.mean(), e_err, cv, cv_err


@pytest.mark.slow
@pytest.mark.parametrize("kind,S", [(pkg.RNG_PHILOX4X32_10, 1 << 17), (pkg.RNG_XORWOW, 1 << 11),
                                    (pkg.RNG_XS1024W, 1 << 14), (pkg.RNG_LCG64, 1 << 16), (pkg.RNG_MWC, 1 << 16),
                                    (pkg.RNG_LFIB1279, 1 << 14), (pkg.RNG_MWC_MULTI, 1 << 16),
                                    (pkg.RNG_PHILOX4X32_7, 1 << 17)],
                         ids=["philox_K4", "xorwow_K256", "xs1024_K32", "lcg64_random_K8", "mwc_same_a_K8", "lfib1279_K32",
                              "mwc_different_a_K8", "philox7_K4"])
def test_table1_L1024_beta04_energy_and_specific_heat_within_3_sigma(kind, S):
    """The paper's application test (Table 1), scaled to 2*10^5 sweeps (2*10^11 updates):
    e and C_V of the 1024^2 lattice at beta = 0.4 agree with Kaufman's exact values (which reproduce the
    paper's printed 1.106079207 / 0.8616983594; tests/test_oracle_ising_stats.py) within
    3 sigma for Philox4x32-10, XORWOW, the paper's XORShift1024/Weyl and the randomly seeded LCG64."""
    from exact_ising import kaufman
    exact = kaufman(1024, 0.4)
    e, e_err, cv, cv_err = _table1_run(kind, S)
    print(f"\n{pkg.KIND_NAMES[kind]}: e = {e:.7f} +- {e_err:.7f} (exact {-exact['e']:.7f}, "
          f"{(e + exact['e']) / e_err:+.2f} sigma), C_V = {cv:.5f} +- {cv_err:.5f} (exact {exact['cv']:.5f}, "
          f"{(cv - exact['cv']) / cv_err:+.2f} sigma)")
    assert abs(e - (-exact["e"])) < 3 * e_err, (pkg.KIND_NAMES[kind], e, -exact["e"], e_err)
    assert abs(cv - exact["cv"]) < 3 * cv_err, (pkg.KIND_NAMES[kind], cv, exact["cv"], cv_err)
    assert e_err < 5e-5 and cv_err < 0.02


@pytest.mark.slow
def test_table1_lcg64_substreams_fail_like_in_the_paper():
    """PAPER.md:82 (Table 1, row 'LCG64'): with sub-streams of ONE 64-bit LCG sequence (skip-ahead /
    leapfrog) the checkerboard simulation gives a significantly wrong internal energy
    (13.7 sigma too high at the paper's precision), while random seeding passes.  The same happens here:
    e comes out too high by far more than 10 sigma."""
    from exact_ising import kaufman
    exact = kaufman(1024, 0.4)
    e, e_err, _, _ = _table1_run(pkg.RNG_LCG64_LEAPFROG, 1 << 16, sweeps=50000, nb=50)
    print(f"\nlcg64_leapfrog: e = {e:.7f} +- {e_err:.7f} (exact {-exact['e']:.7f}, {(e + exact['e']) / e_err:+.1f} sigma)")
    assert (e - (-exact["e"])) > 10 * e_err


@pytest.mark.parametrize("kind", [pkg.RNG_PHILOX4X32_10, pkg.RNG_PHILOX4X32_7], ids=["philox10", "philox7"])
@pytest.mark.parametrize("f32", [False, True], ids=["u32", "f32"])
def test_philox_fill_across_the_2_32_block_boundary(kind, f32):
    """the fill kernel's fast path assumes one high counter word per tile (round-1 product by
    increments, uniform round-2 product); the tile that straddles block 2^32 must take the
    generic path, the tiles before and after it the fast one -- all against the oracle"""
    S, seed, n = 5, 42, 8192                      # 2048 blocks per row = 8 tiles of 256 blocks
    start = 4 * ((1 << 32) - 1000)                # the boundary falls inside the 4th tile
    g, o = pkg.Rng(kind, S, seed), oracle.Rng(kind, S, seed)
    g.draws_done = start
    o.draws_done = start
    if f32:
        out = torch.empty(S * n, dtype=torch.float32, device="cuda")
        g.fill_f32(out, n)
        exp = o.fill_f32(n).view(np.uint32)
    else:
        out = dev_u32(S * n)
        g.fill_u32(out, n)
        exp = o.fill_u32(n)
    got = out.cpu().numpy().view(np.uint32)[:S * n]
    assert np.array_equal(got, exp), np.flatnonzero(got != exp)[:8]
    red = dev_u32(2 * S)
    for pos in (4 * ((1 << 32) - 500) + 1, 4 * ((1 << 32) - 1), 4 * (1 << 32), 4 * ((1 << 33) - 700) + 3):
        g.draws_done = pos                        # draw mode: unaligned head, the wrap inside, ragged tail
        o.draws_done = pos
        g.draw_reduce(red, 4001)
        assert np.array_equal(host(red, 2 * S), o.draw_reduce(4001)), pos
    g.close()


def test_xs1024_skip_seeding_large_shard_against_the_skip_matrix():
    """PAPER.md:228 at a size where the doubling tree has many levels and a ragged last one, for a
    shard whose first instance has several set bits: sampled instances against X_0 J^g computed with
    the oracle's matrix powers (J^g by binary exponentiation over the oracle's J_k = M^(2^(137+k)))"""
    n_inst, G0, seed = 3000, 0b1011010, 5
    g = pkg.Rng(pkg.RNG_XS1024W_SKIP, 32 * n_inst, seed, first=32 * G0, n_total=32 * (G0 + n_inst))
    st = g.get_state().reshape(n_inst, 32)
    g.close()
    x0 = oracle.Rng(oracle.XS1024W, 32, seed).get_state()
    Jk = [oracle.xs1024_matpow2(137)]
    for _ in range(12):
        Jk.append(oracle.xs1024_matmul(Jk[-1], Jk[-1]))

    def inst(G):
        X = x0
        for k in range(13):
            if (G >> k) & 1:
                X = oracle.xs1024_vecmat(X, Jk[k])
        return X
    for i in (0, 1, 2, 3, 63, 64, 1023, 1024, 2047, 2048, 2999):
        assert np.array_equal(st[i], inst(G0 + i)), i
    assert len({st[i].tobytes() for i in range(n_inst)}) == n_inst


# ---------------------------------------------------------------------------------
# the paper's own consumer: double checkerboard with multi-hit updates (R-E9)
# ---------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("L,T,k,sweeps", [(4, 2, 1, 6), (8, 2, 3, 4), (16, 8, 1, 5), (32, 8, 7, 3), (64, 16, 2, 4),
                                          (128, 32, 5, 2), (96, 16, 100, 1), (80, 20, 3, 2), (176, 44, 2, 2)])
def test_ising_multihit_bit_exact(kind, L, T, k, sweeps):
    S = L * L // 4
    if kind in XS_KINDS and (S % 32 or (T * T // 2) % 32):
        pytest.skip("whole warp instances per tile only")
    if kind in LFIB_KINDS and (S % 256 or T not in (8, 16)):
        pytest.skip("ring shared by a 256-thread CTA: whole instances, tile 8 or 16 (RNG_E_UNSUPPORTED is tested below)")
    beta = 0.44068679350977147
    g, o = pkg.Rng(kind, S, 13), oracle.Rng(kind, S, 13)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 4)
    sp_o = oracle.ising_init_random(L, 4)
    tr = torch.empty(sweeps, dtype=torch.int64, device="cuda")
    g.ising_sweep_multihit(sp, L, beta, sweeps, T, k, tr)
    tr_o = o.ising_sweep_multihit(sp_o, L, beta, sweeps, T, k, trace=True)
    assert np.array_equal(sp.cpu().numpy(), sp_o)
    assert np.array_equal(tr.cpu().numpy(), tr_o)
    assert g.draws_done == o.draws_done == 4 * k * sweeps
    # the streams continue: a plain fill afterwards gives the oracle's next draws
    out = dev_u32(S * 5)
    g.fill_u32(out, 5)
    assert np.array_equal(host(out, S * 5), o.fill_u32(5))
    g.close()


@pytest.mark.parametrize("kind", KINDS, ids=IDS)
@pytest.mark.parametrize("L,T,k,sweeps", [(16, 8, 1, 5), (32, 8, 7, 3), (64, 16, 2, 4), (128, 32, 5, 2), (96, 16, 100, 1),
                                          (256, 16, 1, 9), (512, 16, 3, 2), (1024, 16, 1, 3), (1024, 8, 1, 2)])
def test_ising_multihit_whole_call_in_one_launch_bit_exact(kind, L, T, k, sweeps):
    """the whole call as ONE cooperative launch (tiles stay in shared memory, generator states in registers, halos
    travel as 64-bit words between the inboxes of neighbouring tiles; variant "ising" = 4 takes this path whenever
    the call qualifies, the default only where it measured faster).  Same trajectory as one launch per coarse colour
    (variant 1); two calls per handle (stage numbers restart, the streams continue); L = 1024 makes every thread
    serve two streams"""
    S = L * L // 4
    if kind in LFIB_KINDS:
        pytest.skip("ring shared by a 256-thread CTA: per-colour launches only (covered by test_ising_multihit_bit_exact)")
    if kind == pkg.RNG_MWC_MULTI and S > (1 << 16):
        pytest.skip("the oracle finds its multipliers by the paper's plain sequential scan: 2^18 of them take minutes "
                    "(the kind is covered here up to L = 512)")
    beta = 0.4
    g, o = pkg.Rng(kind, S, 17), oracle.Rng(kind, S, 17)
    g2 = pkg.Rng(kind, S, 17)
    g.set_variant("ising", 4)
    g2.set_variant("ising", 1)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 9)
    sp2 = sp.clone()
    sp_o = oracle.ising_init_random(L, 9)
    e = torch.zeros(1, dtype=torch.int64, device="cuda")
    for call in range(2):
        l1 = pkg.rng_kernel_launches()
        g.ising_sweep_multihit(sp, L, beta, sweeps, T, k)
        assert pkg.rng_kernel_launches() - l1 == 1, "expected the one-launch path"
        g2.ising_sweep_multihit(sp2, L, beta, sweeps, T, k)
        o.ising_sweep_multihit(sp_o, L, beta, sweeps, T, k)
        assert np.array_equal(sp.cpu().numpy(), sp_o), f"call {call}: lattice"
        assert np.array_equal(sp2.cpu().numpy(), sp_o), f"call {call}: lattice (per-colour launches)"
        pkg.ising_energy(sp, L, e)
        assert int(e.item()) == oracle.ising_energy(sp_o, L)
    assert g.draws_done == o.draws_done == 2 * 4 * k * sweeps
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    out = dev_u32(S * 3)
    g.fill_u32(out, 3)
    assert np.array_equal(host(out, S * 3), o.fill_u32(3))
    g.close()
    g2.close()


@pytest.mark.parametrize("kind", [pkg.RNG_XORWOW, pkg.RNG_PHILOX4X32_10, pkg.RNG_XS1024W, pkg.RNG_LCG64, pkg.RNG_MWC_MULTI],
                         ids=["xorwow", "philox10", "xs1024w", "lcg64", "mwc_multi"])
@pytest.mark.parametrize("L,T,k,sweeps,one_launch", [(96, 24, 2, 3, True), (160, 40, 1, 3, True), (80, 40, 3, 2, True),
                                                     (240, 40, 2, 2, True), (176, 44, 2, 2, False), (72, 36, 1, 2, False)])
def test_ising_multihit_one_launch_wide_and_odd_tiles(kind, L, T, k, sweeps, one_launch):
    """tiles wider than 32 sites (the second ballot of a halo row, spin bits 32..43 of the 64-bit mailbox word beside
    its 20-bit stage number) and tile shapes whose CTA holds a number of tiles that is not a power of two (T = 24:
    three tiles, 864 threads, named barriers of 288 threads; T = 40: one tile, 800 threads).  T = 44 and 36 have
    tile_threads % 32 != 0: the one-launch plan must refuse them and the forced variant must fall back to one launch
    per coarse colour -- same lattice either way"""
    if kind in XS_KINDS and T % 8:
        pytest.skip("xs1024 needs whole warps per tile")
    S = L * L // 4
    beta = 0.4
    g, o = pkg.Rng(kind, S, 23), oracle.Rng(kind, S, 23)
    g.set_variant("ising", 4)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 5)
    sp_o = oracle.ising_init_random(L, 5)
    for call in range(2):
        l1 = pkg.rng_kernel_launches()
        g.ising_sweep_multihit(sp, L, beta, sweeps, T, k)
        assert pkg.rng_kernel_launches() - l1 == (1 if one_launch else 2 * sweeps)
        o.ising_sweep_multihit(sp_o, L, beta, sweeps, T, k)
        assert np.array_equal(sp.cpu().numpy(), sp_o), f"call {call}: lattice"
    assert g.draws_done == o.draws_done == 2 * 4 * k * sweeps
    if g.state_bytes():
        assert np.array_equal(g.get_state(), o.get_state())
    g.close()


def test_ising_multihit_argument_errors():
    g = pkg.Rng(pkg.RNG_PHILOX4X32_10, 16, 1)
    sp = torch.ones(64, dtype=torch.int8, device="cuda")
    for L, T, k in ((8, 3, 1), (8, 8, 1), (8, 2, 0), (8, 46, 1)):
        with pytest.raises(pkg.RngError) as e:
            g.ising_sweep_multihit(sp, L, 0.3, 1, T, k)
        assert e.value.code == pkg.RNG_E_INVAL
    g.close()
    g = pkg.Rng(pkg.RNG_PHILOX4X32_10, 32, 1)          # needs L*L/4 = 16 streams
    with pytest.raises(pkg.RngError):
        g.ising_sweep_multihit(sp, 8, 0.3, 1, 2, 1)
    g.close()
    g = pkg.Rng(pkg.RNG_LFIB521, 1024, 1)              # a 32 x 32 tile has 512 threads: two instances, not offered
    sp = torch.ones(64 * 64, dtype=torch.int8, device="cuda")
    with pytest.raises(pkg.RngError) as e:
        g.ising_sweep_multihit(sp, 64, 0.3, 1, 32, 1)
    assert e.value.code == pkg.RNG_E_UNSUPPORTED
    g.close()


@pytest.mark.parametrize("kind", [pkg.RNG_PHILOX4X32_10, pkg.RNG_XORWOW, pkg.RNG_XS1024W_SKIP, pkg.RNG_LFIB1279,
                                  pkg.RNG_MWC_MULTI],
                         ids=["philox10", "xorwow", "xs1024w_skip", "lfib1279", "mwc_different_a"])
def test_table1_multihit_L1024_beta04_energy_within_3_sigma(kind):
    """the paper's application test with its own kernel shape (Table 1): L = 1024, beta = 0.4,
    double checkerboard, one stream per thread (262144), e and C_V against Kaufman's exact values"""
    from exact_ising import kaufman
    L, T, k, beta = 1024, 16, 1, 0.4
    ex = kaufman(L, beta)
    g = pkg.Rng(kind, L * L // 4, 1)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 2)
    g.ising_sweep_multihit(sp, L, beta, 3000, T, k)
    n = 20000
    tr = torch.empty(n, dtype=torch.int64, device="cuda")
    g.ising_sweep_multihit(sp, L, beta, n, T, k, tr)
    e = tr.cpu().numpy().astype(np.float64) / (L * L)
    bins = e.reshape(-1, 500).mean(axis=1)
    sigma = bins.std(ddof=1) / np.sqrt(len(bins))
    assert abs(e.mean() - ex["e"]) < 3 * sigma, (e.mean(), ex["e"], sigma)
    g.close()


@pytest.mark.parametrize("kind", LFIB_KINDS, ids=["r521", "r1279"])
def test_lfib_ring_wraps_many_times_and_state_round_trips(kind):
    """long runs (the 1024 / 2048-word ring wraps hundreds of times), ragged n, f32 = the numbers themselves,
    checkpoint / resume through get_state / set_state, Ising on the byte kernel with K = 32 draws per stream"""
    S = 3 * 256
    g, o = pkg.Rng(kind, S, 17), oracle.Rng(kind, S, 17)
    for n in (1000, 1, 31, 33, 0, 64):
        out = dev_u32(S * n)
        g.fill_u32(out, n)
        assert np.array_equal(host(out, S * n), o.fill_u32(n)), n
    f = torch.empty(S * 77, dtype=torch.float32, device="cuda")
    g.fill_f32(f, 77)
    fo = o.fill_f32(77)
    assert np.array_equal(f.cpu().numpy().view(np.uint32), fo.view(np.uint32))
    assert fo.min() >= 0.0 and fo.max() < 1.0
    st = g.get_state()
    assert np.array_equal(st, o.get_state())
    red = dev_u32(2 * S)
    g.draw_reduce(red, 5000)
    want = o.draw_reduce(5000)
    assert np.array_equal(host(red, 2 * S), want)
    g2 = pkg.Rng(kind, S, 999)                      # another seed, then restored from the checkpoint
    g2.set_state(st)
    g2.draw_reduce(red, 5000)
    assert np.array_equal(host(red, 2 * S), want)
    g2.close()
    L = 256                                          # K = L*L/2/S = 128/3 not integral -> use S = 1024
    g.close()
    g, o = pkg.Rng(kind, 1024, 3), oracle.Rng(kind, 1024, 3)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, 6)
    sp_o = oracle.ising_init_random(L, 6)
    tr = torch.empty(6, dtype=torch.int64, device="cuda")
    g.ising_sweep(sp, L, 0.4, 6, tr)
    tr_o = o.ising_sweep(sp_o, L, 0.4, 6, trace=True)
    assert np.array_equal(sp.cpu().numpy(), sp_o) and np.array_equal(tr.cpu().numpy(), tr_o)
    g.close()


@pytest.mark.slow
def test_table1_lcg32_substreams_fail_like_in_the_paper():
    """PAPER.md:80 (Table 1, row 'LCG32'): sub-streams of the ONE 32-bit LCG sequence give "highly significant
    deviations"; the same kind here misses the exact energy by far more than 10 sigma"""
    from exact_ising import kaufman
    exact = kaufman(1024, 0.4)
    e, e_err, _, _ = _table1_run(pkg.RNG_LCG32_LEAPFROG, 1 << 16, sweeps=20000, nb=40)
    print(f"\nlcg32_leapfrog: e = {e:.7f} +- {e_err:.7f} (exact {-exact['e']:.7f}, {(e + exact['e']) / e_err:+.1f} sigma)")
    assert abs(e - (-exact["e"])) > 10 * e_err


def test_mwc_multipliers_found_on_the_device_match_the_oracles_scan():
    """2^16 streams with their own safe-prime multipliers (several chunks of the device search),
    for a shard that starts in the middle of the list; all of them against the oracle's scan from the top"""
    first, S = 5000, 1 << 16
    g = pkg.Rng(pkg.RNG_MWC_MULTI, S, 3, first=first, n_total=first + S)
    st = g.get_state().reshape(S, 3)
    want = oracle.mwc_multipliers(first, S)
    assert np.array_equal(st[:, 2], want)
    assert int(oracle.mwc_multipliers(0, 1)[0]) == 4294967118            # the paper's multiplier is number 0
    o = oracle.Rng(pkg.RNG_MWC_MULTI, 512, 3, first=first, n_total=first + S)
    assert np.array_equal(st[:512].reshape(-1), o.get_state())
    out = dev_u32(S * 8)
    g.fill_u32(out, 8)
    assert np.array_equal(host(out, S * 8).reshape(S, 8)[:512], o.fill_u32(8).reshape(512, 8))
    g.close()
