"""CPU ORACLE bindings (TEST INFRASTRUCTURE -- never imported by the product path).

ctypes wrapper around ``oracle/oracle.c`` (plain C written from PAPER.md).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1204_6193_b200`` and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")

LCG64, LCG64_LEAPFROG, XORWOW, PHILOX4X32_10, XS1024W, PHILOX4X32_7, LCG32, XS1024W_SKIP, LCG64_BOTH, LFIB521, LFIB1279, LCG32_LEAPFROG, MWC, MWC_MULTI = range(14)


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared oracle.c -> liboracle.so (in-tree)."""
    src = os.path.join(_HERE, "oracle.c")
    hdr = os.path.join(_HERE, "oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    cmd = ["gcc", "-std=gnu99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", _SO, src, "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        u64, u32, i32, vp = C.c_uint64, C.c_uint32, C.c_int, C.c_void_p
        L.orc_splitmix64.restype = u64
        L.orc_splitmix64.argtypes = [u64, u64]
        L.orc_lcg64_step.restype = u64
        L.orc_lcg64_step.argtypes = [u64]
        L.orc_lcg32_step.restype = u32
        L.orc_lcg32_step.argtypes = [u32]
        L.orc_lcg64_jump.restype = None
        L.orc_lcg64_jump.argtypes = [u64, C.POINTER(u64), C.POINTER(u64)]
        L.orc_philox4x32.restype = None
        L.orc_philox4x32.argtypes = [i32, vp, vp, vp]
        L.orc_xorwow_next.restype = u32
        L.orc_xorwow_next.argtypes = [vp]
        L.orc_xs1024_update.restype = None
        L.orc_xs1024_update.argtypes = [vp]
        for f, a in (("orc_xs1024_matrix", [vp]), ("orc_xs1024_vecmat", [vp, vp, vp]),
                     ("orc_xs1024_matmul", [vp, vp, vp]), ("orc_xs1024_matpow2", [C.c_uint, vp])):
            getattr(L, f).restype = None
            getattr(L, f).argtypes = a
        L.orc_u32_to_f32.restype = C.c_float
        L.orc_u32_to_f32.argtypes = [u32]
        L.orc_create.restype = vp
        L.orc_create.argtypes = [i32, u64, u64, u64, u64]
        L.orc_destroy.restype = None
        L.orc_destroy.argtypes = [vp]
        L.orc_draws_done.restype = u64
        L.orc_draws_done.argtypes = [vp]
        L.orc_set_draws_done.restype = C.c_int
        L.orc_set_draws_done.argtypes = [vp, u64]
        for name in ("orc_fill_u32", "orc_fill_f32", "orc_draw_reduce"):
            f = getattr(L, name)
            f.restype = None
            f.argtypes = [vp, vp, u64]
        L.orc_state_words32.restype = u64
        L.orc_state_words32.argtypes = [vp]
        L.orc_get_state.restype = None
        L.orc_get_state.argtypes = [vp, vp]
        L.orc_ising_accept_table.restype = None
        L.orc_ising_accept_table.argtypes = [C.c_double, vp]
        L.orc_ising_init_random.restype = None
        L.orc_ising_init_random.argtypes = [vp, u32, u64]
        L.orc_ising_energy.restype = C.c_int64
        L.orc_ising_energy.argtypes = [vp, u32]
        L.orc_ising_sweep.restype = i32
        L.orc_ising_sweep.argtypes = [vp, vp, u32, C.c_double, u32, vp]
        L.orc_ising_sweep_multihit.restype = i32
        L.orc_ising_sweep_multihit.argtypes = [vp, vp, u32, C.c_double, u32, u32, u32, vp]
        L.orc_threads.restype = i32
        L.orc_set_threads.argtypes = [i32]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


# ---- elementary pieces -------------------------------------------------------
def splitmix64(seed: int, k: int) -> int:
    return int(lib().orc_splitmix64(seed & (2**64 - 1), k & (2**64 - 1)))


def lcg64_step(x: int) -> int:
    return int(lib().orc_lcg64_step(x))


def lcg32_step(x: int) -> int:
    return int(lib().orc_lcg32_step(x))


def lcg64_jump(n: int):
    A, Cc = C.c_uint64(), C.c_uint64()
    lib().orc_lcg64_jump(n, C.byref(A), C.byref(Cc))
    return int(A.value), int(Cc.value)


def philox4x32(ctr, key, rounds: int = 10):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32(rounds, _p(c), _p(k), _p(o))
    return o


def xorwow_next(state: np.ndarray) -> int:
    """advances `state` (6 x uint32, in place) and returns the draw."""
    assert state.dtype == np.uint32 and state.size == 6
    return int(lib().orc_xorwow_next(_p(state)))


def mwc_multipliers(first: int, count: int) -> np.ndarray:
    out = np.empty(count, dtype=np.uint32)
    L = lib()
    L.orc_mwc_multipliers.restype = C.c_int
    L.orc_mwc_multipliers.argtypes = [C.c_uint64, C.c_uint64, C.c_void_p]
    if L.orc_mwc_multipliers(first, count, _p(out)) != 0:
        raise ValueError("ran out of multipliers")
    return out


def is_prime64(n: int) -> bool:
    """the oracle's primality decision for n < 2^64 (trial division + Miller-Rabin)"""
    L = lib()
    L.orc_is_prime64.restype = C.c_int
    L.orc_is_prime64.argtypes = [C.c_uint64]
    return bool(L.orc_is_prime64(n))


def xs1024_matpow2(k: int) -> np.ndarray:
    """M^(2^k) as a [1024, 32] uint32 bit matrix (row r = image of unit vector word r//32, bit r%32)"""
    out = np.empty((1024, 32), dtype=np.uint32)
    lib().orc_xs1024_matpow2(k, _p(out))
    return out


def xs1024_matmul(A: np.ndarray, B: np.ndarray) -> np.ndarray:
    out = np.empty((1024, 32), dtype=np.uint32)
    lib().orc_xs1024_matmul(_p(np.ascontiguousarray(A)), _p(np.ascontiguousarray(B)), _p(out))
    return out


def xs1024_vecmat(X: np.ndarray, A: np.ndarray) -> np.ndarray:
    out = np.empty(32, dtype=np.uint32)
    lib().orc_xs1024_vecmat(_p(np.ascontiguousarray(X, dtype=np.uint32)), _p(np.ascontiguousarray(A)), _p(out))
    return out


def xs1024_update(X: np.ndarray) -> None:
    assert X.dtype == np.uint32 and X.size == 32
    lib().orc_xs1024_update(_p(X))


def u32_to_f32(u: int) -> float:
    return float(lib().orc_u32_to_f32(u))


def threads() -> int:
    return int(lib().orc_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


# ---- stream object -----------------------------------------------------------
class Rng:
    def __init__(self, kind: int, n_streams: int, seed: int, first: int = 0, n_total: int | None = None):
        self.kind, self.n_streams, self.seed = kind, n_streams, seed
        n_total = n_streams + first if n_total is None else n_total
        self._h = lib().orc_create(kind, n_total, first, n_streams, seed & (2**64 - 1))
        if not self._h:
            raise ValueError("orc_create: invalid arguments")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    @property
    def draws_done(self) -> int:
        return int(lib().orc_draws_done(self._h))

    @draws_done.setter
    def draws_done(self, v: int):
        if lib().orc_set_draws_done(self._h, v) != 0:
            raise ValueError("only counter-based (Philox) streams can be repositioned")

    def fill_u32(self, n: int) -> np.ndarray:
        out = np.empty(self.n_streams * n, dtype=np.uint32)
        lib().orc_fill_u32(self._h, _p(out), n)
        return out

    def fill_f32(self, n: int) -> np.ndarray:
        out = np.empty(self.n_streams * n, dtype=np.float32)
        lib().orc_fill_f32(self._h, _p(out), n)
        return out

    def draw_reduce(self, n: int) -> np.ndarray:
        out = np.empty(self.n_streams * 2, dtype=np.uint32)
        lib().orc_draw_reduce(self._h, _p(out), n)
        return out

    def get_state(self) -> np.ndarray:
        out = np.empty(int(lib().orc_state_words32(self._h)), dtype=np.uint32)
        lib().orc_get_state(self._h, _p(out))
        return out

    def ising_sweep(self, spins: np.ndarray, L: int, beta: float, n_sweeps: int, trace: bool = False):
        assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
        tr = np.empty(n_sweeps, dtype=np.int64) if trace else None
        rc = lib().orc_ising_sweep(self._h, _p(spins), L, float(beta), n_sweeps, _p(tr) if trace else None)
        if rc != 0:
            raise ValueError("orc_ising_sweep: invalid arguments")
        return tr

    def ising_sweep_multihit(self, spins: np.ndarray, L: int, beta: float, n_sweeps: int, tile: int, k_hits: int,
                             trace: bool = False):
        assert spins.dtype == np.int8 and spins.size == L * L and spins.flags.c_contiguous
        tr = np.empty(n_sweeps, dtype=np.int64) if trace else None
        rc = lib().orc_ising_sweep_multihit(self._h, _p(spins), L, float(beta), n_sweeps, tile, k_hits,
                                            _p(tr) if trace else None)
        if rc != 0:
            raise ValueError("orc_ising_sweep_multihit: invalid arguments")
        return tr


def ising_accept_table(beta: float) -> np.ndarray:
    P = np.empty(5, dtype=np.float32)
    lib().orc_ising_accept_table(float(beta), _p(P))
    return P


def ising_init_random(L: int, seed: int) -> np.ndarray:
    sp = np.empty(L * L, dtype=np.int8)
    lib().orc_ising_init_random(_p(sp), L, seed & (2**64 - 1))
    return sp


def ising_energy(spins: np.ndarray, L: int) -> int:
    assert spins.dtype == np.int8 and spins.size == L * L
    return int(lib().orc_ising_energy(_p(spins), L))
