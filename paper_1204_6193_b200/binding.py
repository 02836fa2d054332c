"""ctypes binding of include/rng_b200.h -- same names, argument marshalling only.

Low-level functions take raw addresses (``tensor.data_ptr()`` for device buffers,
``ndarray.ctypes.data`` for host buffers) exactly like the C prototypes and raise
``RngError`` (carrying the negative C return code) instead of returning it.
``Rng`` is a small convenience wrapper that owns a handle and accepts torch tensors
(device) or numpy arrays (host) directly.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "librng_b200.so")

RNG_LCG64, RNG_LCG64_LEAPFROG, RNG_XORWOW, RNG_PHILOX4X32_10, RNG_XS1024W, RNG_PHILOX4X32_7, RNG_LCG32, RNG_XS1024W_SKIP, RNG_LCG64_BOTH, RNG_LFIB521, RNG_LFIB1279, RNG_LCG32_LEAPFROG, RNG_MWC, RNG_MWC_MULTI = range(14)
RNG_OK, RNG_E_INVAL, RNG_E_NOMEM, RNG_E_CUDA, RNG_E_UNSUPPORTED = 0, -1, -2, -3, -4
KIND_NAMES = {RNG_LCG64: "lcg64", RNG_LCG64_LEAPFROG: "lcg64_leapfrog", RNG_XORWOW: "xorwow",
              RNG_PHILOX4X32_10: "philox4x32_10", RNG_XS1024W: "xs1024w",
              RNG_PHILOX4X32_7: "philox4x32_7", RNG_LCG32: "lcg32", RNG_XS1024W_SKIP: "xs1024w_skip",
              RNG_LCG64_BOTH: "lcg64_both", RNG_LFIB521: "lfib521", RNG_LFIB1279: "lfib1279",
              RNG_LCG32_LEAPFROG: "lcg32_leapfrog", RNG_MWC: "mwc", RNG_MWC_MULTI: "mwc_multi"}

_u64, _u32, _i32, _vp, _dbl = C.c_uint64, C.c_uint32, C.c_int, C.c_void_p, C.c_double

# every symbol include/rng_b200.h declares: name -> (restype, argtypes)
EXPORTS = {
    "rng_create": (_i32, [_i32, _u64, _u64, C.POINTER(_vp)]),
    "rng_create_shard": (_i32, [_i32, _u64, _u64, _u64, _u64, C.POINTER(_vp)]),
    "rng_destroy": (_i32, [_vp]),
    "rng_fill_u32": (_i32, [_vp, _vp, _u64, _vp]),
    "rng_fill_f32": (_i32, [_vp, _vp, _u64, _vp]),
    "rng_draw_reduce": (_i32, [_vp, _vp, _u64, _vp]),
    "ising_sweep": (_i32, [_vp, _vp, _u32, _dbl, _u32, _vp, _vp]),
    "ising_sweep_multihit": (_i32, [_vp, _vp, _u32, _dbl, _u32, _u32, _u32, _vp, _vp]),
    "ising_sweep_philox_static": (_i32, [_u64, _u64, _u64, _vp, _u32, _dbl, _u32, _vp, _vp]),
    "ising_init_random": (_i32, [_vp, _u32, _u64, _vp]),
    "ising_energy": (_i32, [_vp, _u32, _vp, _vp]),
    "ising_accept_table": (_i32, [_dbl, _vp, _vp]),
    "rng_fill_u32_host": (_i32, [_vp, _vp, _u64, _vp]),
    "rng_fill_f32_host": (_i32, [_vp, _vp, _u64, _vp]),
    "rng_draw_reduce_host": (_i32, [_vp, _vp, _u64, _vp]),
    "ising_sweep_host": (_i32, [_vp, _vp, _u32, _dbl, _u32, _vp, _vp]),
    "rng_state_bytes": (_u64, [_i32, _u64]),
    "rng_get_state": (_i32, [_vp, _vp, _u64]),
    "rng_set_state": (_i32, [_vp, _vp, _u64]),
    "rng_draws_done": (_u64, [_vp]),
    "rng_set_draws_done": (_i32, [_vp, _u64]),
    "rng_set_variant": (_i32, [_vp, C.c_char_p, _i32]),
    "rng_kernel_launches": (_u64, []),
    "rng_last_error": (C.c_char_p, []),
    "rng_version": (C.c_char_p, []),
}


class RngError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"rng_b200 error {code}: {msg}")
        self.code = code


def library_path() -> str:
    return _SO


_lib = None


def lib():
    """Load librng_b200.so (built in-tree by paper_1204_6193_b200.build).  Fails
    loudly if it is missing: there is no fallback implementation."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RngError(RNG_E_CUDA, f"{_SO} not built; run `python -m paper_1204_6193_b200.build` "
                                       "(no CPU fallback exists)")
        L = C.CDLL(_SO)
        for name, (res, args) in EXPORTS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _check(rc: int) -> None:
    if rc != RNG_OK:
        raise RngError(rc, rng_last_error())


def _ptr(x) -> int | None:
    """address of a device tensor / host ndarray / int / None"""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if hasattr(x, "ctypes"):
        return int(x.ctypes.data)
    raise TypeError(f"cannot take the address of {type(x)!r}")


def _stream(s) -> int | None:
    if s is None or isinstance(s, int):
        return s or None
    return int(s.cuda_stream)  # torch.cuda.Stream


# ---- C-ABI, one to one ----------------------------------------------------------
def rng_last_error() -> str:
    return (lib().rng_last_error() or b"").decode()


def rng_version() -> str:
    return lib().rng_version().decode()


def rng_kernel_launches() -> int:
    return int(lib().rng_kernel_launches())


def rng_create(kind: int, n_streams: int, seed: int) -> int:
    h = _vp()
    _check(lib().rng_create(kind, n_streams, seed & (2**64 - 1), C.byref(h)))
    return h.value


def rng_create_shard(kind: int, n_total: int, first: int, n_local: int, seed: int) -> int:
    h = _vp()
    _check(lib().rng_create_shard(kind, n_total, first, n_local, seed & (2**64 - 1), C.byref(h)))
    return h.value


def rng_destroy(h: int) -> None:
    _check(lib().rng_destroy(h))


def rng_fill_u32(h, d_out, n: int, cuda_stream=None) -> None:
    _check(lib().rng_fill_u32(h, _ptr(d_out), n, _stream(cuda_stream)))


def rng_fill_f32(h, d_out, n: int, cuda_stream=None) -> None:
    _check(lib().rng_fill_f32(h, _ptr(d_out), n, _stream(cuda_stream)))


def rng_draw_reduce(h, d_out, n: int, cuda_stream=None) -> None:
    _check(lib().rng_draw_reduce(h, _ptr(d_out), n, _stream(cuda_stream)))


def ising_sweep(h, d_spins, L: int, beta: float, n_sweeps: int, d_energy_trace=None, cuda_stream=None) -> None:
    _check(lib().ising_sweep(h, _ptr(d_spins), L, float(beta), n_sweeps, _ptr(d_energy_trace), _stream(cuda_stream)))


def ising_sweep_multihit(h, d_spins, L: int, beta: float, n_sweeps: int, tile: int, k_hits: int, d_energy_trace=None,
                         cuda_stream=None) -> None:
    _check(lib().ising_sweep_multihit(h, _ptr(d_spins), L, float(beta), n_sweeps, tile, k_hits, _ptr(d_energy_trace),
                                      _stream(cuda_stream)))


RNG_ISING_STATIC_MAX_L = 4096


def ising_sweep_philox_static(n_streams: int, seed: int, draws_done: int, d_spins, L: int, beta: float, n_sweeps: int,
                              d_energy_trace=None, cuda_stream=None) -> None:
    """ising_sweep for callers that cannot allocate device memory (no handle, Philox4x32-10, the bit planes in
    a fixed 2 MiB array of the library: L <= RNG_ISING_STATIC_MAX_L).  The caller keeps the stream position:
    the next call takes draws_done + n_sweeps * L * L // n_streams.  See include/rng_b200.h."""
    _check(lib().ising_sweep_philox_static(n_streams, seed & (2**64 - 1), draws_done, _ptr(d_spins), L, float(beta), n_sweeps,
                                           _ptr(d_energy_trace), _stream(cuda_stream)))


def ising_init_random(d_spins, L: int, seed: int, cuda_stream=None) -> None:
    _check(lib().ising_init_random(_ptr(d_spins), L, seed & (2**64 - 1), _stream(cuda_stream)))


def ising_energy(d_spins, L: int, d_out, cuda_stream=None) -> None:
    _check(lib().ising_energy(_ptr(d_spins), L, _ptr(d_out), _stream(cuda_stream)))


def ising_accept_table(beta: float):
    """-> (P float32[5], T uint32[5]) as Python lists (host-side, needs no GPU)"""
    P = (C.c_float * 5)()
    T = (_u32 * 5)()
    _check(lib().ising_accept_table(float(beta), C.addressof(P), C.addressof(T)))
    return list(P), list(T)


def rng_fill_u32_host(h, h_out, n: int, cuda_stream=None) -> None:
    _check(lib().rng_fill_u32_host(h, _ptr(h_out), n, _stream(cuda_stream)))


def rng_fill_f32_host(h, h_out, n: int, cuda_stream=None) -> None:
    _check(lib().rng_fill_f32_host(h, _ptr(h_out), n, _stream(cuda_stream)))


def rng_draw_reduce_host(h, h_out, n: int, cuda_stream=None) -> None:
    _check(lib().rng_draw_reduce_host(h, _ptr(h_out), n, _stream(cuda_stream)))


def ising_sweep_host(h, h_spins, L: int, beta: float, n_sweeps: int, h_energy_trace=None, cuda_stream=None) -> None:
    _check(lib().ising_sweep_host(h, _ptr(h_spins), L, float(beta), n_sweeps, _ptr(h_energy_trace),
                                  _stream(cuda_stream)))


def rng_state_bytes(kind: int, n_streams: int) -> int:
    return int(lib().rng_state_bytes(kind, n_streams))


def rng_get_state(h, h_buf, nbytes: int) -> None:
    _check(lib().rng_get_state(h, _ptr(h_buf), nbytes))


def rng_set_state(h, h_buf, nbytes: int) -> None:
    _check(lib().rng_set_state(h, _ptr(h_buf), nbytes))


def rng_draws_done(h) -> int:
    return int(lib().rng_draws_done(h))


def rng_set_draws_done(h, draws_done: int) -> None:
    _check(lib().rng_set_draws_done(h, draws_done))


def rng_set_variant(h, name: str, value: int) -> None:
    _check(lib().rng_set_variant(h, name.encode(), value))


# ---- convenience owner ----------------------------------------------------------
class Rng:
    """Owns one rng_handle.  Methods forward to the C-ABI calls of the same name."""

    def __init__(self, kind: int, n_streams: int, seed: int, first: int = 0, n_total: int | None = None):
        self.kind, self.n_streams, self.seed, self.first = kind, n_streams, seed, first
        self.n_total = n_streams + first if n_total is None else n_total
        self._h = None
        self._h = rng_create_shard(kind, self.n_total, first, n_streams, seed)

    def close(self):
        if self._h:
            rng_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def handle(self) -> int:
        return self._h

    @property
    def draws_done(self) -> int:
        return rng_draws_done(self._h)

    @draws_done.setter
    def draws_done(self, v: int):
        rng_set_draws_done(self._h, v)

    def fill_u32(self, d_out, n, stream=None):
        rng_fill_u32(self._h, d_out, n, stream)

    def fill_f32(self, d_out, n, stream=None):
        rng_fill_f32(self._h, d_out, n, stream)

    def draw_reduce(self, d_out, n, stream=None):
        rng_draw_reduce(self._h, d_out, n, stream)

    def ising_sweep(self, d_spins, L, beta, n_sweeps, d_energy_trace=None, stream=None):
        ising_sweep(self._h, d_spins, L, beta, n_sweeps, d_energy_trace, stream)

    def ising_sweep_multihit(self, d_spins, L, beta, n_sweeps, tile, k_hits, d_energy_trace=None, stream=None):
        ising_sweep_multihit(self._h, d_spins, L, beta, n_sweeps, tile, k_hits, d_energy_trace, stream)

    def fill_u32_host(self, h_out, n, stream=None):
        rng_fill_u32_host(self._h, h_out, n, stream)

    def fill_f32_host(self, h_out, n, stream=None):
        rng_fill_f32_host(self._h, h_out, n, stream)

    def draw_reduce_host(self, h_out, n, stream=None):
        rng_draw_reduce_host(self._h, h_out, n, stream)

    def ising_sweep_host(self, h_spins, L, beta, n_sweeps, h_energy_trace=None, stream=None):
        ising_sweep_host(self._h, h_spins, L, beta, n_sweeps, h_energy_trace, stream)

    def state_bytes(self) -> int:
        return rng_state_bytes(self.kind, self.n_streams)

    def get_state(self):
        import numpy as np
        buf = np.empty(self.state_bytes() // 4, dtype=np.uint32)
        rng_get_state(self._h, buf, buf.nbytes)
        return buf

    def set_state(self, buf):
        rng_set_state(self._h, buf, buf.nbytes)

    def set_variant(self, name: str, value: int):
        rng_set_variant(self._h, name, value)
