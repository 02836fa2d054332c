"""rng-b200: per-thread random streams and the Ising consumer on one B200 (sm_100a).

Thin Python binding over the C-ABI of ``include/rng_b200.h`` (``librng_b200.so``,
hand-written CUDA).  Argument marshalling only: every step of the path runs in the
library's kernels.  PyTorch is used by callers for device memory and streams; this
package itself only needs ``ctypes``.  There is no CPU fallback: if the shared
library is missing or no CUDA device is present, calls raise ``RngError``.
"""
from .binding import (  # noqa: F401
    RNG_LCG64, RNG_LCG64_LEAPFROG, RNG_XORWOW, RNG_PHILOX4X32_10, RNG_XS1024W, RNG_PHILOX4X32_7, RNG_LCG32, RNG_XS1024W_SKIP, RNG_LCG64_BOTH, RNG_LFIB521, RNG_LFIB1279, RNG_LCG32_LEAPFROG, RNG_MWC, RNG_MWC_MULTI,
    RNG_OK, RNG_E_INVAL, RNG_E_NOMEM, RNG_E_CUDA, RNG_E_UNSUPPORTED,
    KIND_NAMES, RngError, Rng, lib, library_path, EXPORTS,
    rng_create, rng_create_shard, rng_destroy, rng_fill_u32, rng_fill_f32, rng_draw_reduce,
    ising_sweep, ising_sweep_multihit, ising_sweep_philox_static, RNG_ISING_STATIC_MAX_L, ising_init_random, ising_energy, ising_accept_table,
    rng_fill_u32_host, rng_fill_f32_host, rng_draw_reduce_host, ising_sweep_host,
    rng_state_bytes, rng_get_state, rng_set_state, rng_draws_done, rng_set_draws_done,
    rng_set_variant, rng_kernel_launches, rng_last_error, rng_version,
)
