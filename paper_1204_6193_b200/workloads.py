"""BASELINE.json configs C1-C5 as plain data (sizes, seeds, shapes).

This module holds NONE of the method's arithmetic: every input of this hot path is a
(kind, n_streams, seed, n) tuple or a lattice drawn from a seed by a counter-based
rule that the oracle and the CUDA path each implement for themselves.  tests/,
bench.py and __graft_entry__.py read their workload definitions from here.
"""
from __future__ import annotations

from dataclasses import dataclass

LCG64, LCG64_LEAPFROG, XORWOW, PHILOX4X32_10, XS1024W, PHILOX4X32_7, LCG32, XS1024W_SKIP, LCG64_BOTH, LFIB521, LFIB1279, LCG32_LEAPFROG, MWC, MWC_MULTI = range(14)
MASTER_SEED = 1                    # "seeded via splitmix64(master seed 1)" (config 1)
LATTICE_SEED = 2                   # ising_init_random seed
BETA_C = 0.44068679350977147       # ln(1+sqrt 2)/2 as a double (config 5)


@dataclass(frozen=True)
class FillCfg:
    name: str
    kind: int
    n_streams: int
    n_per_stream: int          # per call
    calls: int = 1             # successive calls into one reused buffer (state persists)
    seed: int = MASTER_SEED

    @property
    def draws_per_call(self) -> int:
        return self.n_streams * self.n_per_stream


@dataclass(frozen=True)
class IsingCfg:
    name: str
    kind: int
    L: int
    beta: float
    n_streams: int
    n_sweeps: int
    seed: int = MASTER_SEED
    lattice_seed: int = LATTICE_SEED
    tile: int = 0              # > 0: the paper's double-checkerboard multi-hit kernel with this tile size
    k_hits: int = 1            # hits per tile visit (k = 1 and k = 100)


# C1: 64-bit LCG, 1024 streams x 4096 u32 (16 MiB) -- the small case the oracle does in ms
C1 = FillCfg("C1_lcg64_1024x4096", LCG64, 1024, 4096)
# C2: Philox4x32-10, 2^20 streams x 1024 u32 = 4 GiB -- the config `metric` is quoted on
C2 = FillCfg("C2_philox_2^20x1024", PHILOX4X32_10, 1 << 20, 1024)
# C3: XORWOW, 2^22 threads x 256 draws in-register, {xor,sum} checksum per thread
C3 = FillCfg("C3_xorwow_2^22x256", XORWOW, 1 << 22, 256)
# C4: the paper's generator, 2^16 blocks x 256 threads = 2^24 streams x 4096 u32.
# 256 GiB of output cannot be resident: fill mode = 64 calls x 64 draws into one 4 GiB buffer.
C4_FILL = FillCfg("C4_xs1024_2^24x4096_fill", XS1024W, 1 << 24, 64, calls=64)
C4_DRAW = FillCfg("C4_xs1024_2^24x4096_draw", XS1024W, 1 << 24, 4096)
# supplementary 4 GiB fills for the stateful per-thread generators (SURVEY.md 8(d) C1 note)
C1_BIG = FillCfg("C1big_lcg64_2^20x1024", LCG64, 1 << 20, 1024)
C3_FILL = FillCfg("C3fill_xorwow_2^20x1024", XORWOW, 1 << 20, 1024)
# SURVEY.md 8(f)-1, the cheap extra kinds of the paper's Table 2, C2's shape
N1_PHILOX7 = FillCfg("N1_philox7_2^20x1024", PHILOX4X32_7, 1 << 20, 1024)
N1_LCG32 = FillCfg("N1_lcg32_2^20x1024", LCG32, 1 << 20, 1024)
N1_PHILOX7_DRAW = FillCfg("N1_philox7_2^22x256", PHILOX4X32_7, 1 << 22, 256)
N1_PHILOX10_DRAW = FillCfg("N1_philox10_2^22x256", PHILOX4X32_10, 1 << 22, 256)
N1_LCG32_DRAW = FillCfg("N1_lcg32_2^22x256", LCG32, 1 << 22, 256)
N1_LCG64_DRAW = FillCfg("N1_lcg64_2^22x256", LCG64, 1 << 22, 256)
N1_LCG64BOTH_DRAW = FillCfg("N1_lcg64both_2^22x256", LCG64_BOTH, 1 << 22, 256)
N3_MWC_DRAW = FillCfg("N3_mwc_2^22x256", MWC, 1 << 22, 256)  # PAPER.md:62-68; Table 2 row "MWC"
N1_LCG64BOTH = FillCfg("N1_lcg64both_2^20x1024", LCG64_BOTH, 1 << 20, 1024)
# the float lagged Fibonacci generators (Table 2), same shapes
N4_LFIB521 = FillCfg("N4_lfib521_2^20x1024", LFIB521, 1 << 20, 1024)
N4_LFIB1279 = FillCfg("N4_lfib1279_2^20x1024", LFIB1279, 1 << 20, 1024)
N4_LFIB521_DRAW = FillCfg("N4_lfib521_2^22x256", LFIB521, 1 << 22, 256)
N4_LFIB1279_DRAW = FillCfg("N4_lfib1279_2^22x256", LFIB1279, 1 << 22, 256)

# C5a: L=4, beta=0.3 vs exact enumeration; 8 streams (K = 1 site per stream per colour)
C5A_PHILOX = IsingCfg("C5a_ising_L4_philox", PHILOX4X32_10, 4, 0.3, 8, 1000)
C5A_XORWOW = IsingCfg("C5a_ising_L4_xorwow", XORWOW, 4, 0.3, 8, 1000)
# C5b: L=8192 at beta_c, 1000 sweeps from a random start
C5B_PHILOX = IsingCfg("C5b_ising_L8192_philox_K4", PHILOX4X32_10, 8192, BETA_C, 1 << 23, 1000)
C5B_XORWOW = IsingCfg("C5b_ising_L8192_xorwow_K256", XORWOW, 8192, BETA_C, 1 << 17, 1000)
C5B_XORWOW_K8 = IsingCfg("C5b_ising_L8192_xorwow_K8", XORWOW, 8192, BETA_C, 1 << 22, 1000)

# the paper's Table 1 workload: 1024^2 at beta = 0.4, double checkerboard,
# one stream per thread (262144), k = 1 and k = 100 hits; and the same at L = 8192 (2^24 streams) to fill a B200
T1_XORWOW_K1 = IsingCfg("T1_multihit_L1024_xorwow_k1", XORWOW, 1024, 0.4, 1 << 18, 1000, tile=16, k_hits=1)
T1_XORWOW_K100 = IsingCfg("T1_multihit_L1024_xorwow_k100", XORWOW, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1_PHILOX_K100 = IsingCfg("T1_multihit_L1024_philox_k100", PHILOX4X32_10, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1_XS1024_K100 = IsingCfg("T1_multihit_L1024_xs1024skip_k100", XS1024W_SKIP, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1_LCG32_K100 = IsingCfg("T1_multihit_L1024_lcg32_k100", LCG32, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1_MWC_K100 = IsingCfg("T1_multihit_L1024_mwc_k100", MWC, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1_LFIB521_K100 = IsingCfg("T1_multihit_L1024_lfib521_k100", LFIB521, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1_LFIB1279_K100 = IsingCfg("T1_multihit_L1024_lfib1279_k100", LFIB1279, 1024, 0.4, 1 << 18, 10, tile=16, k_hits=100)
T1BIG_XORWOW_K100 = IsingCfg("T1big_multihit_L8192_xorwow_k100", XORWOW, 8192, 0.4, 1 << 24, 2, tile=16, k_hits=100)
T1BIG_XORWOW_K1 = IsingCfg("T1big_multihit_L8192_xorwow_k1", XORWOW, 8192, 0.4, 1 << 24, 100, tile=16, k_hits=1)
T1BIG_XORWOW_K100_T8 = IsingCfg("T1big_multihit_L8192_xorwow_k100_tile8", XORWOW, 8192, 0.4, 1 << 24, 2, tile=8, k_hits=100)
T1_XORWOW_K100_T8 = IsingCfg("T1_multihit_L1024_xorwow_k100_tile8", XORWOW, 1024, 0.4, 1 << 18, 10, tile=8, k_hits=100)

FILL_CONFIGS = [C1, C2, C3_FILL, C1_BIG, C4_FILL]
DRAW_CONFIGS = [C3, C4_DRAW]
ISING_CONFIGS = [C5A_PHILOX, C5A_XORWOW, C5B_PHILOX, C5B_XORWOW, C5B_XORWOW_K8]
