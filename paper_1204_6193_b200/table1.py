"""Reproduce the paper's Table 1 on one B200 with this library.

    python -m paper_1204_6193_b200.table1 [--sweeps 100000] [--therm 3000] [--tile 16] [--only KIND,...] [--markdown]

For every generator of the table: a Metropolis simulation of the 1024 x 1024 Ising model at beta = 0.4 with
the paper's double-checkerboard kernel (ising_sweep_multihit, k = 1, one stream per thread = 262144 streams),
internal energy e = -E/N and specific heat C_V with jackknife errors and their deviation from the exact values
the paper prints (e = 1.106079207, C_V = 0.8616983594), and the time per spin update t_up for k = 1
and k = 100.  The paper used 10^7 sweeps; the default here is 10^5 (errors about 10 times larger).
Needs a CUDA device; nothing here runs on the CPU except the statistics of the energy trace.
"""
from __future__ import annotations

import argparse
import math

EXACT_E, EXACT_CV = 1.106079207, 0.8616983594  # PAPER.md:74 (Ref.[9]); e is printed as -E/N
L, BETA = 1024, 0.4

# (row label of the paper, kind name in this library, paper's t_up k=1 / k=100 in ns, paper's Delta_rel of e)
ROWS = [
    ("LCG32", "RNG_LCG32_LEAPFROG", 0.2221, 0.0402, None),
    ("LCG32, random", "RNG_LCG32", 0.2221, 0.0402, -0.97),
    ("LCG64", "RNG_LCG64_LEAPFROG", 0.2311, 0.0471, 13.72),
    ("LCG64, random", "RNG_LCG64", 0.2311, 0.0471, 0.62),
    ("MWC, same a", "RNG_MWC", 0.2293, 0.0435, 0.45),
    ("MWC, different a", "RNG_MWC_MULTI", 0.2336, 0.0438, 0.28),
    ("Fibonacci, r = 521", "RNG_LFIB521", 0.2601, 0.0661, 6.43),
    ("Fibonacci, r = 1279", "RNG_LFIB1279", 0.2904, 0.0700, 0.40),
    ("XORWOW", "RNG_XORWOW", 0.7956, 0.0576, -9.13),
    ("XORShift/Weyl", "RNG_XS1024W_SKIP", 0.2613, 0.0721, -0.23),
    ("Philox4x32_7", "RNG_PHILOX4X32_7", 0.2399, 0.0523, -0.79),
    ("Philox4x32_10", "RNG_PHILOX4X32_10", 0.2577, 0.0622, -0.85),
]


def jackknife(e, nb):
    import numpy as np
    n = len(e) // nb * nb
    e = e[:n]
    bins = e.reshape(nb, -1)
    e_err = bins.mean(axis=1).std(ddof=1) / math.sqrt(nb)
    N = L * L
    tot1, tot2 = e.sum(), (e * e).sum()
    b1, b2, m = bins.sum(axis=1), (bins * bins).sum(axis=1), n - bins.shape[1]
    jk = BETA * BETA * N * ((tot2 - b2) / m - ((tot1 - b1) / m) ** 2)
    cv = BETA * BETA * N * (tot2 / n - (tot1 / n) ** 2)
    cv_err = math.sqrt((nb - 1) / nb * float(((jk - jk.mean()) ** 2).sum()))
    return float(e.mean()), float(e_err), float(cv), cv_err


def time_updates(pkg, torch, kind, tile, k_hits, sweeps, seed):
    g = pkg.Rng(kind, L * L // 4, seed)
    sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
    pkg.ising_init_random(sp, L, seed + 100)
    g.ising_sweep_multihit(sp, L, BETA, max(1, sweeps // 10), tile, k_hits)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.ising_sweep_multihit(sp, L, BETA, sweeps, tile, k_hits)
    e1.record()
    torch.cuda.synchronize()
    g.close()
    return e0.elapsed_time(e1) * 1e6 / (float(L) * L * sweeps * k_hits)  # ns per spin update


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sweeps", type=int, default=100000)
    ap.add_argument("--therm", type=int, default=3000)
    ap.add_argument("--tile", type=int, default=16)
    ap.add_argument("--bins", type=int, default=100)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--markdown", action="store_true")
    ap.add_argument("--only", default="", help="comma-separated kind names (e.g. RNG_XORWOW,RNG_LFIB521); default: all rows")
    a = ap.parse_args()
    only = {k.strip() for k in a.only.split(",") if k.strip()}
    import numpy as np
    import torch

    import paper_1204_6193_b200 as pkg
    if not torch.cuda.is_available():
        raise SystemExit("table1: needs a CUDA device (this library has no CPU fallback)")
    sep = " | " if a.markdown else "  "
    head = ["method", "e", "D_rel", "C_V", "D_rel", "t_up k=1 [ns]", "t_up k=100 [ns]", "paper: D_rel(e), t_up k=1 / k=100"]
    if a.markdown:
        print("| " + " | ".join(head) + " |\n|" + "---|" * len(head))
    else:
        print(sep.join(head))
    for label, kname, t1_paper, t100_paper, d_paper in ROWS:
        if only and kname not in only:
            continue
        kind = getattr(pkg, kname)
        g = pkg.Rng(kind, L * L // 4, a.seed)
        sp = torch.empty(L * L, dtype=torch.int8, device="cuda")
        pkg.ising_init_random(sp, L, a.seed + 100)
        g.ising_sweep_multihit(sp, L, BETA, a.therm, a.tile, 1)
        tr = torch.empty(a.sweeps, dtype=torch.int64, device="cuda")
        g.ising_sweep_multihit(sp, L, BETA, a.sweeps, a.tile, 1, tr)
        g.close()
        e = -tr.cpu().numpy().astype(np.float64) / (L * L)
        em, ee, cv, cve = jackknife(e, a.bins)
        t1 = time_updates(pkg, torch, kind, a.tile, 1, 2000, a.seed)
        t100 = time_updates(pkg, torch, kind, a.tile, 100, 20, a.seed)
        cells = [label, f"{em:.7f}({ee * 1e7:.0f})", f"{(em - EXACT_E) / ee:+.2f}", f"{cv:.5f}({cve * 1e5:.0f})",
                 f"{(cv - EXACT_CV) / cve:+.2f}", f"{t1:.5f}", f"{t100:.5f}",
                 f"{'n/a' if d_paper is None else format(d_paper, '+.2f')}, {t1_paper} / {t100_paper}"]
        print(("| " + " | ".join(cells) + " |") if a.markdown else sep.join(cells), flush=True)


if __name__ == "__main__":
    main()
