"""The performance column of the paper's Table 2 on one B200 with this library.

    python -m paper_1204_6193_b200.table2 [--markdown]

For every generator of the table that this library has: 10^9 32-bit numbers per second with the numbers consumed
in-register (rng_draw_reduce: the paper's "compute-bound" peak figure) on a fully loaded device,
the state size per stream, and the paper's number on its GTX 480.  Needs a CUDA device.
"""
from __future__ import annotations

import argparse

# (row label, kind name, streams, draws per stream, state bits per thread as the paper counts them, paper's 10^9/s)
ROWS = [
    ("LCG32", "RNG_LCG32", 1 << 22, 1024, "32", 58.0),
    ("LCG64", "RNG_LCG64", 1 << 22, 1024, "64", 46.0),
    ("LCG64, both words (PAPER.md:58)", "RNG_LCG64_BOTH", 1 << 22, 1024, "64", None),
    ("MWC", "RNG_MWC_MULTI", 1 << 20, 1024, "64+32", 44.0),
    ("Fibonacci, r = 521", "RNG_LFIB521", 1 << 22, 1024, ">= 80", 23.0),
    ("Fibonacci, r = 1279", "RNG_LFIB1279", 1 << 22, 1024, ">= 80", 23.0),
    ("XORWOW", "RNG_XORWOW", 1 << 22, 1024, "192", 19.0),
    ("XORShift/Weyl", "RNG_XS1024W", 1 << 24, 1024, "32", 18.0),
    ("Philox4x32_7", "RNG_PHILOX4X32_7", 1 << 22, 1024, "(128)", 41.0),
    ("Philox4x32_10", "RNG_PHILOX4X32_10", 1 << 22, 1024, "(128)", 30.0),
]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--markdown", action="store_true")
    ap.add_argument("--reps", type=int, default=5)
    a = ap.parse_args()
    import torch

    import paper_1204_6193_b200 as pkg
    if not torch.cuda.is_available():
        raise SystemExit("table2: needs a CUDA device (this library has no CPU fallback)")
    head = ["generator", "bits/thread", "10^9 numbers/s (B200, in-register)", "paper (GTX 480)", "ratio"]
    if a.markdown:
        print("| " + " | ".join(head) + " |\n|" + "---|" * len(head))
    else:
        print("  ".join(head))
    out = torch.empty(2 << 24, dtype=torch.int32, device="cuda")
    for label, kname, S, n, bits, paper in ROWS:
        g = pkg.Rng(getattr(pkg, kname), S, 1)
        g.draw_reduce(out, n)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(a.reps):
            g.draw_reduce(out, n)
        e1.record()
        torch.cuda.synchronize()
        g.close()
        rate = S * n * a.reps / (e0.elapsed_time(e1) * 1e-3) / 1e9
        cells = [label, bits, f"{rate:.0f}", "-" if paper is None else f"{paper:.0f}",
                 "-" if paper is None else f"{rate / paper:.0f}x"]
        print(("| " + " | ".join(cells) + " |") if a.markdown else "  ".join(cells), flush=True)


if __name__ == "__main__":
    main()
