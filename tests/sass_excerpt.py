"""Per-kernel counts of the SASS mnemonics that back the claims in DESIGN.md (TMA tensor stores, programmatic
dependent launch, streaming 128-bit stores, Philox's wide multiplies, warp shuffles), from `cuobjdump -sass` of
the built library.  Text evidence for profiles/; nothing here runs a kernel.

    python tests/sass_excerpt.py > profiles/r03_sass_excerpt.txt

A profiling aid kept beside the tests (it is not part of the library package).
"""
from __future__ import annotations

import re
import subprocess
import sys

import os

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_1204_6193_b200.build import build  # noqa: E402

MNEMONICS = ["UTMASTG", "ACQBULK", "PREEXIT", "STG.E.EF.128", "STS.128", "IMAD.WIDE.U32", "SHFL", "ATOMG", "I2FP",
             "BAR.SYNC", "UBLKCP", "LOP3", "SHF"]


def main() -> int:
    so = build()
    out = subprocess.run(["cuobjdump", "-sass", so], capture_output=True, text=True, check=True).stdout
    print(f"# cuobjdump -sass {so.split('/root/repo/')[-1]} | per kernel: instruction count and counts of {', '.join(MNEMONICS)}")
    print("# written by: python tests/sass_excerpt.py")
    name, counts, total = None, {}, 0
    rows = []

    def flush():
        if name is not None:
            rows.append((name, total, dict(counts)))

    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            flush()
            name = subprocess.run(["c++filt", "-p", m.group(1)], capture_output=True, text=True).stdout.strip() or m.group(1)
            counts, total = {k: 0 for k in MNEMONICS}, 0
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and name is not None:
            total += 1
            op = m.group(1)
            for k in MNEMONICS:
                if op == k or op.startswith(k + ".") or (k in ("STG.E.EF.128", "IMAD.WIDE.U32", "STS.128") and op.startswith(k)):
                    counts[k] += 1
    flush()
    tot = {k: sum(r[2][k] for r in rows) for k in MNEMONICS}
    print(f"# {len(rows)} kernels; library totals: " + ", ".join(f"{k} {v}" for k, v in tot.items()))
    for name, total, c in sorted(rows):
        nz = ", ".join(f"{k} {v}" for k, v in c.items() if v)
        print(f"{name}: {total} instructions; {nz}")
    return 0


if __name__ == "__main__":
    sys.exit(main())
