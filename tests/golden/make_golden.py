"""Writes tests/golden/tiny_oracle.txt: a few oracle outputs for BASELINE config 1 (Tiny).

Calls only oracle/ and the seeded input module; never the CUDA path.  Re-run after a justified
change to the oracle's arithmetic (the commit message must cite the passage / DESIGN.md reading).
    python tests/golden/make_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import ecei_synth as es  # noqa: E402
from oracle import delta_oracle as o  # noqa: E402

wl = es.WORKLOADS["tiny"]
r = o.analyze_chunk(es.tiny(), wl.nfft, wl.hop, wl.max_lag)
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle.txt")
with open(out, "w") as fh:
    fh.write("# oracle outputs for BASELINE.json configs[0] (Tiny), written by make_golden.py\n")
    fh.write("# quantity  row(pair or channel)  column(bin or lag index)  value\n")
    for name, ncol in (("G", 129), ("A", 129), ("P", 129), ("R", 257), ("Sauto", 129)):
        nrow = r[name].shape[0]
        for p in (0, nrow // 2, nrow - 1):
            for q in (0, 3, 10, 31, ncol // 2, ncol - 1):
                fh.write(f"{name} {p} {q} {r[name][p, q]!r}\n")
print("wrote", out)
