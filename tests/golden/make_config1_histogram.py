"""Writes tests/golden/config1_histogram.txt from the ORACLE only (never from the CUDA path).

Usage: python tests/golden/make_config1_histogram.py
"""
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

from oracle import hec_oracle as O                      # noqa: E402
from paper_1805_11991_b200 import workloads as W        # noqa: E402

rows = W.generate(W.CONFIGS[1])
cnt, sf, _ = O.count(3, 2, rows)
tup, mult = O.histogram(cnt)
out = Path(__file__).resolve().parent / "config1_histogram.txt"
with out.open("w") as fh:
    fh.write("# N_1 N_2 multiplicity -- all 1944 f in F_3[x] of degree 5 or 6 (BASELINE.json config 1); "
             "written by make_config1_histogram.py from oracle/ (definition: PAPER.md:41-49, 63-69)\n")
    for t, m in zip(tup, mult):
        fh.write(f"{t[0]} {t[1]} {m}\n")
print(f"wrote {out} ({len(tup)} tuples)")
