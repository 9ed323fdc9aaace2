"""Writes tests/golden/oracle_tiny.txt: the oracle's result for the first 48 tracks of config 1
("tiny", seed 317401).  Calls only oracle/ and the seeded input generator -- never the CUDA path.

The paper prints no worked example (PAPER.md has no numeric table for the tracker), so this fixture
is NOT a pin of the oracle against the paper; it freezes the oracle's own output so that an
unintended change of its arithmetic shows up as a diff.  Re-run only together with a commit that
names the passage or DESIGN.md reading that justifies the change:
    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as O                                   # noqa: E402
from paper_2003_03174_b200 import workloads as W                 # noqa: E402

N = 48


def table():
    spec = W.CONFIGS["tiny"]
    d = W.generate(spec)
    r = O.match(W.matcher_config(spec), d, hi=N)
    rows = []
    for i in range(N):
        rows.append(" ".join([str(i)] + [str(int(v)) for v in r["idx"][:, i]] + [str(int(r["n_matched"][i])),
                             str(int(r["sector"][i]))] + [f"{v:.12e}" for v in [r["chi2"][i], *r["par"][:, i]]]))
    return "# track idx0..idx5 n_matched sector chi2 y z sinphi tanlambda q/pT   (oracle, config tiny, seed 317401)\n" \
        + "\n".join(rows) + "\n"


if __name__ == "__main__":
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny.txt"), "w") as f:
        f.write(table())
