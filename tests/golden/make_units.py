"""Writes tests/golden/units_timeframe.json: the oracle's operation counters (n_prop, n_rot, n_road, n_cand,
n_upd, and n_distinct_cand = distinct tracklets found inside some road) for each 500k-track batch of BASELINE.json configs[4] ("timeframe", seed 317405), i.e. the number of
algorithmic units one trd_match launch of bench.py processes.
Calls only oracle/ and the seeded input generator -- never the CUDA path.  Takes a few minutes of CPU.
    python tests/golden/make_units.py
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as O                                   # noqa: E402
from paper_2003_03174_b200 import workloads as W                 # noqa: E402


def main():
    spec = W.CONFIGS["timeframe"]
    d = W.generate(spec)
    cfg = W.matcher_config(spec)
    batches = []
    for lo in range(0, spec.n_tracks, spec.batch):
        r = O.match(cfg, d, lo=lo, hi=lo + spec.batch, count_distinct=True)
        c = dict(r["counters"]); c["n_tracks"] = spec.batch
        c["n_matched_ge2"] = int((r["n_matched"] >= 2).sum())
        c["n_fragile_1e-4"] = int((r["margin"] < 1e-4).sum())
        c["oracle_seconds"] = r["seconds"]
        batches.append(c)
        print(lo, c, flush=True)
    out = dict(config="timeframe", seed=spec.seed, n_tracks=spec.n_tracks, n_tracklets=int(d["tl_y"].shape[0]),
               n_hyp=spec.n_hyp, n_sigma_road=spec.n_sigma_road, batches=batches)
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "units_timeframe.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
