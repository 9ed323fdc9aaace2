"""The comparator itself: it must flag what the north_star tolerances forbid and accept what they allow."""
import copy

import numpy as np

from oracle import oracle as O
from paper_2003_03174_b200 import parity as P, workloads as W


def _want():
    spec = W.CONFIGS["tiny"]; d = W.generate(spec)
    return O.match(W.matcher_config(spec), d)


def test_identical_result_passes_and_perturbations_fail():
    want = _want()
    got = {k: (v.astype(np.float32) if v.dtype == np.float64 else v.copy()) for k, v in want.items()
           if isinstance(v, np.ndarray)}
    assert P.compare(got, want)["ok"]
    robust = int(np.nonzero((want["margin"] > 1e-2) & (want["n_matched"] > 2))[0][0])
    g = copy.deepcopy(got); g["idx"][0, robust] = 123456
    r = P.compare(g, want); assert not r["ok"] and r["n_unexplained"] == 1 and r["unexplained_tracks"] == [robust]
    g = copy.deepcopy(got); g["par"][0, robust] *= 1.0 + 3e-4
    if abs(want["par"][0, robust]) > 0.1:
        assert P.compare(g, want)["n_par_bad"] == 1
    g = copy.deepcopy(got); g["chi2"][robust] *= 1.0 + 2e-3
    assert P.compare(g, want)["n_chi2_bad"] == 1
    g = copy.deepcopy(got); g["chi2"][robust] *= 1.0 + 5e-4
    assert P.compare(g, want)["ok"]
    g = copy.deepcopy(got); g["n_matched"][robust] += 1
    assert P.compare(g, want)["n_int_bad"] == 1
    g = copy.deepcopy(got); g["cov"][0, robust] *= 1.01
    assert P.compare(g, want)["n_cov_bad"] == 1


def test_a_flip_on_a_fragile_track_is_reported_but_allowed():
    want = _want()
    got = {k: (v.astype(np.float32) if v.dtype == np.float64 else v.copy()) for k, v in want.items()
           if isinstance(v, np.ndarray)}
    i = int(np.argmin(want["margin"]))
    want["margin"][i] = 1e-6
    got["idx"][2, i] = -1 if got["idx"][2, i] >= 0 else 7
    r = P.compare(got, want)
    assert r["ok"] and r["n_assign_mismatch"] == 1 and r["n_unexplained"] == 0
