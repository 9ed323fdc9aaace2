"""Pins of the oracle's road search and top-N selection: brute force on
small inputs, an independently written greedy matcher, exhaustive enumeration of all chains."""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W

SKIP = np.iinfo(np.int32).max


def dense_spec(n_tracks=40, n_noise=60000, n_hyp=4, road=3.0, number=1):
    """Few tracks, very dense noise: several in-road candidates per layer."""
    return dataclasses.replace(W.CONFIGS["tiny"], name="dense", number=number, n_tracks=n_tracks,
                               n_noise=n_noise, n_hyp=n_hyp, n_sigma_road=road)


@pytest.mark.parametrize("name", ["tiny", "central8"])
def test_sorted_index_equals_loop_over_all_tracklets(name):
    spec = W.CONFIGS[name]; d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d); b = O.match(cfg, d, brute=True)
    for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
        np.testing.assert_array_equal(a[k], b[k])
    assert a["counters"]["n_cand"] == b["counters"]["n_cand"]
    assert a["counters"]["n_scanned"] < b["counters"]["n_scanned"]


def test_threads_do_not_change_results():
    spec = W.CONFIGS["central8"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d, n_threads=1); b = O.match(cfg, d, n_threads=4)
    for k in ("idx", "par", "cov", "chi2", "n_matched", "n_evals", "margin"):
        np.testing.assert_array_equal(a[k], b[k])
    assert a["counters"] == b["counters"]


def test_inclination_is_a_veto_not_a_chi2_term(base_cfg):
    """only y and z enter chi2; the tracklet slope only excludes beyond 4 sigma."""
    p = np.array([5.0, 20.0, 0.1, 0.3, 0.5]); c15 = O.full_to_tri(np.diag([0.01, 0.02, 1e-6, 1e-6, 1e-4]))
    tanphi = 0.1 / math.sqrt(1 - 0.01)
    lim = base_cfg["n_sigma_angle"] * base_cfg["sigma_dydx"]
    tl = dict(tl_y=np.array([5.05] * 4, np.float32), tl_z=np.array([20.0] * 4, np.float32),
              tl_dydx=np.array([tanphi, tanphi + 0.9 * lim, tanphi - 0.99 * lim, tanphi + 1.01 * lim], np.float32),
              tl_chamber=np.array([3 * 30 + 2 * 6 + 1] * 4, np.int32))
    idx, chi2 = O.candidates(base_cfg, tl, p, c15, sector=3, layer=1)
    assert idx.tolist() == [0, 1, 2]
    assert chi2[0] == chi2[1] == chi2[2]
    rd = O.road(base_cfg, p, c15)
    ry = float(np.float32(5.05)) - 5.0
    assert chi2[0] == pytest.approx(ry * ry / (0.01 + base_cfg["sigma_y"] ** 2), rel=1e-12)
    assert rd["road_y"] == pytest.approx(3 * math.sqrt(0.01 + 0.04 ** 2), rel=1e-12)
    assert rd["road_z"] == pytest.approx(3 * math.sqrt(0.02) + 4.0, rel=1e-12)
    # other sector / other layer / outside the windows / beyond the cut: not candidates
    tl2 = dict(tl_y=np.array([5.05, 5.05, 5.0 + 1.01 * rd["road_y"], 5.0, 5.0 + 0.99 * rd["road_y"]], np.float32),
               tl_z=np.array([20.0, 20.0, 20.0, 20.0 + 1.01 * rd["road_z"], 20.0], np.float32),
               tl_dydx=np.full(5, tanphi, np.float32),
               tl_chamber=np.array([4 * 30 + 1, 3 * 30 + 2, 3 * 30 + 1, 3 * 30 + 1, 3 * 30 + 6 + 1], np.int32))
    idx, chi2 = O.candidates(base_cfg, tl2, p, c15, sector=3, layer=1)
    assert idx.tolist() == [4]                       # any stack of the right sector and layer counts [R12]
    assert chi2[0] < base_cfg["chi2_cut"]
    idx, _ = O.candidates(dict(base_cfg, chi2_cut=5.0), tl2, p, c15, sector=3, layer=1)
    assert idx.tolist() == []                        # (0.99 * 3 sigma)^2 = 8.8 >= 5


def greedy_reference(cfg, d, i):
    """nHyp = 1 written independently (about 30 lines): follow the single best candidate, else skip."""
    p = d["par"][:, i].astype(float); c15 = d["cov"][:, i].astype(float)
    x = float(d["x"][i]); sec = int(d["sector"][i]); alive = abs(p[2]) < cfg["max_snp"]
    idx = [-1] * 6; chi2 = 0.0
    for L in range(6):
        if not alive:
            continue
        ok, p2, c2, x2, sec2 = O.propagate_to_layer(cfg, p, c15, x, sec, cfg["layer_x"][L])
        if not ok:
            alive = False
            continue
        p, c15, x, sec = p2, c2, x2, sec2
        ci, cc = O.candidates(cfg, d, p, c15, sec, L, brute=True)
        if len(ci) == 0:
            continue
        k = np.lexsort((ci, cc))[0]
        p, c15, inc = O.update(cfg, p, c15, float(d["tl_y"][ci[k]]), float(d["tl_z"][ci[k]]))
        idx[L] = int(ci[k]); chi2 += inc
        alive = abs(p[2]) < cfg["max_snp"]
    return idx, chi2, p


def test_single_hypothesis_equals_greedy_matcher():
    spec = dataclasses.replace(W.CONFIGS["pileup"], n_tracks=300, n_noise=30000, n_hyp=1)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.match(cfg, d)
    for i in range(spec.n_tracks):
        idx, chi2, p = greedy_reference(cfg, d, i)
        assert r["idx"][:, i].tolist() == idx
        assert r["chi2"][i] == pytest.approx(chi2, rel=1e-12, abs=1e-12)
        np.testing.assert_allclose(r["par"][:, i], p, rtol=1e-12, atol=1e-12)


def enumerate_chains(cfg, d, i):
    """Depth-first enumeration of ALL chains of track i: at each layer every accepted candidate of the
    chain's own propagated state, or skip.  Returns the sorted list of (score, idx tuple)."""
    out = []

    def rec(L, p, c15, x, sec, alive, score, idx):
        if L == 6:
            out.append((score, tuple(idx)))
            return
        if alive:
            ok, p2, c2, x2, sec2 = O.propagate_to_layer(cfg, p, c15, x, sec, cfg["layer_x"][L])
            if ok:
                p, c15, x, sec = p2, c2, x2, sec2
                ci, cc = O.candidates(cfg, d, p, c15, sec, L, brute=True)
                for k in range(len(ci)):
                    pn, cn, inc = O.update(cfg, p, c15, float(d["tl_y"][ci[k]]), float(d["tl_z"][ci[k]]))
                    rec(L + 1, pn, cn, x, sec, abs(pn[2]) < cfg["max_snp"], score + inc, idx + [int(ci[k])])
            else:
                alive = False
        rec(L + 1, p, c15, x, sec, alive, score + cfg["chi2_penalty"], idx + [-1])

    rec(0, d["par"][:, i].astype(float), d["cov"][:, i].astype(float), float(d["x"][i]), int(d["sector"][i]),
        abs(float(d["par"][2, i])) < cfg["max_snp"], 0.0, [])
    out.sort()
    return out


def test_beam_search_against_exhaustive_enumeration():
    """With nHyp >= number of chains the beam search is exhaustive and must return the global optimum;
    with the configs' nHyp = 8 / 4 the optimum survives the pruning on these inputs (north_star)."""
    spec = dense_spec(n_tracks=30, n_noise=40000)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    big = O.match(dict(cfg, n_hyp=4096), d)
    r8 = O.match(dict(cfg, n_hyp=8), d); r4 = O.match(dict(cfg, n_hyp=4), d); r1 = O.match(dict(cfg, n_hyp=1), d)
    n_multi = 0; kept8 = kept4 = kept1 = 0
    for i in range(spec.n_tracks):
        chains = enumerate_chains(cfg, d, i)
        assert len(chains) <= 4096
        n_multi += len(chains) > 8
        best_score, best_idx = chains[0]
        assert tuple(big["idx"][:, i].tolist()) == best_idx
        n_skip = sum(1 for t in best_idx if t < 0)
        assert big["chi2"][i] + cfg["chi2_penalty"] * n_skip == pytest.approx(best_score, rel=1e-12, abs=1e-12)
        kept8 += tuple(r8["idx"][:, i].tolist()) == best_idx
        kept4 += tuple(r4["idx"][:, i].tolist()) == best_idx
        kept1 += tuple(r1["idx"][:, i].tolist()) == best_idx
    assert n_multi >= 10                 # the input really has combinatorics
    assert kept8 == spec.n_tracks and kept4 == spec.n_tracks
    assert kept1 >= spec.n_tracks - 6    # greedy may lose the optimum; that is why hypotheses are kept


def test_output_conventions():
    """chi2 excludes penalties, n_matched counts attached layers, a dead seed only skips."""
    spec = W.CONFIGS["tiny"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    d = dict(d); d["par"] = d["par"].copy(); d["par"][2, 0] = 0.96            # |sin(phi)| >= max_snp
    d["sector"] = d["sector"].copy(); d["sector"][1] = 99                     # not a sector
    r = O.match(cfg, d)
    for i in (0, 1):
        assert r["idx"][:, i].tolist() == [-1] * 6 and r["n_matched"][i] == 0 and r["chi2"][i] == 0.0
        assert r["x"][i] == 247.0
        np.testing.assert_array_equal(r["par"][:, i], d["par"][:, i].astype(float))
    np.testing.assert_array_equal(r["n_matched"], (r["idx"] >= 0).sum(axis=0))
    assert np.all(r["margin"] >= 0)


def test_oracle_output_is_frozen():
    """tests/golden/oracle_tiny.txt (written by tests/golden/make_golden.py from the oracle alone)."""
    import os
    here = os.path.dirname(os.path.abspath(__file__))
    want = [l.split() for l in open(os.path.join(here, "golden", "oracle_tiny.txt")) if not l.startswith("#")]
    spec = W.CONFIGS["tiny"]; d = W.generate(spec)
    r = O.match(W.matcher_config(spec), d, hi=len(want))
    for i, row in enumerate(want):
        assert [int(v) for v in row[1:7]] == r["idx"][:, i].tolist()
        assert int(row[7]) == r["n_matched"][i] and int(row[8]) == r["sector"][i]
        got = [r["chi2"][i], *r["par"][:, i]]
        np.testing.assert_allclose([float(v) for v in row[9:]], got, rtol=1e-9, atol=1e-12)
