"""Pins of the oracle's TRD-only refit (PAPER.md:33 calibration step 3: refits "ignoring the TPC
clusters"; "a minimum of two tracklets").  Reading R31 of DESIGN.md."""
import dataclasses

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W


def test_refit_is_the_inward_composition_of_the_pinned_propagation_and_update():
    """Orchestration pin: covariance reset, inward order over the attached tracklets only, final step to x_ref --
    rebuilt here from the separately pinned propagate_to_layer and update."""
    spec = dataclasses.replace(W.CONFIGS["pileup"], n_tracks=400, n_noise=20000, n_hyp=2, chamber_dx_sigma=0.2, res_model=1)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    m = O.match(cfg, d); r = O.refit(cfg, d, m)
    n_checked = 0
    for i in range(spec.n_tracks):
        att = [l for l in range(6) if m["idx"][l, i] >= 0]
        if len(att) < 2:
            assert r["n_used"][i] == 0 and np.array_equal(r["par"][:, i], m["par"][:, i]) and r["x"][i] == m["x"][i]
            continue
        p = m["par"][:, i].copy(); c15 = O.full_to_tri(np.diag(O.REFIT_VAR)); x = float(m["x"][i]); sec = int(m["sector"][i])
        ok, chi2, used = True, 0.0, 0
        for l in reversed(att):
            k = int(m["idx"][l, i]); ch = int(d["tl_chamber"][k])
            X = cfg["layer_x"][l] + float(d["chamber_dx"][ch])
            if x != X:
                ok, p, c15, x, sec = O.propagate_to_layer(cfg, p, c15, x, sec, X)
            if not ok:
                break
            if ch // 30 != sec:
                continue
            p, c15, inc = O.update(cfg, p, c15, float(d["tl_y"][k]), float(d["tl_z"][k]), l)
            chi2 += inc; used += 1
            if abs(p[2]) >= cfg["max_snp"]:
                ok = False
        if ok:
            ok, p, c15, x, sec = O.propagate_to_layer(cfg, p, c15, x, sec, 247.0)
        if not ok:
            assert r["n_used"][i] == 0
            continue
        assert r["n_used"][i] == used and r["sector"][i] == sec and r["x"][i] == 247.0
        np.testing.assert_allclose(r["par"][:, i], p, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(r["cov"][:, i], c15, rtol=1e-10, atol=1e-18)
        assert r["chi2"][i] == pytest.approx(chi2, rel=1e-12)
        n_checked += 1
    assert n_checked > 300


def test_noise_free_chains_give_back_the_true_track_at_the_reference_plane():
    spec = dataclasses.replace(W.CONFIGS["central"], smear_seed=False, smear_tracklets=False, exact_z=True, efficiency=1.0,
                               n_noise=0, n_tracks=3000, number=18)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.refit(cfg, d, O.match(cfg, d))
    ok = (r["n_used"] == 6) & (r["sector"] == d["sector"])
    assert ok.mean() > 0.9 and np.all(r["x"][ok] == 247.0)
    np.testing.assert_allclose(r["par"][:, ok], d["truth_par"][:, ok], rtol=0, atol=1e-4)     # float32 tracklets
    assert r["chi2"][ok].max() < 1e-6


def test_pulls_at_the_reference_plane_and_independence_from_the_seed():
    spec = dataclasses.replace(W.CONFIGS["central"], n_noise=0, efficiency=1.0, n_tracks=20000, number=17)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    m = O.match(cfg, d); r = O.refit(cfg, d, m)
    ok = (r["n_used"] == 6) & (r["sector"] == d["sector"])
    assert ok.mean() > 0.9
    for k in (0, 2, 4):                                  # y, sin(phi), q/pT: Gaussian measurement errors
        pull = (r["par"][k, ok] - d["truth_par"][k, ok]) / np.sqrt(r["cov"][k * (k + 1) // 2 + k, ok])
        assert abs(pull.mean()) < 0.05 and pull.std() == pytest.approx(1.0, abs=0.06)
    # "ignoring the TPC": the refit's errors are the TRD's own, far larger than the seeded track's at the same plane
    assert np.sqrt(r["cov"][0, ok]).mean() > 1.5 * 0.1
    # and a different (worse) seed covariance in the matcher output does not change the refit
    m2 = dict(m); m2["cov"] = m["cov"] * 7.0
    r2 = O.refit(cfg, d, m2)
    np.testing.assert_array_equal(r2["par"], r["par"])


def test_fewer_than_two_tracklets_pass_through():
    spec = dataclasses.replace(W.CONFIGS["tiny"], efficiency=0.25, n_noise=0, number=19)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    m = O.match(cfg, d); r = O.refit(cfg, d, m)
    few = m["n_matched"] < 2
    assert few.sum() > 100
    assert np.all(r["n_used"][few] == 0) and np.array_equal(r["par"][:, few], m["par"][:, few])
    assert np.array_equal(r["cov"][:, few], m["cov"][:, few]) and np.array_equal(r["x"][few], m["x"][few])
    assert np.all(r["n_used"][~few] >= 0)
