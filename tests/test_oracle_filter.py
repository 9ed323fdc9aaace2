"""Pins of the oracle's Kalman update and of the whole chain."""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W

RNG = np.random.default_rng(777)


def random_cov():
    A = RNG.normal(size=(5, 5)) * np.array([0.1, 0.1, 1e-3, 1e-3, 1e-2])[:, None]
    return A @ A.T + np.diag([1e-4, 1e-4, 1e-8, 1e-8, 1e-6])


def test_update_equals_information_form(base_cfg):
    """Gain form == (C^-1 + H^T R^-1 H)^-1 and its mean, computed with numpy.linalg."""
    H = np.zeros((2, 5)); H[0, 0] = H[1, 1] = 1.0
    Rm = np.diag([base_cfg["sigma_y"] ** 2, base_cfg["sigma_z"] ** 2])
    for _ in range(100):
        Cm = random_cov(); p = RNG.normal(size=5); m = p[:2] + RNG.normal(size=2) * [0.1, 2.0]
        q, c15, chi2 = O.update(base_cfg, p, O.full_to_tri(Cm), m[0], m[1])
        Ci = np.linalg.inv(Cm)
        Cpost = np.linalg.inv(Ci + H.T @ np.linalg.inv(Rm) @ H)
        ppost = Cpost @ (Ci @ p + H.T @ np.linalg.solve(Rm, m))
        np.testing.assert_allclose(O.tri_to_full(c15), Cpost, rtol=1e-7, atol=1e-16)
        np.testing.assert_allclose(q, ppost, rtol=1e-8, atol=1e-10)
        r = m - p[:2]
        assert chi2 == pytest.approx(r @ np.linalg.solve(Cm[:2, :2] + Rm, r), rel=1e-10)
        # information never decreases: det and trace shrink, matrix stays positive definite
        assert np.linalg.det(Cpost) < np.linalg.det(Cm) and np.trace(O.tri_to_full(c15)) < np.trace(Cm)
        np.linalg.cholesky(O.tri_to_full(c15))


def test_update_one_dimensional_weighted_mean(base_cfg):
    """Diagonal covariance: y is the inverse-variance weighted mean, untouched components stay."""
    c = np.diag([0.09, 4.0, 1e-6, 1e-6, 1e-4]); p = np.array([1.0, 10.0, 0.1, 0.2, 0.3])
    q, c15, chi2 = O.update(base_cfg, p, O.full_to_tri(c), 1.5, 12.0)
    sy2, sz2 = base_cfg["sigma_y"] ** 2, base_cfg["sigma_z"] ** 2
    assert q[0] == pytest.approx((1.0 / 0.09 + 1.5 / sy2) / (1 / 0.09 + 1 / sy2), rel=1e-12)
    assert q[1] == pytest.approx((10.0 / 4.0 + 12.0 / sz2) / (1 / 4.0 + 1 / sz2), rel=1e-12)
    assert np.array_equal(q[2:], p[2:])
    assert O.tri_to_full(c15)[0, 0] == pytest.approx(1 / (1 / 0.09 + 1 / sy2), rel=1e-12)
    assert chi2 == pytest.approx(0.25 / (0.09 + sy2) + 4.0 / (4.0 + sz2), rel=1e-12)


def test_six_updates_equal_batch_least_squares(base_cfg):
    """Bz = 0 and tiny angles make the model linear (y' = y + dx s, z' = z + dx t up to O(s^2) ~ 1e-10);
    six propagate+update steps must equal the generalised least-squares fit of all six measurements with
    the seed as a Gaussian prior, solved as one stacked system with numpy.linalg.lstsq."""
    cfg = dict(base_cfg, bz_tesla=0.0)
    xs = np.array(cfg["layer_x"]); x0 = 247.0
    p0 = np.array([1.0, -5.0, 2e-5, -3e-5, 0.7]); C0 = np.diag([0.01, 0.01, 1e-6, 1e-6, 1e-4])
    meas = np.stack([p0[0] + (xs - x0) * p0[2] + RNG.normal(size=6) * 0.04,
                     p0[1] + (xs - x0) * p0[3] + RNG.normal(size=6) * 2.3], axis=1)
    p, c15, x = p0.copy(), O.full_to_tri(C0), x0
    chi2 = 0.0
    for L in range(6):
        ok, p, c15, x = O.propagate(cfg, p, c15, x, xs[L]); assert ok
        p, c15, inc = O.update(cfg, p, c15, meas[L, 0], meas[L, 1]); chi2 += inc
    # unknowns: state at the LAST plane (y, z, s, t); rows whitened by their sigma
    xl = xs[-1]; rows, rhs = [], []
    for i, sg in enumerate(np.sqrt(np.diag(C0))[:4]):              # prior on the state at x0
        a = np.zeros(4); a[i] = 1.0
        if i < 2: a[i + 2] = x0 - xl
        rows.append(a / sg); rhs.append(p0[i] / sg)
    for L in range(6):
        for i, sg in ((0, cfg["sigma_y"]), (1, cfg["sigma_z"])):
            a = np.zeros(4); a[i] = 1.0; a[i + 2] = xs[L] - xl
            rows.append(a / sg); rhs.append(meas[L, i] / sg)
    A = np.array(rows); bvec = np.array(rhs)
    sol, res, *_ = np.linalg.lstsq(A, bvec, rcond=None)
    np.testing.assert_allclose(p[:4], sol, rtol=0, atol=2e-8)
    np.testing.assert_allclose(O.tri_to_full(c15)[:4, :4], np.linalg.inv(A.T @ A), rtol=1e-6, atol=1e-14)
    assert chi2 == pytest.approx(float(res[0]), rel=1e-6)         # sum of increments == minimum of the GLS chi2


def _variant(name, **kw):
    return dataclasses.replace(W.CONFIGS[name], **kw)


def test_noise_free_chain_recovers_truth_exactly():
    """Unsmeared seed, unsmeared tracklets with exact z, no noise, 100 % efficiency: every layer is
    matched to the track's own tracklet, chi2 ~ 0 and the state at layer 5 is the true helix."""
    spec = _variant("tiny", n_noise=0, smear_seed=False, smear_tracklets=False, exact_z=True, efficiency=1.0)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.match(cfg, d)
    ti = d["truth_idx"]                                  # (n, 6)
    np.testing.assert_array_equal(r["idx"].T, ti)
    full = (ti >= 0).all(axis=1)
    assert full.sum() > 700
    assert r["chi2"].max() < 1e-6                        # inputs are float32-rounded truth: residual ~ 4e-6 cm
    last = d["truth_last"]
    sel = full & (r["sector"] == last[:, 3].astype(int))
    assert sel.sum() == full.sum()
    assert np.abs(r["par"][0][sel] - last[sel, 0]).max() < 2e-5
    assert np.abs(r["par"][1][sel] - last[sel, 1]).max() < 2e-4
    assert np.abs(r["par"][2][sel] - last[sel, 2]).max() < 1e-6
    assert np.all(r["x"][full] == 364.0)


def test_smeared_chain_has_unit_pulls_and_chi2_equal_ndf():
    """Signal only: <chi2_inc> = 2 per matched layer; pulls of all five parameters at the last layer
    have mean 0 and width 1 (the z measurement error is uniform, its variance is still pad^2/12)."""
    spec = _variant("central", n_noise=0, n_tracks=20000)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.match(cfg, d)
    assert r["chi2"].sum() / r["n_matched"].sum() == pytest.approx(2.0, abs=0.03)
    last = d["truth_last"]
    sel = (r["n_matched"] == 6) & (r["sector"] == np.nan_to_num(last[:, 3], nan=-1).astype(int)) & (r["x"] == 364.0)
    sel &= (r["idx"].T == d["truth_idx"]).all(axis=1)      # correctly associated tracks only (no fakes from neighbours)
    assert sel.sum() > 8000
    truth5 = np.stack([last[:, 0], last[:, 1], last[:, 2], d["truth_par"][3], d["truth_par"][4]])
    diag = [0, 2, 5, 9, 14]
    for i in range(5):
        pull = (r["par"][i][sel] - truth5[i][sel]) / np.sqrt(r["cov"][diag[i]][sel])
        assert abs(pull.mean()) < 0.04, (i, pull.mean())
        assert pull.std() == pytest.approx(1.0, abs=0.05), (i, pull.std())


def test_purity_falls_with_density():
    """purity ~ 1 at low density and lower at high density (configs 1 >= 2 >= 4)."""
    pur = []
    for name in ("tiny", "central", "pileup"):
        spec = W.CONFIGS[name]; d = W.generate(spec)
        r = O.match(W.matcher_config(spec), d)
        q = W.efficiency_purity(r["idx"].T, d)
        assert q["efficiency"] > 0.98
        pur.append(q["purity"])
    assert pur[0] >= pur[1] >= pur[2] > 0.95


def test_low_pt_tracks_do_not_reach_the_trd():
    """primaries below ~0.3 GeV/c never reach the TRD: 2R < 364 cm at 0.5 T for pT < 0.273."""
    pt = 0.27; radius = pt / (0.00299792458 * 0.5)
    assert 2 * radius < W.LAYER_X[-1]
    d = W.generate(W.CONFIGS["pileup"])
    assert (1.0 / np.abs(d["truth_par"][4])).min() >= 0.3
