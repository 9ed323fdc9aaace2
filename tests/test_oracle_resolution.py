"""Pins of the oracle's measurement model with res_model = 1 (PAPER.md:62 + Fig. 3: sigma_y, sigma_dydx as
second-order polynomials of sin(phi) with the optimum at the Lorentz angle; pads tilted by +-2
degrees, correlated y-z errors, y corrected from the extrapolated z).  Readings R24-R26 of DESIGN.md."""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W


def model_cfg(base_cfg, **over):
    cfg = dict(base_cfg, res_model=1, sy_c0=W.SY_C0, sy_c2=W.SY_C2, sd_c0=W.SD_C0, sd_c2=W.SD_C2,
               sin_lorentz=W.sin_lorentz(0.5), tan_tilt=math.tan(math.radians(W.TILT_DEG)))
    cfg.update(over)
    return cfg


def rotated_R(cfg, s, layer):
    """R = Rot(tau) diag(sy^2, sz^2) Rot(tau)^T built from the rotation matrix (not from the closed form)."""
    ds = s - cfg["sin_lorentz"]
    sy = cfg["sy_c0"] + cfg["sy_c2"] * ds * ds
    tau = math.atan(cfg["tan_tilt"]) * (1 if layer % 2 == 0 else -1)
    u = np.array([math.cos(tau), -math.sin(tau)])        # across the pad (precise)
    v = np.array([math.sin(tau), math.cos(tau)])         # along the pad (coarse)
    return sy ** 2 * np.outer(u, u) + cfg["sigma_z"] ** 2 * np.outer(v, v), math.tan(tau)


def test_constant_coefficients_and_no_tilt_reduce_to_the_configs_model_bit_for_bit():
    spec = W.CONFIGS["central8"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d)
    b = O.match(dict(cfg, res_model=1, sy_c0=cfg["sigma_y"], sy_c2=0.0, sd_c0=cfg["sigma_dydx"], sd_c2=0.0,
                     sin_lorentz=0.3, tan_tilt=0.0), d)
    for k in ("idx", "par", "cov", "chi2", "n_matched", "n_evals", "margin"):
        np.testing.assert_array_equal(a[k], b[k])


@pytest.mark.parametrize("layer", [0, 1, 4, 5])
def test_chi2_and_road_against_rotation_matrix_and_corrected_residual(base_cfg, layer):
    """chi2 = r^T S^-1 r must equal the chi2 of the tilt-corrected residual r' = A r with covariance A S A^T, and
    the y road is n sigma of (A S A^T)_yy = C-part + sigma_y^2 (1 + tan^2): sigma_z drops out of the y road."""
    cfg = model_cfg(base_cfg)
    rng = np.random.default_rng(layer)
    for _ in range(20):
        s = rng.uniform(-0.6, 0.6)
        p = np.array([rng.uniform(-40, 40), rng.uniform(-300, 300), s, rng.uniform(-0.8, 0.8), rng.uniform(-1, 1)])
        L_ = rng.normal(size=(5, 5)) * np.array([0.05, 0.1, 1e-3, 1e-3, 1e-2])[:, None]
        Cm = L_ @ L_.T + np.diag([1e-4, 1e-3, 1e-8, 1e-8, 1e-6])
        c15 = O.full_to_tri(Cm)
        R, t = rotated_R(cfg, s, layer)
        S = Cm[:2, :2] + R
        A = np.array([[1.0, -t], [0.0, 1.0]])
        Sp = A @ S @ A.T
        rd = O.road(cfg, p, c15, layer)
        assert rd["road_y"] == pytest.approx(cfg["n_sigma_road"] * math.sqrt(Sp[0, 0]), rel=1e-12)
        ds = s - cfg["sin_lorentz"]; sy = cfg["sy_c0"] + cfg["sy_c2"] * ds * ds
        Cpart = Cm[0, 0] - 2 * t * Cm[1, 0] + t * t * Cm[1, 1]
        assert Sp[0, 0] == pytest.approx(Cpart + sy * sy * (1 + t * t), rel=1e-10)
        np.testing.assert_allclose(rd["Sinv"], np.linalg.inv(S), rtol=1e-10)
        # one tracklet inside the road: chi2 from the corrected residual
        ym = np.float32(p[0] + 0.3 * rd["road_y"] + t * 2.0); zm = np.float32(p[1] + 2.0)
        tanphi = s / math.sqrt(1 - s * s)
        tl = dict(tl_y=np.array([ym], np.float32), tl_z=np.array([zm], np.float32),
                  tl_dydx=np.array([tanphi], np.float32), tl_chamber=np.array([3 * 30 + layer], np.int32))
        idx, chi2 = O.candidates(dict(cfg, chi2_cut=1e9), tl, p, c15, sector=3, layer=layer, brute=True)
        r = np.array([float(ym) - p[0], float(zm) - p[1]])
        rp = A @ r
        if abs(rp[0]) <= rd["road_y"] and abs(r[1]) <= rd["road_z"]:
            assert idx.tolist() == [0]
            assert chi2[0] == pytest.approx(rp @ np.linalg.inv(Sp) @ rp, rel=1e-9)
            assert chi2[0] == pytest.approx(r @ np.linalg.inv(S) @ r, rel=1e-9)


def test_update_with_correlated_R_equals_information_form(base_cfg):
    cfg = model_cfg(base_cfg)
    rng = np.random.default_rng(3)
    for layer in (0, 1):
        s = 0.25
        p = np.array([3.0, -50.0, s, 0.4, 0.6])
        L_ = rng.normal(size=(5, 5)) * np.array([0.05, 0.1, 1e-3, 1e-3, 1e-2])[:, None]
        Cm = L_ @ L_.T + np.diag([1e-4, 1e-3, 1e-8, 1e-8, 1e-6])
        R, _ = rotated_R(cfg, s, layer)
        H = np.zeros((2, 5)); H[0, 0] = H[1, 1] = 1.0
        m = np.array([3.1, -48.0])
        p2, c2, chi2 = O.update(cfg, p, O.full_to_tri(Cm), m[0], m[1], layer)
        Cn = np.linalg.inv(np.linalg.inv(Cm) + H.T @ np.linalg.inv(R) @ H)
        pn = Cn @ (np.linalg.inv(Cm) @ p + H.T @ np.linalg.inv(R) @ m)
        np.testing.assert_allclose(O.tri_to_full(c2), Cn, rtol=1e-7, atol=1e-14)
        np.testing.assert_allclose(p2, pn, rtol=1e-9, atol=1e-12)
        r = m - p[:2]
        assert chi2 == pytest.approx(r @ np.linalg.inv(Cm[:2, :2] + R) @ r, rel=1e-10)


def test_optimum_at_the_lorentz_angle(base_cfg):
    """best resolution at the Lorentz angle (about +-8 degrees)."""
    cfg = model_cfg(base_cfg)
    c15 = O.full_to_tri(np.diag([1e-6, 1e-4, 1e-8, 1e-8, 1e-6]))
    roads = {s: O.road(cfg, [0, 0, s, 0, 0.1], c15, 0)["road_y"] for s in (cfg["sin_lorentz"] - 0.3, cfg["sin_lorentz"], cfg["sin_lorentz"] + 0.3)}
    sL = cfg["sin_lorentz"]
    assert roads[sL] < roads[sL - 0.3] and roads[sL] < roads[sL + 0.3]
    assert roads[sL - 0.3] == pytest.approx(roads[sL + 0.3], rel=1e-9)
    assert sL == pytest.approx(math.sin(math.radians(8.0)))


def test_pulls_and_chi2_with_the_model_on_and_sensitivity_to_the_tilt_sign():
    """Smeared input generated with the tilt and the sin(phi)-dependent resolutions, noise removed: <chi2> = 2 per
    matched layer and unit pulls.  With the tilt sign flipped in the matcher the chi2 degrades visibly, so the
    pin is sensitive to the sign convention shared by generator (R25) and oracle."""
    spec = dataclasses.replace(W.CONFIGS["central"], res_model=1, n_noise=0, efficiency=1.0, n_tracks=20000, number=12)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.match(cfg, d)
    ok = (r["n_matched"] == 6) & np.all(r["idx"].T == d["truth_idx"], axis=1)
    assert ok.mean() > 0.9
    chi2_per = r["chi2"][ok].sum() / (6 * ok.sum())
    assert chi2_per == pytest.approx(2.0, abs=0.05)
    # pulls of y and sin(phi) at the last layer against the truth helix there
    y_true, s_true = d["truth_last"][ok, 0], d["truth_last"][ok, 2]
    for k, truth in ((0, y_true), (2, s_true)):
        pull = (r["par"][k, ok] - truth) / np.sqrt(r["cov"][k * (k + 1) // 2 + k, ok])
        assert abs(pull.mean()) < 0.05 and pull.std() == pytest.approx(1.0, abs=0.06)
    wrong = O.match(dict(cfg, tan_tilt=-cfg["tan_tilt"]), d)
    okw = wrong["n_matched"] > 0
    assert wrong["chi2"][okw].sum() / wrong["n_matched"][okw].sum() > 1.5 * chi2_per


def test_sorted_index_equals_brute_force_with_the_model_on():
    spec = dataclasses.replace(W.CONFIGS["central8"], res_model=1)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d); b = O.match(cfg, d, brute=True)
    for k in ("idx", "par", "cov", "chi2", "n_matched", "n_evals"):
        np.testing.assert_array_equal(a[k], b[k])
