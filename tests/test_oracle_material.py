"""Pins of the oracle's material step (second half: "energy loss and multiple scattering as
process noise", C' = F C F^T + Q; "taking into account ... energy loss").  Readings R32-R34 of DESIGN.md."""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W

M = W.PION_MASS
DIAG = [0, 2, 5, 9, 14]


def _cfg(base_cfg, **kw):
    return dict(dict(base_cfg, mass=M), **kw)


def _random_states(rng, n):
    for _ in range(n):
        p = np.array([rng.uniform(-20, 20), rng.uniform(-300, 300), rng.uniform(-0.7, 0.7), rng.uniform(-0.9, 0.9),
                      rng.choice([-1.0, 1.0]) / math.exp(rng.uniform(math.log(0.3), math.log(20.0)))])
        a = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 1e-3, 1e-3, 0.01 * abs(p[4])])[:, None]
        yield p, O.full_to_tri(a @ a.T + np.diag([1e-4, 1e-4, 1e-8, 1e-8, 1e-8]))


def test_scattering_noise_is_the_geometry_of_two_small_angles(base_cfg):
    """Q from first principles: the unit direction d = (cos phi cos lam, sin phi cos lam, sin lam) is tilted by two
    independent angles of variance theta0^2 about two orthonormal axes perpendicular to it, |p| fixed; (s, t, c) are
    read back from the tilted vector and differentiated numerically.  theta0 is Highland's width for the path
    1 / d_x through a slab normal to x."""
    cfg = _cfg(base_cfg, x_over_x0=0.037, eloss=0.0)
    rng = np.random.default_rng(1)
    for p, c15 in _random_states(rng, 200):
        ok, p1, c1 = O.material(cfg, p, c15, +1)
        assert ok and np.array_equal(p1, p)                       # scattering alone moves nothing
        dQ = O.tri_to_full(c1) - O.tri_to_full(c15)
        phi, lam = math.asin(p[2]), math.atan(p[3])
        d = np.array([math.cos(phi) * math.cos(lam), math.sin(phi) * math.cos(lam), math.sin(lam)])
        e1 = np.array([-math.cos(phi) * math.sin(lam), -math.sin(phi) * math.sin(lam), math.cos(lam)])
        e2 = np.array([-math.sin(phi), math.cos(phi), 0.0])
        assert abs(d @ e1) < 1e-14 and abs(d @ e2) < 1e-14 and abs(e1 @ e2) < 1e-14
        mom = math.sqrt(1 + p[3] ** 2) / abs(p[4])
        q = math.copysign(1.0, p[4])

        def stc(v):
            v = v / np.linalg.norm(v)
            tr = math.hypot(v[0], v[1])
            return np.array([v[1] / tr, v[2] / tr, q / (mom * tr)])
        eps = 1e-6
        J = np.stack([(stc(d + eps * e) - stc(d - eps * e)) / (2 * eps) for e in (e1, e2)], axis=1)   # 3 x 2
        beta = mom / math.hypot(mom, M)
        theta0 = 0.0136 / (beta * mom) * math.sqrt(0.037 / d[0])
        want = np.zeros((5, 5))
        want[2:, 2:] = theta0 ** 2 * J @ J.T
        np.testing.assert_allclose(dQ, want, rtol=2e-7, atol=1e-9 * theta0 ** 2 * (1 + p[4] ** 2))


def test_energy_loss_moves_the_energy_and_nothing_else(base_cfg):
    cfg = _cfg(base_cfg, x_over_x0=0.0, eloss=2.5e-3, eloss_fluct=0.0)
    rng = np.random.default_rng(2)

    def energy(p):
        return math.hypot(math.sqrt(1 + p[3] ** 2) / abs(p[4]), M)
    for p, c15 in _random_states(rng, 200):
        mom = math.sqrt(1 + p[3] ** 2) / abs(p[4])
        beta = mom / math.hypot(mom, M)
        path = 1.0 / (math.cos(math.asin(p[2])) * math.cos(math.atan(p[3])))
        dE = 2.5e-3 * path / beta ** 2
        for direction in (+1, -1):
            ok, p1, c1 = O.material(cfg, p, c15, direction)
            assert ok and np.array_equal(p1[:4], p[:4]) and p1[4] * p[4] > 0      # position, direction, charge kept
            assert np.array_equal(c1, c15)                                         # no fluctuation, no scattering: C kept
            assert energy(p1) == pytest.approx(energy(p) - direction * dE, rel=1e-12)
    # textbook limit: beta -> 1 at normal incidence, pT drops by exactly eloss
    p = np.array([0.0, 0.0, 0.0, 0.0, 1.0 / 5000.0])
    ok, p1, _ = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2.5e-3, mass=0.0), p, np.zeros(15), +1)
    assert ok and 1.0 / p1[4] == pytest.approx(5000.0 - 2.5e-3, rel=1e-13)
    # a particle that cannot pay the loss stops: state untouched
    slow = np.array([0.0, 0.0, 0.0, 0.0, 1.0 / 0.02])
    ok, p1, c1 = O.material(_cfg(base_cfg, x_over_x0=0.01, eloss=0.05), slow, np.full(15, 0.5), +1)
    assert not ok and np.array_equal(p1, slow) and np.all(c1 == 0.5)


def test_energy_loss_fluctuation_is_the_derivative_of_the_mean_correction(base_cfg):
    """sigma(c) = |dc/dE| sigma_E: the derivative is taken numerically through the pinned mean correction (the loss
    scaled up and down by the relative width), which a wrong dc/dE = c E / p^2 would not match."""
    f = 1e-4
    rng = np.random.default_rng(3)
    for p, c15 in _random_states(rng, 100):
        lo = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2e-3 * (1 - f)), p, c15, +1)[1][4]
        hi = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2e-3 * (1 + f)), p, c15, +1)[1][4]
        _, _, c1 = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2e-3, eloss_fluct=f), p, c15, +1)
        dq = c1 - c15
        assert np.all(dq[:14] == 0.0)
        mom = math.sqrt(1 + p[3] ** 2) / abs(p[4])
        assert math.sqrt(dq[14]) == pytest.approx(abs(hi - lo) / 2, rel=0.05 + 0.2 / mom ** 2 * 2e-3)
        # exact to first order in dE / E: compare at a tenth of the loss as well
    p = np.array([0.0, 0.0, 0.1, 0.3, 1.0 / 2.0]); c15 = np.zeros(15)
    lo = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2e-5 * (1 - f)), p, c15, +1)[1][4]
    hi = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2e-5 * (1 + f)), p, c15, +1)[1][4]
    c1 = O.material(_cfg(base_cfg, x_over_x0=0.0, eloss=2e-5, eloss_fluct=f), p, c15, +1)[2]
    assert math.sqrt(c1[14]) == pytest.approx((hi - lo) / 2, rel=1e-4)


def test_no_material_is_the_plain_matcher_bit_for_bit():
    spec = W.CONFIGS["central8"]
    d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d)
    b = O.match(dict(cfg, x_over_x0=0.0, eloss=0.0, eloss_fluct=0.3, mass=0.5), d)
    for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
        np.testing.assert_array_equal(a[k], b[k])
    ra, rb = O.refit(cfg, d, a), O.refit(dict(cfg, x_over_x0=0.0, eloss=0.0), d, a)
    for k in ra:
        np.testing.assert_array_equal(ra[k], rb[k])


def test_the_slab_is_crossed_after_the_propagation_and_before_the_road(base_cfg):
    """Orchestration pin on one track and one tracklet: the first layer's result equals pinned propagate_to_layer ->
    pinned material -> pinned update, and the road is the wider one."""
    cfg = _cfg(dict(base_cfg, n_hyp=1), x_over_x0=0.05, eloss=2e-3, eloss_fluct=0.3)
    p0 = np.array([1.0, 10.0, 0.05, 0.2, 1.0 / 0.6], np.float32).astype(float)
    c0 = O.full_to_tri(np.diag(np.array([0.01, 0.01, 1e-6, 1e-6, 1e-4], np.float32).astype(float)))
    ok, p1, c1, x1, sec = O.propagate_to_layer(cfg, p0, c0, 247.0, 4, 300.0)
    ok2, p2, c2 = O.material(cfg, p1, c1, +1)
    assert ok and ok2 and sec == 4
    y_m, z_m = np.float32(p2[0] + 0.03), np.float32(W.pad_row_centre(p2[1]))
    tl = dict(tl_y=np.array([y_m], np.float32), tl_z=np.array([z_m], np.float32),
              tl_dydx=np.array([p2[2] / math.sqrt(1 - p2[2] ** 2)], np.float32), tl_chamber=np.array([4 * 5 + 2], np.int32))   # one layer: 5 chambers per sector
    data = dict(tl, par=p0.astype(np.float32)[:, None], cov=c0.astype(np.float32)[:, None], x=np.array([247.0], np.float32),
                sector=np.array([4], np.int32))
    cfg1 = dict(cfg, n_layers=1)
    r = O.match(cfg1, data)
    p3, c3, chi2 = O.update(cfg1, p2, c2, float(y_m), float(z_m), 0)
    assert r["n_matched"][0] == 1
    np.testing.assert_allclose(r["par"][:, 0], p3, rtol=1e-13)
    np.testing.assert_allclose(r["cov"][:, 0], c3, rtol=1e-12)
    assert r["chi2"][0] == pytest.approx(chi2, rel=1e-12)
    assert O.road(cfg, p2, c2)["road_y"] == O.road(cfg, p1, c1)["road_y"]              # position block untouched by a thin slab
    assert c2[5] > c1[5] and c2[9] > c1[9] and abs(p2[4]) > abs(p1[4])


@pytest.fixture(scope="module")
def scattered():
    spec = dataclasses.replace(W.CONFIGS["pileup"], n_tracks=20000, n_noise=0, n_hyp=1, efficiency=1.0, number=19,
                               x_over_x0=W.X_OVER_X0, eloss=W.ELOSS, eloss_fluct=W.ELOSS_FLUCT)
    return spec, W.generate(spec), W.matcher_config(spec)


def _pulls(cfg, d):
    r = O.match(cfg, d)
    ok = (r["n_matched"] == 6) & np.all(r["idx"].T == d["truth_idx"], axis=1) & (r["sector"] == d["truth_last"][:, 3])
    tp = d["truth_last_par"]
    width = [float(((r["par"][k, ok] - tp[k, ok]) / np.sqrt(r["cov"][DIAG[k], ok])).std()) for k in range(5)]
    mean = [float(((r["par"][k, ok] - tp[k, ok]) / np.sqrt(r["cov"][DIAG[k], ok])).mean()) for k in range(5)]
    return r, ok, width, mean


def test_unit_pulls_of_all_five_parameters_on_scattered_particles(scattered):
    """The generator scatters and slows the true particle in every slab (its own small-angle kicks on the global
    direction); with the same material in the filter all five pulls at the last layer are unit width and
    <chi2> = ndf, which fails for a dropped Q term, a missing path or 1/beta factor or a wrong sign of the loss."""
    spec, d, cfg = scattered
    r, ok, width, mean = _pulls(cfg, d)
    assert ok.mean() > 0.85
    assert r["chi2"][ok].sum() / (12 * ok.sum()) == pytest.approx(1.0, abs=0.04)
    for k in range(5):
        assert width[k] == pytest.approx(1.0, abs=0.06) and abs(mean[k]) < 0.03


def test_sensitivity_of_the_pulls_to_every_ingredient(scattered):
    spec, d, cfg = scattered
    _, ok0, w_none, _ = _pulls(dict(cfg, x_over_x0=0.0, eloss=0.0), d)
    assert ok0.mean() < 0.6 and w_none[2] > 3 and w_none[3] > 3
    _, _, w_ms, _ = _pulls(dict(cfg, eloss=0.0), d)                      # energy loss ignored: q/pT is off
    assert w_ms[4] > 2.0 and abs(w_ms[2] - 1) < 0.06
    _, _, w_half, _ = _pulls(dict(cfg, x_over_x0=cfg["x_over_x0"] / 2), d)
    assert w_half[2] > 1.25 and w_half[3] > 1.25
    r, ok, _, _ = _pulls(dict(cfg, eloss=2 * cfg["eloss"]), d)             # twice the loss: |q/pT| overestimated
    bias = np.sign(r["par"][4, ok]) * (r["par"][4, ok] - d["truth_last_par"][4, ok]) / np.sqrt(r["cov"][14, ok])
    assert bias.mean() > 1.0


def test_generator_without_material_steps_along_the_analytic_helix():
    for name in ("tiny", "pileup"):
        a = W.generate(W.CONFIGS[name])
        b = W.generate(dataclasses.replace(W.CONFIGS[name], x_over_x0=1e-30))
        m = np.isfinite(a["truth_last"][:, 0])
        assert np.array_equal(m, np.isfinite(b["truth_last"][:, 0]))
        np.testing.assert_allclose(b["truth_last"][m], a["truth_last"][m], rtol=0, atol=1e-10)


def test_refit_with_material_is_the_inward_composition_and_has_unit_pulls(scattered):
    spec, d, cfg = scattered
    m = O.match(cfg, d)
    r = O.refit(cfg, d, m)
    n_checked = 0
    for i in range(300):
        att = [l for l in range(6) if m["idx"][l, i] >= 0]
        if len(att) < 2:
            continue
        p = m["par"][:, i].copy(); c15 = O.full_to_tri(np.diag(O.REFIT_VAR)); x = float(m["x"][i]); sec = int(m["sector"][i])
        ok, used = True, 0
        for l in range(att[-1], -1, -1):                      # every plane from the outermost attached tracklet inward
            X = cfg["layer_x"][l]
            if x != X:
                ok, p, c15, x, sec = O.propagate_to_layer(cfg, p, c15, x, sec, X)
            if not ok:
                break
            if l in att and int(d["tl_chamber"][m["idx"][l, i]]) // 30 == sec:
                k = int(m["idx"][l, i])
                p, c15, _ = O.update(cfg, p, c15, float(d["tl_y"][k]), float(d["tl_z"][k]), l)
                used += 1
                if abs(p[2]) >= cfg["max_snp"]:
                    ok = False
                    break
            ok, p, c15 = O.material(cfg, p, c15, -1)
            if not ok:
                break
        if ok:
            ok, p, c15, x, sec = O.propagate_to_layer(cfg, p, c15, x, sec, 247.0)
        if not ok:
            assert r["n_used"][i] == 0
            continue
        assert r["n_used"][i] == used and r["sector"][i] == sec
        np.testing.assert_allclose(r["par"][:, i], p, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(r["cov"][:, i], c15, rtol=1e-10, atol=1e-18)
        n_checked += 1
    assert n_checked > 250
    # pulls against the true state at the reference plane (before any slab).  The start values are the matcher's (far
    # better than the reset covariance says), so the reset variances are widened until they carry no weight
    r = O.refit(dict(cfg, refit_var=[100.0 * v for v in O.REFIT_VAR]), d, m)
    good = (r["n_used"] == 6) & np.all(m["idx"].T == d["truth_idx"], axis=1) & (r["sector"] == d["sector"])
    assert good.mean() > 0.8
    for k in range(5):
        pull = (r["par"][k, good] - d["truth_par"][k, good]) / np.sqrt(r["cov"][DIAG[k], good])
        assert pull.std() == pytest.approx(1.0, abs=0.07), k
        assert abs(pull.mean()) < 0.05, k
