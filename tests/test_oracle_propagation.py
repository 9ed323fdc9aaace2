"""Pins of the oracle's track model: closed forms, invariants,
finite differences.  Nothing here calls the CUDA path."""
import math

import numpy as np
import pytest

from oracle import oracle as O

B = -0.00299792458
RNG = np.random.default_rng(12345)
DIAG = O.full_to_tri(np.diag([0.01, 0.01, 1e-6, 1e-6, 1e-4]))


def random_state(bz=0.5, max_s=0.5):
    y = RNG.uniform(-40, 40); z = RNG.uniform(-300, 300)
    s = RNG.uniform(-max_s, max_s); t = RNG.uniform(-0.9, 0.9)
    c = RNG.choice([-1, 1]) / math.exp(RNG.uniform(math.log(0.5), math.log(20)))
    return np.array([y, z, s, t, c])


def test_straight_line_at_zero_field(base_cfg):
    """Bz = 0: y' = y + dx tan(phi), z' = z + dx tan(lambda)/cos(phi) exactly."""
    cfg = dict(base_cfg, bz_tesla=0.0)
    for _ in range(200):
        p = random_state(); dx = RNG.uniform(1, 120)
        ok, q, _, x = O.propagate(cfg, p, DIAG, 247.0, 247.0 + dx)
        assert ok and x == 247.0 + dx
        phi = math.asin(p[2])
        assert q[0] == pytest.approx(p[0] + dx * math.tan(phi), abs=1e-11)
        assert q[1] == pytest.approx(p[1] + dx * p[3] / math.cos(phi), abs=1e-11)
        assert np.array_equal(q[2:], p[2:])


def circle_crossing(p, x0, x1, bz):
    """Independent geometry: centre of the circle from the state, intersection with x = x1
    from the circle equation, z from the swept angle measured with atan2."""
    y, z, s, t, c = p
    kappa = B * bz * c
    R = 1.0 / kappa                                   # signed radius
    cphi = math.sqrt(1 - s * s)
    cx, cy = x0 - R * s, y + R * cphi                 # centre = point + R * (left normal of direction)
    # (x1 - cx)^2 + (y1 - cy)^2 = R^2, branch continuous with the start point
    root = math.sqrt(R * R - (x1 - cx) ** 2)
    y1 = cy - math.copysign(root, R)
    a0 = math.atan2(y - cy, x0 - cx); a1 = math.atan2(y1 - cy, x1 - cx)
    dphi = (a1 - a0 + math.pi) % (2 * math.pi) - math.pi
    return y1, z + t * dphi * R, (x1 - cx) / R


def test_analytic_circle(base_cfg):
    for _ in range(500):
        p = random_state(); x1 = RNG.choice([300.0, 313.0, 364.0, 250.0])
        ok, q, _, _ = O.propagate(base_cfg, p, DIAG, 247.0, x1)
        if not ok:
            assert abs(p[2] + B * 0.5 * p[4] * (x1 - 247.0)) >= base_cfg["max_snp"]
            continue
        y1, z1, s1 = circle_crossing(p, 247.0, x1, 0.5)
        assert q[0] == pytest.approx(y1, abs=2e-8)     # the circle form cancels at high pT: R ~ 1e4 cm
        assert q[1] == pytest.approx(z1, abs=2e-8)
        assert q[2] == pytest.approx(s1, abs=1e-12)


def test_composition_and_inverse(base_cfg):
    for _ in range(200):
        p = random_state(max_s=0.3)
        ok1, a, ca, xa = O.propagate(base_cfg, p, DIAG, 247.0, 300.0)
        ok2, b, cb, xb = O.propagate(base_cfg, a, ca, xa, 364.0)
        ok3, d, cd, xd = O.propagate(base_cfg, p, DIAG, 247.0, 364.0)
        if not (ok1 and ok2 and ok3):
            continue
        np.testing.assert_allclose(b, d, rtol=0, atol=1e-11)
        np.testing.assert_allclose(cb, cd, rtol=1e-9, atol=1e-16)   # F(x1->x2) F(x0->x1) = F(x0->x2)
        ok4, e, ce, _ = O.propagate(base_cfg, b, cb, xb, 247.0)
        assert ok4
        np.testing.assert_allclose(e, p, rtol=0, atol=1e-11)
        np.testing.assert_allclose(ce, DIAG, rtol=1e-8, atol=1e-15)


def state_map(cfg, p, x0, x1):
    ok, q, _, _ = O.propagate(cfg, p, DIAG, x0, x1)
    assert ok
    return q


@pytest.mark.parametrize("dx", [53.0, 13.0, 12.0, 1e-3, -40.0])
def test_propagation_jacobian_finite_differences(base_cfg, dx):
    steps = np.array([1e-4, 1e-4, 1e-6, 1e-6, 1e-6])
    for _ in range(100):
        p = random_state(max_s=0.4)
        ok, _, _, _, F = O.propagate(base_cfg, p, DIAG, 300.0, 300.0 + dx, want_jacobian=True)
        if not ok:
            continue
        num = np.zeros((5, 5))
        for j in range(5):
            e = np.zeros(5); e[j] = steps[j]
            num[:, j] = (state_map(base_cfg, p + e, 300.0, 300.0 + dx) - state_map(base_cfg, p - e, 300.0, 300.0 + dx)) / (2 * steps[j])
        # 2e-6 relative; 2e-7 absolute is the round-off floor of the difference quotient (|z| ~ 300, step 1e-6)
        assert np.all(np.abs(F - num) <= 2e-6 * np.abs(num) + 2e-7), (p, F - num)


def test_jacobian_small_curvature_limits(base_cfg):
    """kappa -> 0: the textbook small-step entries."""
    p = np.array([3.0, -20.0, 0.3, 0.5, 1e-9]); dx = 13.0
    ok, _, _, _, F = O.propagate(base_cfg, p, DIAG, 300.0, 313.0, want_jacobian=True)
    s, t = p[2], p[3]; r = math.sqrt(1 - s * s); b = B * 0.5
    assert F[0, 2] == pytest.approx(dx / r ** 3, rel=1e-8)
    assert F[0, 4] == pytest.approx(0.5 * b * dx * dx / r ** 3, rel=1e-8)
    assert F[1, 2] == pytest.approx(dx * t * s / r ** 3, rel=1e-8)
    assert F[1, 3] == pytest.approx(dx / r, rel=1e-8)
    assert F[1, 4] == pytest.approx(0.5 * b * t * dx * dx * s / r ** 3, rel=1e-7)
    assert F[2, 4] == pytest.approx(b * dx, rel=1e-12)


def test_covariance_transport_is_F_C_Ft(base_cfg):
    """C' = F C F^T recomputed with numpy on the full matrices."""
    for _ in range(50):
        p = random_state(max_s=0.4)
        A = RNG.normal(size=(5, 5)) * np.array([0.1, 0.1, 1e-3, 1e-3, 1e-2])[:, None]
        Cfull = A @ A.T
        ok, _, c1, _, F = O.propagate(base_cfg, p, O.full_to_tri(Cfull), 300.0, 338.0, want_jacobian=True)
        if ok:
            np.testing.assert_allclose(O.tri_to_full(c1), F @ Cfull @ F.T, rtol=1e-10, atol=1e-18)


def to_global(x, y, sector):
    a = (sector + 0.5) * math.radians(20.0)
    return x * math.cos(a) - y * math.sin(a), x * math.sin(a) + y * math.cos(a)


def test_rotation_roundtrip_and_same_point(base_cfg):
    beta = math.radians(20.0)
    for _ in range(200):
        p = random_state(max_s=0.5)
        ok, q, cq, xq = O.rotate(base_cfg, p, DIAG, 300.0, beta)
        assert ok
        gx0, gy0 = to_global(300.0, p[0], 4); gx1, gy1 = to_global(xq, q[0], 5)
        assert gx0 == pytest.approx(gx1, abs=1e-10) and gy0 == pytest.approx(gy1, abs=1e-10)
        # direction: phi' = phi - beta
        assert math.asin(q[2]) == pytest.approx(math.asin(p[2]) - beta, abs=1e-12)
        ok, r, cr, xr = O.rotate(base_cfg, q, cq, xq, -beta)
        assert ok and xr == pytest.approx(300.0, abs=1e-10)
        np.testing.assert_allclose(r, p, atol=1e-11)
        np.testing.assert_allclose(cr, DIAG, rtol=1e-9, atol=1e-18)


@pytest.mark.parametrize("sign", [1, -1])
def test_rotation_jacobian_finite_differences(base_cfg, sign):
    """Perturb in the old frame, rotate, bring the track back to the unperturbed plane x' = const
    with the (separately pinned) exact propagation; the difference quotient must equal J."""
    beta = sign * math.radians(20.0)
    steps = np.array([1e-4, 1e-4, 1e-6, 1e-6, 1e-6])

    def mapped(pp, xref):
        ok, q, cq, xq = O.rotate(base_cfg, pp, DIAG, 300.0, beta)
        assert ok
        return state_map(base_cfg, q, xq, xref)

    for _ in range(100):
        p = random_state(max_s=0.5)
        ok, q, _, xq, J = O.rotate(base_cfg, p, DIAG, 300.0, beta, want_jacobian=True)
        num = np.zeros((5, 5))
        for j in range(5):
            e = np.zeros(5); e[j] = steps[j]
            num[:, j] = (mapped(p + e, xq) - mapped(p - e, xq)) / (2 * steps[j])
        assert np.max(np.abs(J - num)) < 5e-7, (J - num)


def test_propagate_to_layer_crosses_sector_like_the_global_helix(base_cfg):
    """A track aimed at the sector edge ends in the neighbour frame at the same global point the
    single-frame propagation reaches, with |y| inside the new sector."""
    edge = 300.0 * math.tan(math.radians(10.0))
    n_rot = 0
    for _ in range(300):
        p = random_state(max_s=0.2); p[0] = RNG.choice([-1, 1]) * RNG.uniform(40.0, 43.5); p[4] *= 0.2
        p[2] = math.copysign(RNG.uniform(0.1, 0.4), p[0])
        ok0, q0, _, _ = O.propagate(base_cfg, p, DIAG, 247.0, 300.0)
        ok, q, cq, x, sec = O.propagate_to_layer(base_cfg, p, DIAG, 247.0, 7, 300.0)
        assert ok0 and ok and x == 300.0 and abs(q[0]) <= edge
        if abs(q0[0]) <= edge:
            assert sec == 7 and np.allclose(q, q0, atol=1e-12)
            continue
        n_rot += 1
        assert sec == (8 if q0[0] > 0 else 6)
        # global point of (300, q) in the new sector lies on the same circle: check with the circle centre
        y0, z0, s0, t0, c0 = p; R = 1.0 / (B * 0.5 * c0)
        cx, cy = 247.0 - R * s0, y0 + R * math.sqrt(1 - s0 * s0)
        gcx, gcy = to_global(cx, cy, 7); gx, gy = to_global(300.0, q[0], sec)
        assert math.hypot(gx - gcx, gy - gcy) == pytest.approx(abs(R), rel=1e-12)
        assert np.all(np.linalg.eigvalsh(O.tri_to_full(cq)) > 0)
    assert n_rot > 20


def test_max_snp_kills(base_cfg):
    p = np.array([0.0, 0.0, 0.9, 0.1, 1.0 / 0.5])       # pT = 0.5: kappa dx = -0.003 * 53 = -0.159
    assert O.propagate(base_cfg, p, DIAG, 247.0, 300.0)[0]
    p[2] = -0.9
    ok, q, c, x = O.propagate(base_cfg, p, DIAG, 247.0, 300.0)
    assert not ok and x == 247.0 and np.array_equal(q, p)   # untouched on failure
