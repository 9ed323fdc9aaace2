"""Pins of the oracle's per-track `margin` and of its replay of fragile decisions.

The margin is the smallest relative distance of any discrete decision from its threshold.  Each test builds ONE
track and at most two tracklets so that exactly one decision sits at a known distance delta from its threshold -- a
road edge in y, the road in z, the inclination veto, the chi2 cut, the sector edge, max_snp, the rank gap
at the keep boundary -- and every other decision is far away; the reported margin must equal that distance to 1e-12
(computed here from the float32 inputs with the separately pinned propagation / road functions).  The replay
(`match_alternatives`) must then reach the chain with that one decision taken the other way, and must not reach it
when eps is below delta.
"""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W

DELTA = 3.7e-5
SECTOR, LAYER0_X = 4, 300.0


def one_track(cfg, y=3.0, z=21.3, s=0.05, t=0.3, c=0.4):
    """A seed in the middle of sector 4, far from every threshold; float32 as the matcher receives it."""
    par = np.array([[y], [z], [s], [t], [c]], np.float32)
    cov = np.zeros((15, 1), np.float32)
    for k, v in enumerate((0.01, 0.01, 1e-6, 1e-6, (0.01 * c) ** 2)):
        cov[k * (k + 1) // 2 + k, 0] = v
    return dict(par=par, cov=cov, x=np.array([247.0], np.float32), sector=np.array([SECTOR], np.int32))


def at_layer0(cfg, trk):
    ok, p, c15, x, sec = O.propagate_to_layer(cfg, trk["par"][:, 0].astype(float), trk["cov"][:, 0].astype(float),
                                              float(trk["x"][0]), int(trk["sector"][0]), LAYER0_X)
    assert ok and sec == SECTOR
    return p, c15, O.road(cfg, p, c15, layer=0)


def with_tracklets(trk, y, z, dydx):
    n = len(y)
    return dict(trk, tl_y=np.array(y, np.float32), tl_z=np.array(z, np.float32), tl_dydx=np.array(dydx, np.float32),
                tl_chamber=np.full(n, SECTOR * 30 + 2 * 6 + 0, np.int32))


def cfg_of(base_cfg, **over):
    return dict(base_cfg, n_hyp=1, **over)


def check_margin(cfg, data, expected, attached):
    res = O.match(cfg, data)
    assert res["margin"][0] == pytest.approx(expected, rel=1e-12, abs=1e-15)
    assert expected == pytest.approx(DELTA, rel=0.05)              # and that distance is the one that was built in
    assert (res["idx"][0, 0] >= 0) == attached
    return res


def check_replay(cfg, data, res):
    """The chain with the one fragile decision taken the other way is an alternative at eps = 1e-4, not at eps < delta."""
    natural = res["idx"][:, :1]
    n_tl = data["tl_y"].shape[0]
    other = natural.copy()
    if natural[0, 0] < 0:
        other[0, 0] = 0
    elif n_tl == 2:
        other[0, 0] = 1 - natural[0, 0]
    else:
        other[0, 0] = -1
    a = O.match_alternatives(cfg, data, [0], natural, eps=1e-4)
    assert a["found"][0] == 1                                       # the natural result needs no replay
    np.testing.assert_array_equal(a["par"][:, 0], res["par"][:, 0])
    b = O.match_alternatives(cfg, data, [0], other, eps=1e-4)
    assert b["found"][0] == 2, b["found"]                           # one flipped decision
    np.testing.assert_array_equal(b["idx"], other)
    assert b["n_matched"][0] == int((other >= 0).sum())
    c = O.match_alternatives(cfg, data, [0], other, eps=0.5 * DELTA)
    assert c["found"][0] < 0                                        # not fragile at that eps: not an alternative
    # an impossible chain is never "found"
    bogus = natural.copy(); bogus[3, 0] = 0
    assert O.match_alternatives(cfg, data, [0], bogus, eps=1e-4)["found"][0] < 0
    return b


@pytest.mark.parametrize("side", [-1, +1])
def test_margin_of_the_y_road_edge(base_cfg, side):
    cfg = cfg_of(base_cfg); trk = one_track(cfg)
    p, c15, rd = at_layer0(cfg, trk)
    data = with_tracklets(trk, [p[0] + rd["road_y"] * (1.0 + side * DELTA)], [p[1]], [rd["tanphi"]])
    ry = abs(float(data["tl_y"][0]) - p[0])
    res = check_margin(cfg, data, abs(ry - rd["road_y"]) / rd["road_y"], attached=side < 0)
    alt = check_replay(cfg, data, res)
    if side > 0:                                                    # forced inside: updated with the tracklet
        pu, cu, chi2 = O.update(cfg, p, c15, float(data["tl_y"][0]), float(data["tl_z"][0]))
        assert alt["chi2"][0] == pytest.approx(chi2, rel=1e-12)


def test_margin_of_the_z_road(base_cfg):
    cfg = cfg_of(base_cfg); trk = one_track(cfg)
    p, c15, rd = at_layer0(cfg, trk)
    data = with_tracklets(trk, [p[0]], [p[1] - rd["road_z"] * (1.0 - DELTA)], [rd["tanphi"]])
    rz = abs(float(data["tl_z"][0]) - p[1])
    res = check_margin(cfg, data, abs(rz - rd["road_z"]) / rd["road_z"], attached=True)
    check_replay(cfg, data, res)


def test_margin_of_the_inclination_veto(base_cfg):
    cfg = cfg_of(base_cfg); trk = one_track(cfg)
    p, c15, rd = at_layer0(cfg, trk)
    veto = cfg["n_sigma_angle"] * cfg["sigma_dydx"]                  # PAPER.md:60, 4 sigma
    data = with_tracklets(trk, [p[0]], [p[1]], [rd["tanphi"] + veto * (1.0 + DELTA)])
    da = abs(float(data["tl_dydx"][0]) - rd["tanphi"])
    res = check_margin(cfg, data, abs(da - veto) / veto, attached=False)
    check_replay(cfg, data, res)


def test_margin_of_the_chi2_cut(base_cfg):
    cfg = cfg_of(base_cfg, chi2_cut=5.0, chi2_penalty=5.0); trk = one_track(cfg)
    p, c15, rd = at_layer0(cfg, trk)
    ry = math.sqrt(5.0 * (1.0 - DELTA) / rd["Sinv"][0, 0])
    data = with_tracklets(trk, [p[0] + ry], [p[1]], [rd["tanphi"]])
    r = np.array([float(data["tl_y"][0]) - p[0], float(data["tl_z"][0]) - p[1]])
    c2 = float(r @ rd["Sinv"] @ r)
    res = check_margin(cfg, data, abs(c2 - 5.0) / 5.0, attached=True)
    check_replay(cfg, data, res)


def test_margin_of_the_sector_edge(base_cfg):
    cfg = cfg_of(base_cfg)
    edge = LAYER0_X * math.tan(math.pi / cfg["n_sectors"])
    trk = one_track(cfg, y=30.0)
    p, _, _ = at_layer0(cfg, trk)
    trk = one_track(cfg, y=30.0 + edge * (1.0 - DELTA) - p[0])      # y at the plane moves with the seed's y
    ok, p, c15, x = O.propagate(cfg, trk["par"][:, 0].astype(float), trk["cov"][:, 0].astype(float), 247.0, LAYER0_X)
    data = with_tracklets(trk, [], [], [])
    res = O.match(cfg, data)
    assert res["margin"][0] == pytest.approx(abs(abs(p[0]) - edge) / edge, rel=1e-12)
    assert res["margin"][0] == pytest.approx(DELTA, rel=0.05)
    assert res["sector"][0] == SECTOR                               # stayed: the edge itself is inside
    # the replay takes the step over the edge: the track ends in the neighbouring sector frame
    nat = res["idx"][:, :1]
    runs = O.match_alternatives(cfg, data, [0], nat, eps=1e-4)
    assert runs["found"][0] == 1


def test_margin_of_max_snp(base_cfg):
    cfg = cfg_of(base_cfg, bz_tesla=0.0)                            # straight line: sin(phi) stays what it is
    s = cfg["max_snp"] * (1.0 - DELTA)
    trk = one_track(cfg, y=-40.0, s=s, c=0.0)
    data = with_tracklets(trk, [], [], [])
    res = O.match(cfg, data)
    s32 = float(trk["par"][2, 0])
    assert res["margin"][0] == pytest.approx(abs(s32 - cfg["max_snp"]) / cfg["max_snp"], rel=1e-12)
    assert res["margin"][0] == pytest.approx(DELTA, rel=0.05)


def test_margin_of_the_rank_gap_at_the_keep_boundary(base_cfg):
    cfg = cfg_of(base_cfg); trk = one_track(cfg)
    p, c15, rd = at_layer0(cfg, trk)
    ry_a = 1.2 * math.sqrt(1.0 / rd["Sinv"][0, 0])
    ry_b = -ry_a / math.sqrt(1.0 - DELTA)                            # chi2_b (1 - delta) = chi2_a
    data = with_tracklets(trk, [p[0] + ry_a, p[0] + ry_b], [p[1], p[1]], [rd["tanphi"], rd["tanphi"]])
    idx, chi2 = O.candidates(cfg, data, p, c15, sector=SECTOR, layer=0)
    assert idx.tolist() == [0, 1] and chi2[0] < chi2[1]
    res = check_margin(cfg, data, (chi2[1] - chi2[0]) / chi2[1], attached=True)
    assert res["idx"][0, 0] == 0
    alt = check_replay(cfg, data, res)
    assert alt["chi2"][0] == pytest.approx(chi2[1], rel=1e-12)       # the other child was kept and updated


def test_nothing_fragile_nothing_to_replay(base_cfg):
    """A config-2 sample: tracks with margin >= 1e-4 have exactly one result at eps = 1e-4; asking for any other chain
    fails.  Fragile tracks reach at least one other chain or none, never a chain that breaks a non-fragile decision."""
    spec = dataclasses.replace(W.CONFIGS["central"], n_tracks=400, n_noise=40000, n_hyp=4)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    res = O.match(cfg, d)
    solid = np.nonzero(res["margin"] >= 1e-4)[0][:50]
    a = O.match_alternatives(cfg, d, solid, res["idx"][:, solid])
    assert np.all(a["found"] == 1)
    wrong = res["idx"][:, solid].copy()
    wrong[2] = np.where(wrong[2] >= 0, -1, 0)                       # another layer-2 decision
    b = O.match_alternatives(cfg, d, solid, wrong)
    assert np.all(b["found"] < 0) and np.all(b["found"] == -1)      # one replay each: nothing to flip
