"""Pins of the oracle's two-stage propagation with radially displaced chambers (PAPER.md:64:
tracks are extrapolated to the average radius of a chamber, "fast linear extrapolations" to each tracklet's radius
serve the chi2, and "before the tracks are updated ... they are again propagated ... to the exact radius").
Readings R28-R30 of DESIGN.md."""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W

KEYS = ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals")


def test_zero_offsets_are_the_plain_matcher_bit_for_bit():
    spec = W.CONFIGS["central8"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d)
    b = O.match(cfg, dict(d, chamber_dx=np.zeros(540, np.float32)))
    for k in KEYS + ("margin",):
        np.testing.assert_array_equal(a[k], b[k])


def test_noise_free_recovery_at_the_displaced_radius():
    """Unsmeared seed and tracklets, exact z, no noise, full efficiency, chambers displaced by up to 0.9 cm: every
    layer attaches the true tracklet with chi2 = 0 and the final state is the true helix at x_layer + dx."""
    spec = dataclasses.replace(W.CONFIGS["tiny"], smear_seed=False, smear_tracklets=False, exact_z=True, efficiency=1.0,
                               n_noise=0, chamber_dx_sigma=0.3, number=15)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.match(cfg, d)
    full = np.all(d["truth_idx"] >= 0, axis=1)
    assert full.mean() > 0.9
    assert np.array_equal(r["idx"].T[full], d["truth_idx"][full])
    assert r["chi2"][full].max() < 1e-6                      # float32 inputs: (4e-6 cm / 0.04 cm)^2 per layer
    # the state lives at the displaced radius of the last chamber, on the true helix
    last = d["truth_idx"][full, 5]
    x_want = 364.0 + d["chamber_dx"][d["tl_chamber"][last]].astype(np.float64)
    np.testing.assert_allclose(r["x"][full], x_want, rtol=0, atol=1e-12)
    assert np.abs(r["x"][full] - 364.0).max() > 0.3
    np.testing.assert_allclose(r["par"][0, full], d["tl_y"][last].astype(np.float64), atol=2e-5)      # float32 tracklets
    np.testing.assert_allclose(r["par"][1, full], d["tl_z"][last].astype(np.float64), atol=1e-4)
    np.testing.assert_allclose(r["par"][4, full], d["truth_par"][4, full], rtol=1e-6)
    # without the offsets the same input does not fit
    r0 = O.match(cfg, {k: v for k, v in d.items() if k != "chamber_dx"})
    assert r0["chi2"][full].mean() > 1.0


def test_linear_extrapolation_for_the_road_and_exact_propagation_for_the_update(base_cfg):
    """R29: candidate chi2 from the residual against (y + dx tan(phi), z + dx tan(lambda) / cos(phi)) with the
    covariance of the nominal plane.  R30: the attached child's chi2 and state are those of the (separately pinned)
    exact propagation to x + dx followed by the (separately pinned) update."""
    s, t = 0.3, 0.45
    p = np.array([5.0, 20.0, s, t, 0.5]); Cm = np.diag([0.01, 0.02, 1e-6, 1e-6, 1e-4]); c15 = O.full_to_tri(Cm)
    dx = np.zeros(540); ch = 3 * 30 + 2 * 6 + 1; dx[ch] = 0.8
    tanphi = s / math.sqrt(1 - s * s); zsl = t / math.sqrt(1 - s * s)
    ym, zm = np.float32(5.0 + 0.8 * tanphi + 0.05), np.float32(20.0 + 0.8 * zsl - 1.0)
    tl = dict(tl_y=np.array([ym], np.float32), tl_z=np.array([zm], np.float32), tl_dydx=np.array([tanphi], np.float32),
              tl_chamber=np.array([ch], np.int32))
    for brute in (False, True):
        idx, chi2 = O.candidates(base_cfg, tl, p, c15, sector=3, layer=1, brute=brute, chamber_dx=dx)
        res = np.array([float(ym) - (p[0] + 0.8 * tanphi), float(zm) - (p[1] + 0.8 * zsl)])
        S = np.diag([0.01 + base_cfg["sigma_y"] ** 2, 0.02 + base_cfg["sigma_z"] ** 2])
        assert idx.tolist() == [0] and chi2[0] == pytest.approx(res @ np.linalg.inv(S) @ res, rel=1e-12)
    # without the offset the same tracklet looks 0.30 cm off in y: a much worse chi2
    _, chi2_plain = O.candidates(base_cfg, tl, p, c15, sector=3, layer=1)
    assert chi2_plain[0] > 10 * chi2[0]
    # whole step for one track that starts exactly on the plane of layer 1 (layers 0 and 2..5 have no tracklet)
    cfg = dict(base_cfg, n_hyp=1, layer_x=[312.0, 313.0, 326.0, 338.0, 351.0, 364.0])
    data = dict(tl, chamber_dx=dx, par=p[:, None].astype(np.float32), cov=c15[:, None].astype(np.float32),
                x=np.array([313.0], np.float32), sector=np.array([3], np.int32))
    cfg1 = dict(cfg, layer_x=[313.0, 326.0, 338.0, 351.0, 364.0, 377.0])     # make the plane x = 313 layer 0 ...
    data1 = dict(data, tl_chamber=np.array([3 * 30 + 2 * 6 + 0], np.int32)); dx1 = np.zeros(540); dx1[3 * 30 + 2 * 6 + 0] = 0.8
    data1["chamber_dx"] = dx1
    r = O.match(cfg1, data1)
    assert r["idx"][0, 0] == 0
    pf = data1["par"][:, 0].astype(np.float64); cf = data1["cov"][:, 0].astype(np.float64)
    ok, p2, c2, x2 = O.propagate(cfg1, pf, cf, 313.0, 313.8)
    p3, c3, chi2 = O.update(cfg1, p2, c2, float(ym), float(zm), 0)
    assert ok and r["chi2"][0] == pytest.approx(chi2, rel=1e-12)
    # the remaining layers only propagate the state on
    okk, p4, c4, x4, sec4 = O.propagate_to_layer(cfg1, p3, c3, 313.8, 3, 326.0)
    assert okk and r["n_matched"][0] == 1


def test_pulls_with_offsets_and_sensitivity():
    spec = dataclasses.replace(W.CONFIGS["central"], chamber_dx_sigma=0.3, n_noise=0, efficiency=1.0, n_tracks=20000, number=16)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    r = O.match(cfg, d)
    ok = (r["n_matched"] == 6) & np.all(r["idx"].T == d["truth_idx"], axis=1)
    assert ok.mean() > 0.9
    per = r["chi2"][ok].sum() / (6 * ok.sum())
    assert per == pytest.approx(2.0, abs=0.05)
    r0 = O.match(cfg, {k: v for k, v in d.items() if k != "chamber_dx"})
    m0 = r0["n_matched"] > 0
    assert r0["chi2"][m0].sum() / r0["n_matched"][m0].sum() > 1.15 * per
    assert r0["n_matched"].sum() < 0.97 * r["n_matched"].sum()


def test_sorted_index_equals_brute_force_with_offsets():
    spec = dataclasses.replace(W.CONFIGS["central8"], chamber_dx_sigma=0.3, res_model=1, n_interactions=3)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d); b = O.match(cfg, d, brute=True)
    for k in KEYS:
        np.testing.assert_array_equal(a[k], b[k])


def enumerate_chains_two_stage(cfg, d, i):
    """Depth-first enumeration of ALL chains of track i with displaced chambers: at each layer every candidate the
    linear extrapolation accepts (R29) -- attached after the EXACT propagation to its chamber's radius, scored with the
    exact chi2 (R30) -- or skip.  Returns the sorted list of (exact score, idx tuple)."""
    out = []
    dx_ch = d["chamber_dx"].astype(np.float64)

    def rec(L, p, c15, x, sec, alive, score, idx):
        if L == 6:
            out.append((score, tuple(idx)))
            return
        if alive:
            ok, p2, c2, x2, sec2 = O.propagate_to_layer(cfg, p, c15, x, sec, cfg["layer_x"][L])
            if ok:
                p, c15, x, sec = p2, c2, x2, sec2
                ci, _ = O.candidates(cfg, d, p, c15, sec, L, brute=True, chamber_dx=dx_ch)
                for k in ci.tolist():
                    dxk = dx_ch[d["tl_chamber"][k]]
                    pe, ce, xe, ok2 = p, c15, x, True
                    if dxk != 0.0:
                        ok2, pe, ce, xe = O.propagate(cfg, p, c15, x, x + dxk)
                    if not ok2:                                  # cannot get there: keeps its state, only skips from now on
                        rec(L + 1, p, c15, x, sec, False, score, idx + [-1])
                        continue
                    pn, cn, inc = O.update(cfg, pe, ce, float(d["tl_y"][k]), float(d["tl_z"][k]), layer=L)
                    rec(L + 1, pn, cn, xe, sec, abs(pn[2]) < cfg["max_snp"], score + inc, idx + [int(k)])
            else:
                alive = False
        rec(L + 1, p, c15, x, sec, alive, score + cfg["chi2_penalty"], idx + [-1])

    rec(0, d["par"][:, i].astype(float), d["cov"][:, i].astype(float), float(d["x"][i]), int(d["sector"][i]),
        abs(float(d["par"][2, i])) < cfg["max_snp"], 0.0, [])
    out.sort()
    return out


def test_output_is_the_chain_with_the_lowest_exact_score():
    """With every child kept (nHyp = 4096) the matcher is exhaustive, and its output must be the chain with the lowest
    EXACT total score -- the scores of the kept children are replaced by the exact chi2 after the ranking (R30), so the
    first hypothesis of the list is not always the best one; the output is the minimum over the final list."""
    # offsets of 2 cm and a soft spectrum: the linear extrapolation then differs from the exact step by the sagitta
    # kappa dx^2 / 2 ~ 0.01-0.05 cm, of the order of the tracklet resolution, so the two rankings do disagree
    spec = dataclasses.replace(W.CONFIGS["tiny"], name="dense_dx", number=31, n_tracks=60, n_noise=60000, n_hyp=4,
                               chamber_dx_sigma=2.0, pt_spectrum="exp")
    d = W.generate(spec); cfg = W.matcher_config(spec)
    big = O.match(dict(cfg, n_hyp=4096), d)
    n_multi = n_reordered = 0
    for i in range(spec.n_tracks):
        chains = enumerate_chains_two_stage(cfg, d, i)
        assert len(chains) <= 4096
        n_multi += len(chains) > 4
        best_score, best_idx = chains[0]
        if len(chains) > 1 and chains[1][0] - best_score < 1e-9 * max(best_score, 1.0):
            continue                                             # an exact tie: either is right
        assert tuple(big["idx"][:, i].tolist()) == best_idx, i
        n_skip = sum(1 for t in best_idx if t < 0)
        assert big["chi2"][i] + cfg["chi2_penalty"] * n_skip == pytest.approx(best_score, rel=1e-10, abs=1e-10)
    assert n_multi >= 10
