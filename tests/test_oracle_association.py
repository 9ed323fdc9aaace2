"""Pins of the oracle's time-frame association ("tracklets ... matched only to
tracks of the same interaction", "only those tracklets which belong to the same interaction").
Reading R27 of DESIGN.md."""
import dataclasses

import numpy as np

from oracle import oracle as O
from paper_2003_03174_b200 import workloads as W

KEYS = ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals")


def test_association_equals_one_plain_matching_per_interaction():
    """The associated result must be what the (already pinned) plain matcher gives when it is run once per
    interaction on that interaction's tracks and tracklets only -- an independent route through the code."""
    spec = dataclasses.replace(W.CONFIGS["pileup"], n_tracks=6000, n_noise=60000, n_interactions=5, number=13)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    got = O.match(cfg, d)
    assert set(np.unique(d["interaction"])) == set(range(5)) and set(np.unique(d["tl_interaction"])) == set(range(5))
    for k in range(5):
        trk = np.nonzero(d["interaction"] == k)[0]; tl = np.nonzero(d["tl_interaction"] == k)[0]
        sub = dict(par=d["par"][:, trk], cov=d["cov"][:, trk], x=d["x"][trk], sector=d["sector"][trk],
                   tl_y=d["tl_y"][tl], tl_z=d["tl_z"][tl], tl_dydx=d["tl_dydx"][tl], tl_chamber=d["tl_chamber"][tl])
        want = O.match(cfg, sub)
        idx = np.where(want["idx"] >= 0, tl[np.maximum(want["idx"], 0)], -1)          # back to global positions
        np.testing.assert_array_equal(got["idx"][:, trk], idx)
        for key in KEYS[1:]:
            np.testing.assert_array_equal(got[key][..., trk], want[key])
    # and it is not the un-associated result: other collisions' tracklets are fakes that the association removes
    plain = O.match(cfg, {k: v for k, v in d.items() if k not in ("n_interactions", "interaction", "tl_interaction")})
    assert got["counters"]["n_cand"] < plain["counters"]["n_cand"]
    assert (got["idx"] != plain["idx"]).any()


def test_sorted_per_interaction_lists_equal_brute_force_id_comparison():
    spec = dataclasses.replace(W.CONFIGS["central8"], n_interactions=7, number=14)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    a = O.match(cfg, d); b = O.match(cfg, d, brute=True)
    for k in KEYS:
        np.testing.assert_array_equal(a[k], b[k])
    assert a["counters"]["n_cand"] == b["counters"]["n_cand"]


def test_a_single_interaction_is_the_plain_matcher_and_unknown_ids_never_match():
    spec = W.CONFIGS["tiny"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    plain = O.match(cfg, d)
    d1 = dict(d, n_interactions=3, interaction=np.full(spec.n_tracks, 2, np.int32),
              tl_interaction=np.full(d["tl_y"].shape[0], 2, np.int32))
    same = O.match(cfg, d1)
    for k in KEYS:
        np.testing.assert_array_equal(plain[k], same[k])
    d2 = dict(d1); d2["interaction"] = d1["interaction"].copy(); d2["interaction"][:10] = [0, 1, -1, 3, 99, 0, 1, -5, 7, 0]
    d2["tl_interaction"] = d1["tl_interaction"].copy(); d2["tl_interaction"][::5] = 77      # unusable tracklets
    r = O.match(cfg, d2)
    assert r["idx"][:, :10].max() == -1 and r["n_matched"][:10].max() == 0
    assert not np.isin(r["idx"][r["idx"] >= 0], np.arange(0, d["tl_y"].shape[0], 5)).any()


def test_generator_ids():
    spec = dataclasses.replace(W.CONFIGS["central"], n_interactions=4)
    d = W.generate(spec)
    assert d["n_interactions"] == 4 and np.array_equal(np.bincount(d["interaction"]), [1250] * 4)
    sig = d["tl_label"] >= 0
    assert np.array_equal(d["tl_interaction"][sig], d["interaction"][d["tl_label"][sig]])
    # specs without association are untouched by the extra draw
    a = W.generate(W.CONFIGS["central"]); assert "interaction" not in a
