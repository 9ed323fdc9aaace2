"""The seeded input generator: determinism and the sizes BASELINE.json's configs state."""
import numpy as np

from paper_2003_03174_b200 import workloads as W


def test_same_seed_same_bytes():
    a = W.generate(W.CONFIGS["tiny"]); b = W.generate(W.CONFIGS["tiny"])
    for k in ("par", "cov", "x", "sector", "tl_y", "tl_z", "tl_dydx", "tl_chamber", "tl_label"):
        assert a[k].tobytes() == b[k].tobytes()
        assert a[k].dtype in (np.float32, np.int32)


def test_config_sizes():
    d = W.generate(W.CONFIGS["central"])
    assert d["par"].shape == (5, 5000) and d["cov"].shape == (15, 5000)
    n_sig = int((d["tl_label"] >= 0).sum())
    assert 25_000 < n_sig < 30_000 and int((d["tl_label"] < 0).sum()) == 20_000      # "about 30k" + 20k
    assert d["tl_chamber"].min() >= 0 and d["tl_chamber"].max() < 540
    assert np.all(np.abs(d["par"][0]) <= 247.0 * W.TAN_HALF_SECTOR + 1.0)
    # z at pad-row centres, stacks tile |z| < 350
    assert np.allclose((d["tl_z"] / 8.0 - 0.5) % 1.0, 0.0)
    st = (d["tl_chamber"] // 6) % 5
    assert np.array_equal(st, W.stack_of_z(d["tl_z"].astype(float)))


def test_scaled_keeps_density():
    s = W.scaled(W.CONFIGS["timeframe"], 20_000)
    assert s.n_noise == 80_000 and s.batch == 20_000 and s.n_hyp == 4
