"""trd_load_tracklets on the GPU: the sorted store is a stable permutation of the
input by bin key, the first-position table reproduces a CPU counting sort exactly (integer parity).  Both device
sorts (trd_config.index_sort: radix passes, counting sort) must give that same index; only the order of the unusable
tracklets behind the last bin, which nothing reads, is free after a counting sort."""
import numpy as np
import pytest

from paper_2003_03174_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_03174_b200 import binding, build
    build.build()
    return binding


def load(B, cfg, y, z, d, ch):
    import torch
    h = B.trd_create(cfg)
    t = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (y, z, d, ch)]
    B.trd_load_tracklets(h, *t)
    ix = B.trd_copy_index(h)
    return h, ix


def check_index(cfg, ix, y, z, ch):
    n = y.shape[0]
    nb, nz, n_bins = ix["n_ybins"], ix["n_zrows"], ix["n_bins"]
    key, pos, first = ix["sorted_key"].astype(np.int64), ix["sorted_pos"].astype(np.int64), ix["bin_first"]
    assert np.all(np.diff(key) >= 0)                                          # sorted
    assert np.array_equal(np.sort(pos), np.arange(n))                         # a permutation
    n_usable = int(np.searchsorted(key, n_bins, side="left"))
    same = np.diff(key[:n_usable]) == 0
    assert np.all(np.diff(pos[:n_usable])[same] > 0)                          # stable: ties keep input order
    # counting sort on the CPU from the keys the device assigned
    key_of_input = np.empty(n, np.int64); key_of_input[pos] = key
    ref = np.argsort(key_of_input, kind="stable")
    assert np.array_equal(pos[:n_usable], ref[:n_usable])
    if ix["sort_kind"] in (1, 3):
        assert np.array_equal(np.sort(pos[n_usable:]), ref[n_usable:])        # the unusable ones: any order
    else:
        assert np.array_equal(pos, ref)
    assert np.array_equal(first, np.searchsorted(key, np.arange(n_bins + 1), side="left").astype(np.int32))
    assert np.all(np.diff(first) >= 0) and first[0] == 0
    # the key means what the header says: (sector, layer) cell, z row, y bin
    per_sector = cfg["n_stacks"] * cfg["n_layers"]
    usable = (ch >= 0) & (ch < cfg["n_sectors"] * per_sector) & np.isfinite(y) & np.isfinite(z)
    assert np.all(key_of_input[~usable] == n_bins)
    k = key_of_input[usable]
    cell = k // (nz * nb); zrow = (k // nb) % nz; ybin = k % nb
    assert np.array_equal(cell, (ch[usable] // per_sector) * cfg["n_layers"] + ch[usable] % cfg["n_layers"])
    zlo = (zrow - nz // 2) * cfg["pad_length"]
    zz = z[usable].astype(np.float64)
    inside = (zz >= zlo - 1e-3) & (zz < zlo + cfg["pad_length"] + 1e-3)
    edge_row = (zrow == 0) | (zrow == nz - 1)
    assert np.all(inside | edge_row)
    w = ix["ybin_width"]; y_half = w * nb / 2
    ylo = ybin * w - y_half
    yy = y[usable].astype(np.float64)
    inside = (yy >= ylo - 1e-3) & (yy < ylo + w + 1e-3)
    edge_bin = (ybin == 0) | (ybin == nb - 1)
    assert np.all(inside | edge_bin)
    assert first[n_bins] == usable.sum()


@pytest.mark.parametrize("index_sort", [-1, 1])
@pytest.mark.parametrize("name", ["tiny", "central", "pileup"])
def test_index_of_the_configs(B, name, index_sort):
    spec = W.CONFIGS[name]; d = W.generate(spec); cfg = dict(W.matcher_config(spec), index_sort=index_sort)
    h, ix = load(B, cfg, d["tl_y"], d["tl_z"], d["tl_dydx"], d["tl_chamber"])
    try:
        check_index(cfg, ix, d["tl_y"], d["tl_z"], d["tl_chamber"])
        assert ix["n_tracklets"] == d["tl_y"].shape[0]
        assert ix["sort_kind"] == (1 if index_sort > 0 else 0)
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("index_sort", [-1, 0, 1])
@pytest.mark.parametrize("n", [1, 31, 4095, 4096, 4097, 3 * 4096 + 17, 200_003, 1_000_003])
@pytest.mark.parametrize("ybin_width", [0.0, 0.25])
def test_ragged_sizes_and_unusable_tracklets(B, base_cfg, n, ybin_width, index_sort):
    rng = np.random.default_rng(n)
    cfg = dict(base_cfg, ybin_width=ybin_width, index_sort=index_sort)
    y = rng.uniform(-70, 70, n).astype(np.float32)            # some beyond the binned range -> edge bins
    z = rng.uniform(-380, 380, n).astype(np.float32)
    d = rng.uniform(-0.5, 0.5, n).astype(np.float32)
    ch = rng.integers(-3, 545, n).astype(np.int32)            # some outside 0..539
    if n > 10:
        y[3] = np.nan; z[5] = np.inf; y[7] = -np.inf
    h, ix = load(B, cfg, y, z, d, ch)
    try:
        check_index(cfg, ix, y, z, ch)
        # index_sort = 0: up to 2^18 tracklets the counting sort runs as one cooperative launch (3), above it as the
        # multi-kernel counting sort (1)
        assert ix["sort_kind"] == (1 if index_sort > 0 or (index_sort == 0 and n > 1 << 18) else (3 if index_sort == 0 else 0))
        if ybin_width > 0:
            assert ix["ybin_width"] <= ybin_width
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("index_sort", [-1, 0, 1])
def test_skewed_keys_one_bin_and_reload(B, base_cfg, index_sort):
    """All tracklets in one bin (worst case for the scatter ranks; the counting sort hands a bin this long to the
    radix passes on the device), then a smaller reload on the same handle."""
    import torch
    base_cfg = dict(base_cfg, index_sort=index_sort)
    n = 50_000
    y = np.full(n, 1.25, np.float32); z = np.full(n, 4.0, np.float32); d = np.zeros(n, np.float32)
    ch = np.full(n, 7 * 30 + 2 * 6 + 3, np.int32)
    h, ix = load(B, base_cfg, y, z, d, ch)
    try:
        check_index(base_cfg, ix, y, z, ch)
        assert np.array_equal(ix["sorted_pos"], np.arange(n))
        assert ix["sort_kind"] == {1: 2, 0: 3, -1: 0}[index_sort]   # 3: the one-launch sort orders the long bin itself
        t = [torch.from_numpy(a[:100].copy()).cuda() for a in (y, z, d, ch)]
        B.trd_load_tracklets(h, *t)
        ix2 = B.trd_copy_index(h)
        check_index(base_cfg, ix2, y[:100], z[:100], ch[:100])
        B.trd_load_tracklets(h, *[a[:0] for a in t])          # empty load is legal
        ix3 = B.trd_copy_index(h)
        assert ix3["n_tracklets"] == 0 and not ix3["bin_first"].any()
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("n_dup", [2, 7, 32, 33])
def test_counting_sort_keeps_the_callers_order_inside_a_bin(B, base_cfg, n_dup):
    """Groups of n_dup tracklets share a bin (same chamber, y, z), scattered over the input: the counting sort must
    leave each group in input order (up to 32 per bin by its own per-bin pass, beyond that through the radix passes)."""
    rng = np.random.default_rng(n_dup)
    n_groups = 20_000
    ch_g = rng.integers(0, 540, n_groups).astype(np.int32)
    y_g = rng.uniform(-50, 50, n_groups).astype(np.float32); z_g = (8.0 * rng.integers(-40, 40, n_groups) + 4.0).astype(np.float32)
    order = rng.permutation(n_groups * n_dup)
    g = (np.arange(n_groups * n_dup) // n_dup)[order]
    y, z, ch = y_g[g], z_g[g], ch_g[g]
    d = rng.uniform(-0.5, 0.5, g.size).astype(np.float32)
    cfg = dict(base_cfg, index_sort=1, ybin_width=0.01)
    h, ix = load(B, cfg, y, z, d, ch)
    try:
        check_index(cfg, ix, y, z, ch)
        longest = np.diff(ix["bin_first"].astype(np.int64)).max()         # two groups may share a bin
        assert longest >= n_dup and ix["sort_kind"] == (1 if longest <= 32 else 2)
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("n_groups,n_dup", [(5000, 33), (300, 700), (60, 4096), (40, 5000), (3, 80_000)])
def test_one_launch_sort_orders_long_bins_itself(B, base_cfg, n_groups, n_dup):
    """Small loads (index_sort = 0, up to 2^18 tracklets) are indexed by ONE cooperative launch with no radix passes
    behind it: bins longer than 32 are put into the caller's order by a whole block -- a bitonic sort in shared memory
    up to 4096 tracklets, a walk over the caller's arrays beyond."""
    rng = np.random.default_rng(n_dup)
    ch_g = rng.integers(0, 540, n_groups).astype(np.int32)
    y_g = rng.uniform(-50, 50, n_groups).astype(np.float32); z_g = (8.0 * rng.integers(-40, 40, n_groups) + 4.0).astype(np.float32)
    order = rng.permutation(n_groups * n_dup)
    g = (np.arange(n_groups * n_dup) // n_dup)[order]
    y, z, ch = y_g[g], z_g[g], ch_g[g]
    d = rng.uniform(-0.5, 0.5, g.size).astype(np.float32)
    assert g.size <= 1 << 18
    cfg = dict(base_cfg, index_sort=0)
    h, ix = load(B, cfg, y, z, d, ch)
    try:
        check_index(cfg, ix, y, z, ch)
        assert ix["sort_kind"] == 3
        assert np.diff(ix["bin_first"].astype(np.int64)).max() >= n_dup
    finally:
        B.trd_destroy(h)
