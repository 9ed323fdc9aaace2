"""The parity tests proper: the CUDA path (through the C ABI) against the oracle, element by element, on
the same seeded inputs.  Criteria: BASELINE.json north_star, implemented in paper_2003_03174_b200.parity."""
import dataclasses

import numpy as np
import pytest

from oracle import oracle as O
from paper_2003_03174_b200 import parity as P, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_03174_b200 import binding, build
    build.build()
    return binding


def run_gpu(B, cfg, data, batch=None, in_place=False):
    import torch
    dev = B.to_device(data)
    n = data["x"].shape[0]
    h = B.trd_create(cfg)
    try:
        if "chamber_dx" in data:
            B.trd_set_chamber_dx(h, np.ascontiguousarray(data["chamber_dx"], np.float32))
        if data.get("n_interactions", 0) > 1:
            B.trd_load_tracklets_tf(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"], dev["tl_interaction"],
                                    data["n_interactions"])
        else:
            B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"])
        if batch is None:
            out = B.alloc_tracks_out(n)
            if in_place:
                out["par"], out["cov"], out["x"], out["sector"] = dev["par"], dev["cov"], dev["x"], dev["sector"]
            B.trd_match(h, dev, out)
            torch.cuda.synchronize()
            return B.to_numpy(out)
        parts = []
        for lo in range(0, n, batch):
            hi = min(n, lo + batch)
            part = dict(par=dev["par"][:, lo:hi].contiguous(), cov=dev["cov"][:, lo:hi].contiguous(),
                        x=dev["x"][lo:hi].contiguous(), sector=dev["sector"][lo:hi].contiguous())
            if "interaction" in dev:
                part["interaction"] = dev["interaction"][lo:hi].contiguous()
            parts.append(B.to_numpy(B.trd_match(h, part)))
        return {k: np.concatenate([p[k] for p in parts], axis=-1) for k in parts[0]}
    finally:
        B.trd_destroy(h)


FLIPS = []       # (what, tracks, fragile tracks, flipped chains) of every comparison of this session, printed at the end
STATS = dict(max_replays=0, chi2_max_rel_err=0.0, par_max_scaled_err=0.0)


def check_parity(got, want, cfg, data, lo=0, what="", max_flip_frac=0.02, record=True, **tol):
    """north_star criteria (parity.compare) + every flipped chain validated: on a track whose assignment differs the
    oracle is asked whether the CUDA path's chain is one of the results it reaches itself when its decisions closer
    than 1e-4 to their threshold are taken the other way (oracle.match_alternatives); if so, parameters, chi2,
    covariance and integers are compared against THAT result under the same tolerances.  The number of flips is bounded:
    measured 93 of 73 981 fragile tracks (0.13 %) on config 5 at full size and 0-1 elsewhere (BASELINE.md 5,
    profiles/r02_parity_report.txt); at most 2 % of the fragile tracks (and never more than 3 on small inputs) is accepted."""
    rep = P.compare(got, want, **tol)
    assert rep["ok"], {k: v for k, v in rep.items()}
    assert rep["n_evals_bad"] == 0
    STATS["chi2_max_rel_err"] = max(STATS["chi2_max_rel_err"], rep["chi2_max_rel_err"])
    STATS["par_max_scaled_err"] = max(STATS["par_max_scaled_err"], max(rep["par_max_scaled_err"]))
    flips = rep["flip_tracks"]
    if record:
        FLIPS.append((what, rep["n_tracks"], rep["n_fragile"], int(flips.shape[0])))
    if flips.shape[0]:
        n = want["x"].shape[0]
        alt = O.match_alternatives(cfg, data, flips + lo, got["idx"][:, :n][:, flips], eps=P.EPS_MARGIN)
        tol2 = {k: v for k, v in tol.items() if k != "eps_margin"}
        rep2 = P.compare_alternatives({k: v[..., :n] for k, v in got.items()}, alt, flips, **tol2)
        assert rep2["ok"], {k: v for k, v in rep2.items()}
        STATS["max_replays"] = max(STATS["max_replays"], rep2["max_replays"])
        assert flips.shape[0] <= max(3, max_flip_frac * rep["n_fragile"]), (flips.shape[0], rep["n_fragile"])
    return rep


@pytest.fixture(scope="module", autouse=True)
def _report_flips():
    yield
    tot = [sum(f[k] for f in FLIPS) for k in (1, 2, 3)]
    print(f"\n[parity] {len(FLIPS)} comparisons, {tot[0]} tracks, {tot[1]} fragile (margin < 1e-4), {tot[2]} flipped chains, "
          f"every one validated as an alternative result of the oracle (at most {STATS['max_replays']} replays); "
          f"chi2 max rel. error {STATS['chi2_max_rel_err']:.2e}, parameter error at most {STATS['par_max_scaled_err']:.2e} of "
          f"max(|p|, 0.1) on tracks with equal chains")
    for what, n, nf, nfl in FLIPS:
        if what:
            print(f"[parity] {what}: {n} tracks, {nf} fragile, {nfl} flips")


@pytest.mark.parametrize("name", ["tiny", "central", "central8", "pileup"])
def test_configs_1_to_4_full_parity(B, name):
    spec = W.CONFIGS[name]; d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d)
    rep = check_parity(got, want, cfg, d, what=f"config {name}")
    assert rep["n_fragile"] < 0.02 * spec.n_tracks


def test_config_5_scaled_down_in_batches(B):
    """Config 5's generator and cuts (nHyp = 4, 3 sigma) at 100k tracks and 400k noise tracklets (tracklet
    density 1/20 of the full config), matched as 4 batches against one loaded index, every track checked."""
    spec = W.scaled(W.CONFIGS["timeframe"], 100_000)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d, batch=spec.batch // 4)
    check_parity(got, want, cfg, d, what="config timeframe scaled to 100k tracks")


def test_dense_candidates_many_per_road(B):
    """Few tracks in dense noise (12M noise tracklets = about 2/3 of the per-chamber density of the full
    config 5): several in-road candidates per hypothesis and layer; all sub-warp widths (nHyp 1, 2, 3, 4, 8)."""
    for n_hyp, road, n_noise in ((4, 3.0, 12_000_000), (8, 5.0, 12_000_000), (3, 3.0, 4_000_000),
                                 (2, 3.0, 4_000_000), (1, 3.0, 4_000_000)):
        spec = dataclasses.replace(W.CONFIGS["tiny"], name="dense", number=7, n_tracks=3000, n_noise=n_noise,
                                   n_hyp=n_hyp, n_sigma_road=road)
        d = W.generate(spec); cfg = W.matcher_config(spec)
        want = O.match(cfg, d)
        assert want["counters"]["n_cand"] > want["counters"]["n_road"]
        got = run_gpu(B, cfg, d)
        check_parity(got, want, cfg, d, what=f"dense noise, n_hyp {n_hyp}")


def test_config_5_full_size_every_track(B):
    """BASELINE.json configs[4] at full size in the launch configuration bench.py times (one load of all
    ~18.8M tracklets, four trd_match calls of 500k tracks): ALL 2,000,000 tracks are compared with the oracle, which
    matches them in eight slices against the full tracklet set ("parity is still checked on all 2M
    tracks"); every flipped chain is validated as everywhere else."""
    spec = W.CONFIGS["timeframe"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    got = run_gpu(B, cfg, d, batch=spec.batch)
    n_checked = n_fragile = n_flips = 0
    step = 250_000
    for lo in range(0, spec.n_tracks, step):
        hi = min(spec.n_tracks, lo + step)
        want = O.match(cfg, d, lo=lo, hi=hi)
        part = {k: v[..., lo:hi] for k, v in got.items()}
        rep = check_parity(part, want, cfg, d, lo=lo, record=False)
        n_checked += hi - lo; n_fragile += rep["n_fragile"]; n_flips += int(rep["flip_tracks"].shape[0])
        del want
    assert n_checked == spec.n_tracks == 2_000_000
    FLIPS.append(("config timeframe at full size", n_checked, n_fragile, n_flips))
    # properties that hold at any size
    att = got["idx"] >= 0
    assert np.array_equal(att.sum(axis=0), got["n_matched"])
    assert got["idx"].max() < d["tl_y"].shape[0]
    lay = d["tl_chamber"][np.where(att, got["idx"], 0)] % 6
    assert np.all(lay[att] == np.nonzero(att)[0])                          # layer l holds a layer-l tracklet
    sec_tl = d["tl_chamber"][np.where(att, got["idx"], 0)] // 30
    assert np.all(sec_tl[5][att[5]] == got["sector"][att[5]])              # last attached = final sector
    assert np.all(got["chi2"] >= 0) and np.all(got["chi2"] < 15.0 * 6)
    assert np.all(np.isfinite(got["par"])) and np.all(np.isfinite(got["cov"]))


def test_edge_cases(B, base_cfg):
    import torch
    spec = W.CONFIGS["tiny"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    # in-place outputs (out->par == in->par)
    check_parity(run_gpu(B, cfg, d, in_place=True), want, cfg, d)
    # ragged batches
    check_parity(run_gpu(B, cfg, d, batch=333), want, cfg, d)
    # dead seeds: |sin(phi)| >= max_snp, sector outside 0..17
    d2 = dict(d); d2["par"] = d["par"].copy(); d2["par"][2, 0] = 0.96
    d2["sector"] = d["sector"].copy(); d2["sector"][1] = 99; d2["sector"][2] = -1
    want2 = O.match(cfg, d2); got2 = run_gpu(B, cfg, d2)
    check_parity(got2, want2, cfg, d2)
    assert got2["idx"][:, :3].max() == -1 and got2["n_matched"][:3].max() == 0
    # no tracklets at all: every layer skipped, state = last alive propagation
    d3 = dict(d); d3.update(tl_y=d["tl_y"][:0], tl_z=d["tl_z"][:0], tl_dydx=d["tl_dydx"][:0], tl_chamber=d["tl_chamber"][:0])
    want3 = O.match(cfg, d3); got3 = run_gpu(B, cfg, d3)
    check_parity(got3, want3, cfg, d3)
    assert got3["idx"].max() == -1 and np.all(got3["x"] >= 247.0)
    # zero tracks, and trd_match before any load
    h = B.trd_create(cfg)
    try:
        dev = B.to_device(d)
        with pytest.raises(B.TrdError) as e:
            B.trd_match(h, dev)
        assert e.value.code == B.TRD_E_STATE
        B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"])
        empty = dict(par=dev["par"][:, :0].contiguous(), cov=dev["cov"][:, :0].contiguous(),
                     x=dev["x"][:0].contiguous(), sector=dev["sector"][:0].contiguous())
        out = B.trd_match(h, empty)
        assert out["x"].numel() == 0
        with pytest.raises(B.TrdError) as e:                   # NULL array -> TRD_E_ARG, not a crash
            import ctypes as C
            tin, tout = B.TrdTracksIn(), B.TrdTracksOut()
            rc = B.lib().trd_match(h, C.byref(tin), C.byref(tout), 5, None)
            B._check(h, rc)
        assert e.value.code == B.TRD_E_ARG
        assert B.trd_device_bytes(h) > 0 and B.trd_kernel_launches(h) > 0
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("variant", ["exact_z", "bz0", "bz_neg", "fine_bins", "low_pt"])
def test_variants(B, variant):
    spec = dataclasses.replace(W.CONFIGS["central"], n_hyp=4, number=11)
    over = {}
    if variant == "exact_z":
        spec = dataclasses.replace(spec, exact_z=True)         # tracklet z not on pad-row centres
    elif variant == "bz0":
        spec = dataclasses.replace(spec, bz=0.0)               # straight lines
    elif variant == "bz_neg":
        spec = dataclasses.replace(spec, bz=-0.5)
    elif variant == "fine_bins":
        over = dict(ybin_width=0.1)
    elif variant == "low_pt":
        spec = dataclasses.replace(spec, pt_spectrum="exp")    # sector crossings, tracks that curl up
    d = W.generate(spec); cfg = dict(W.matcher_config(spec), **over)
    want = O.match(cfg, d); got = run_gpu(B, cfg, d)
    check_parity(got, want, cfg, d, what=f"variant {variant}")


def test_host_entry_points_equal_device_entry_points(B):
    spec = W.CONFIGS["central8"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    dev_out = run_gpu(B, cfg, d)
    h = B.trd_create(cfg)
    try:
        B.trd_load_tracklets_host(h, d["tl_y"], d["tl_z"], d["tl_dydx"], d["tl_chamber"])
        out = B.trd_match_host(h, d)
    finally:
        B.trd_destroy(h)
    for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
        np.testing.assert_array_equal(out[k], dev_out[k])


def test_quality_trend_of_the_paper(B):
    """purity ~1 at low density and falling with density (config 1 >= 2 >= 4)."""
    pur = []
    for name in ("tiny", "central", "pileup"):
        spec = W.CONFIGS[name]; d = W.generate(spec)
        got = run_gpu(B, W.matcher_config(spec), d)
        q = W.efficiency_purity(got["idx"].T, d)
        pur.append(q["purity"])
        assert q["efficiency"] > 0.9
    assert pur[0] >= pur[1] >= pur[2] and pur[0] > 0.99


@pytest.mark.parametrize("name", ["tiny", "central8", "pileup"])
def test_track_binning_does_not_change_results(B, name):
    """trd_config.track_binning only changes the processing order (tracks.cu): bit-identical outputs with
    binning forced on and off, also with in-place outputs and ragged batches."""
    spec = W.CONFIGS[name]; d = W.generate(spec); cfg = W.matcher_config(spec)
    off = run_gpu(B, dict(cfg, track_binning=-1), d)
    on = run_gpu(B, dict(cfg, track_binning=1), d)
    on_inplace = run_gpu(B, dict(cfg, track_binning=1), d, in_place=True)
    on_ragged = run_gpu(B, dict(cfg, track_binning=1), d, batch=777)
    for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
        np.testing.assert_array_equal(on[k], off[k])
        np.testing.assert_array_equal(on_inplace[k], off[k])
        np.testing.assert_array_equal(on_ragged[k], off[k])
    want = O.match(cfg, d)
    check_parity(on, want, cfg, d)


@pytest.mark.parametrize("n_ia,key_bits", [(2, 12), (7, 14), (40, 16), (64, 17)])
def test_track_sort_over_every_key_width(B, n_ia, key_bits):
    """The track key (interaction, sector, z row) of the binned path is counting-sorted up to 16 bits -- its histogram
    scanned by 1 to 16 blocks that look back over the tile sums before them (tracks.cu scan_hist) -- and radix-sorted
    above: one block (12 bits), four, sixteen, and the radix path, each bit-identical to the unbinned kernel, two
    batches in a row through the same scratch."""
    spec = dataclasses.replace(W.CONFIGS["pileup"], n_interactions=n_ia)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    n_keys = n_ia * cfg["n_sectors"] * 2 * (int(np.ceil(cfg["z_max"] / cfg["pad_length"])) + 1)     # index.cu: z rows
    assert max(12, int(np.ceil(np.log2(n_keys)))) == key_bits
    off = run_gpu(B, dict(cfg, track_binning=-1), d)
    on = run_gpu(B, dict(cfg, track_binning=1), d, batch=13001)
    for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
        np.testing.assert_array_equal(on[k], off[k], err_msg=k)


@pytest.mark.parametrize("name", ["central8", "pileup"])
def test_zero_penalty_scores_of_zero(B, name):
    """chi2_penalty = 0: the skip-children carry score 0, whose child keys (score bits << 32 | parent | position) are
    denormal when read as doubles -- the match kernel compares keys as doubles (match.cu) and must still rank them
    exactly like the oracle's tuples; hypotheses that attach a tracklet compete with chains of skips."""
    spec = W.CONFIGS[name]; d = W.generate(spec); cfg = dict(W.matcher_config(spec), chi2_penalty=0.0)
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d)
    rep = check_parity(got, want, cfg, d)
    assert rep["n_assign_mismatch"] == 0
    assert got["n_matched"].max() == 0                                # nothing beats a chain of free skips


@pytest.mark.parametrize("name,extra", [("central8", {}), ("pileup", dict(chamber_dx_sigma=0.3, res_model=1))])
def test_index_sort_does_not_change_results(B, name, extra):
    """trd_config.index_sort picks the device sort of trd_load_tracklets (index.cu): the store and therefore every
    output are bit-identical with the radix passes and with the counting sort, also with displaced chambers (the
    per-tracklet offsets travel with the store) and with every tracklet given twice (ties by the caller's order)."""
    spec = dataclasses.replace(W.CONFIGS[name], **extra); d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    for dup in (False, True):
        if dup:
            d = dict(d, **{k: np.concatenate([d[k], d[k]]) for k in d if k.startswith("tl_")})
        radix = run_gpu(B, dict(cfg, index_sort=-1), d)
        counting = run_gpu(B, dict(cfg, index_sort=1), d)
        for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
            np.testing.assert_array_equal(counting[k], radix[k])
        if dup:
            n0 = d["tl_y"].shape[0] // 2
            assert np.all(counting["idx"] < n0)                      # of two equal tracklets the first one given wins
        else:
            check_parity(counting, want, cfg, d)


def test_pipelined_host_entry_points(B):
    """trd_match_host_async + trd_wait_host: nine batches through the four-slot ring (the fifth call has to
    retire the first), pinned and pageable buffers, two consecutive loads on one handle; bit-equal to the
    device entry points."""
    spec = W.CONFIGS["pileup"]; d = W.generate(spec); cfg = dict(W.matcher_config(spec), track_binning=1)
    want = run_gpu(B, cfg, d)
    n = spec.n_tracks
    bounds = [(lo, min(n, lo + 2801)) for lo in range(0, n, 2801)]
    h = B.trd_create(cfg)
    try:
        for pinned in (True, False):
            B.trd_load_tracklets_host(h, d["tl_y"][:1000].copy(), d["tl_z"][:1000].copy(), d["tl_dydx"][:1000].copy(),
                                      d["tl_chamber"][:1000].copy())          # superseded by the next load
            B.trd_load_tracklets_host(h, d["tl_y"], d["tl_z"], d["tl_dydx"], d["tl_chamber"])
            ins = [dict(par=np.ascontiguousarray(d["par"][:, lo:hi]), cov=np.ascontiguousarray(d["cov"][:, lo:hi]),
                        x=np.ascontiguousarray(d["x"][lo:hi]), sector=np.ascontiguousarray(d["sector"][lo:hi]))
                   for lo, hi in bounds]
            outs = [B.alloc_tracks_out_host(hi - lo, pinned=pinned) for lo, hi in bounds]
            for t, o in zip(ins, outs):
                B.trd_match_host_async(h, t, o)
            B.trd_wait_host(h)
            for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
                got = np.concatenate([o[k] for o in outs], axis=-1)
                np.testing.assert_array_equal(got, want[k])
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("name,binning", [("central8", -1), ("pileup", 1)])
def test_load_and_match_can_be_captured_in_a_cuda_graph(B, name, binning):
    """After one warm-up pass the device entry points allocate nothing (buffers only grow), create no stream and never
    synchronise: trd_load_tracklets + trd_match can be captured in a CUDA graph and replayed; the replay writes the same
    results (unbinned and binned path)."""
    import torch
    spec = W.CONFIGS[name]; d = W.generate(spec); cfg = dict(W.matcher_config(spec), track_binning=binning)
    want = run_gpu(B, cfg, d)
    dev = B.to_device(d); n = d["x"].shape[0]
    h = B.trd_create(cfg)
    try:
        out = B.alloc_tracks_out(n)
        side = torch.cuda.Stream()

        def step():
            B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"], stream=side)
            B.trd_match(h, dev, out, stream=side)

        with torch.cuda.stream(side):
            step()                                           # warm-up: every buffer has its size
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            step()
        for k in out:
            out[k].fill_(-7)
        for _ in range(2):
            graph.replay()
        torch.cuda.synchronize()
        got = B.to_numpy(out)
        for k in ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals"):
            np.testing.assert_array_equal(got[k], want[k], err_msg=k)
        del graph
    finally:
        B.trd_destroy(h)


def test_host_rows_need_not_be_adjacent(B):
    """The host entry points send rows that follow each other in the caller's memory as one copy (host_api.cu); rows of
    trd_tracks_in / trd_tracks_out are independent pointers, though: here every row is an allocation of its own, except
    a few that are made adjacent on purpose (cov rows 3-6 and idx rows 1-2), in an order that does not ascend."""
    import ctypes as C
    spec = W.CONFIGS["central8"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    want = run_gpu(B, cfg, d)
    n = d["x"].shape[0]
    keep = []

    def own(a):
        keep.append(np.ascontiguousarray(a).copy())
        return keep[-1]

    def ptr(a):
        return a.ctypes.data

    tin, tout = B.TrdTracksIn(), B.TrdTracksOut()
    par_rows = [own(d["par"][k]) for k in (4, 2, 0, 3, 1)]                        # allocated in another order
    tin.par[:] = [ptr(par_rows[(4, 2, 0, 3, 1).index(k)]) for k in range(5)]
    block = own(d["cov"][3:7])                                                     # four adjacent rows
    cov_rows = {k: own(d["cov"][k]) for k in range(15) if not 3 <= k < 7}
    tin.cov[:] = [ptr(block) + 4 * n * (k - 3) if 3 <= k < 7 else ptr(cov_rows[k]) for k in range(15)]
    x, sector = own(d["x"]), own(d["sector"])
    tin.x, tin.sector = ptr(x), ptr(sector)
    o_idx_pair = np.empty((2, n), np.int32)
    o_idx = {l: np.empty(n, np.int32) for l in (0, 3, 4, 5)}
    tout.tracklet_idx[:] = [ptr(o_idx_pair) + 4 * n * (l - 1) if l in (1, 2) else ptr(o_idx[l]) for l in range(6)]
    o_par = [np.empty(n, np.float32) for _ in range(5)][::-1]
    o_cov = [np.empty(n, np.float32) for _ in range(15)]
    tout.par[:] = [ptr(a) for a in o_par]
    tout.cov[:] = [ptr(a) for a in o_cov]
    o = {k: np.empty(n, t) for k, t in (("x", np.float32), ("sector", np.int32), ("chi2", np.float32),
                                         ("n_matched", np.int32), ("n_evals", np.int32))}
    tout.x, tout.sector, tout.chi2, tout.n_matched, tout.n_cand_evals = (ptr(o[k]) for k in ("x", "sector", "chi2", "n_matched", "n_evals"))
    h = B.trd_create(cfg)
    try:
        B.trd_load_tracklets_host(h, d["tl_y"], d["tl_z"], d["tl_dydx"], d["tl_chamber"])
        assert B.lib().trd_match_host(h, C.byref(tin), C.byref(tout), n, None) == B.TRD_OK
    finally:
        B.trd_destroy(h)
    got_idx = np.stack([o_idx_pair[l - 1] if l in (1, 2) else o_idx[l] for l in range(6)])
    np.testing.assert_array_equal(got_idx, want["idx"])
    np.testing.assert_array_equal(np.stack(o_par), want["par"])
    np.testing.assert_array_equal(np.stack(o_cov), want["cov"])
    for k in o:
        np.testing.assert_array_equal(o[k], want[k])


@pytest.mark.parametrize("name,n_hyp", [("central", 1), ("central8", 8), ("pileup", 4)])
def test_resolution_model_and_pad_tilt(B, name, n_hyp):
    """sigma_y(sin phi), sigma_dydx(sin phi) and the +-2 degree pad tilt
    (res_model = 1), inputs generated with the same model; same parity criteria as the configs."""
    spec = dataclasses.replace(W.CONFIGS[name], res_model=1, n_hyp=n_hyp)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    assert cfg["res_model"] == 1 and cfg["tan_tilt"] > 0.03
    want = O.match(cfg, d)
    check_parity(run_gpu(B, cfg, d), want, cfg, d, what=f"resolution model + pad tilt, {name}")
    check_parity(run_gpu(B, dict(cfg, track_binning=1), d, batch=1777), want, cfg, d)
    # the model matters: the same input matched without the tilt loses tracklets
    plain = run_gpu(B, dict(cfg, tan_tilt=0.0), d)
    assert plain["n_matched"].sum() < 0.97 * want["n_matched"].sum()


def test_resolution_model_dense(B):
    spec = dataclasses.replace(W.CONFIGS["tiny"], name="dense", number=8, n_tracks=3000, n_noise=12_000_000, n_hyp=4,
                               res_model=1)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    assert want["counters"]["n_cand"] > want["counters"]["n_road"]
    check_parity(run_gpu(B, cfg, d), want, cfg, d, what="resolution model, dense noise")


@pytest.mark.parametrize("name,n_ia,n_hyp", [("central", 4, 1), ("pileup", 5, 4), ("central8", 7, 8)])
def test_time_frame_association(B, name, n_ia, n_hyp):
    """tracklets are matched only to tracks of the same interaction.
    Pile-up config with its 5 overlapping events as 5 interactions, among others; binned and unbinned batches."""
    spec = dataclasses.replace(W.CONFIGS[name], n_interactions=n_ia, n_hyp=n_hyp)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d)
    check_parity(got, want, cfg, d, what=f"time-frame association, {name}")
    check_parity(run_gpu(B, dict(cfg, track_binning=1), d, batch=2111), want, cfg, d)
    att = got["idx"] >= 0                                     # every attached tracklet is of the track's interaction
    ia_tl = d["tl_interaction"][np.where(att, got["idx"], 0)]
    assert np.all(ia_tl[att] == np.broadcast_to(d["interaction"], att.shape)[att])


def test_time_frame_association_at_scale_and_bad_ids(B):
    """Config 5's generator at 200k tracks as 100 interactions of 2000 tracks (~2000 tracks per central
    event), four batches; tracks and tracklets with ids out of range; NULL interaction array -> TRD_E_ARG."""
    spec = dataclasses.replace(W.scaled(W.CONFIGS["timeframe"], 200_000), n_interactions=100)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    d["interaction"][:5] = [-1, 100, 12345, 3, 99]
    d["tl_interaction"][::97] = 100
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d, batch=50_000)
    check_parity(got, want, cfg, d, what="time-frame association, 200k tracks in 100 interactions")
    assert got["n_matched"][:3].max() == 0
    import torch
    h = B.trd_create(cfg)
    try:
        dev = B.to_device(d)
        B.trd_load_tracklets_tf(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"], dev["tl_interaction"], 100)
        assert B.trd_get_index_info(h)["n_interactions"] == 100
        no_ia = {k: v for k, v in dev.items() if k != "interaction"}
        with pytest.raises(B.TrdError) as e:
            B.trd_match(h, no_ia)
        assert e.value.code == B.TRD_E_ARG
        B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"])     # back to no association
        assert B.trd_get_index_info(h)["n_interactions"] == 1
        B.trd_match(h, no_ia); torch.cuda.synchronize()
    finally:
        B.trd_destroy(h)


@pytest.mark.parametrize("name,n_hyp,extra", [("central", 1, {}), ("pileup", 4, {}), ("central8", 8, dict(res_model=1, n_interactions=3))])
def test_two_stage_propagation_with_displaced_chambers(B, name, n_hyp, extra):
    """chambers displaced radially by N(0, 0.3 cm); linear extrapolation for
    road and chi2, exact re-propagation before the update; also combined with the resolution model and association."""
    spec = dataclasses.replace(W.CONFIGS[name], chamber_dx_sigma=0.3, n_hyp=n_hyp, **extra)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d)
    check_parity(got, want, cfg, d, what=f"two-stage propagation, {name}")
    check_parity(run_gpu(B, dict(cfg, track_binning=1), d, batch=1999), want, cfg, d)
    assert np.abs(got["x"] - 364.0).max() > 0.3                       # states live at the displaced radii
    # the offsets matter, and clearing them gives the plain matcher again
    plain_want = O.match(cfg, {k: v for k, v in d.items() if k != "chamber_dx"})
    assert plain_want["n_matched"].sum() < 0.98 * want["n_matched"].sum()
    h = B.trd_create(cfg)
    try:
        B.trd_set_chamber_dx(h, d["chamber_dx"])
        B.trd_set_chamber_dx(h, None)
        dev = B.to_device(d)
        with pytest.raises(B.TrdError) as e:                          # the index was dropped
            B.trd_match(h, dev)
        assert e.value.code == B.TRD_E_STATE
        with pytest.raises(B.TrdError) as e:
            B.trd_set_chamber_dx(h, np.zeros(17, np.float32))
        assert e.value.code == B.TRD_E_ARG
    finally:
        B.trd_destroy(h)
    no_dx = {k: v for k, v in d.items() if k != "chamber_dx"}
    check_parity(run_gpu(B, cfg, no_dx), plain_want, cfg, no_dx)


MATERIAL = dict(x_over_x0=W.X_OVER_X0, eloss=W.ELOSS, eloss_fluct=W.ELOSS_FLUCT)


@pytest.mark.parametrize("name,n_hyp,extra", [("central", 1, {}), ("pileup", 4, {}),
                                              ("central8", 8, dict(res_model=1, n_interactions=3, chamber_dx_sigma=0.3))])
def test_material_scattering_and_energy_loss(B, name, n_hyp, extra):
    """SURVEY.md 8(f) NEXT#3, material half ("taking into account ... energy loss"; R32, R33): a slab
    in front of every layer, the generator scatters and slows the true particles; alone and combined with the
    measurement model, the association and displaced chambers."""
    spec = dataclasses.replace(W.CONFIGS[name], n_hyp=n_hyp, **MATERIAL, **extra)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    tol = {}                                                          # north_star tolerances
    got = run_gpu(B, cfg, d)
    check_parity(got, want, cfg, d, what=f"material, {name}", **tol)
    check_parity(run_gpu(B, dict(cfg, track_binning=1), d, batch=1999), want, cfg, d, **tol)
    # the material matters on these inputs, and the filter without it is the plain one
    none = dict(cfg, x_over_x0=0.0, eloss=0.0)
    plain_want = O.match(none, d)
    assert plain_want["n_matched"].sum() < 0.99 * want["n_matched"].sum()
    check_parity(run_gpu(B, none, d), plain_want, none, d, **tol)
    # scattering only / energy loss only
    for part in (dict(cfg, eloss=0.0), dict(cfg, x_over_x0=0.0)):
        w = O.match(part, d)
        check_parity(run_gpu(B, part, d), w, part, d, **tol)
    for bad in (dict(cfg, x_over_x0=-1.0), dict(cfg, eloss=float("nan")), dict(cfg, mass=-0.1)):
        with pytest.raises(B.TrdError) as e:
            B.trd_create(bad)
        assert e.value.code == B.TRD_E_ARG


FIELD = dict(bz_r2=W.BZ_R2, bz_z2=W.BZ_Z2)


@pytest.mark.parametrize("name,n_hyp,extra", [("central", 1, {}), ("pileup", 4, {}),
                                              ("central8", 8, dict(MATERIAL, res_model=1, n_interactions=3, chamber_dx_sigma=0.3))])
def test_field_inhomogeneity(B, name, n_hyp, extra):
    """SURVEY.md 8(f) NEXT#3, field half ("taking into account inhomogenities of the magnetic field"; DESIGN.md
    R35): Bz falls by 2 % towards the outer layers; the generator integrates the true particles numerically; alone and
    combined with every other extension."""
    spec = dataclasses.replace(W.CONFIGS[name], n_hyp=n_hyp, **FIELD, **extra)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    want = O.match(cfg, d)
    tol = {}                                                          # north_star tolerances
    got = run_gpu(B, cfg, d)
    check_parity(got, want, cfg, d, what=f"field inhomogeneity, {name}", **tol)
    check_parity(run_gpu(B, dict(cfg, track_binning=1), d, batch=1999), want, cfg, d, **tol)
    # the inhomogeneity matters on these inputs (chi2 grows when it is ignored) and the uniform filter is the plain one
    uni = dict(cfg, bz_r2=0.0, bz_z2=0.0)
    plain_want = O.match(uni, d)
    m = (want["n_matched"] > 0) & (plain_want["n_matched"] == want["n_matched"])
    assert plain_want["chi2"][m].sum() > 1.005 * want["chi2"][m].sum()
    check_parity(run_gpu(B, uni, d), plain_want, uni, d, **tol)
    for part in (dict(cfg, bz_z2=0.0), dict(cfg, bz_r2=0.0)):
        w = O.match(part, d)
        check_parity(run_gpu(B, part, d), w, part, d, **tol)
    for bad in (dict(cfg, bz_r2=float("inf")), dict(cfg, bz_r2=-1e-5)):
        with pytest.raises(B.TrdError) as e:
            B.trd_create(bad)
        assert e.value.code == B.TRD_E_ARG


def test_material_stops_slow_particles(B):
    """Degenerate case of R33: a loss no track can pay -- every hypothesis stops at the first slab on both sides."""
    spec = dataclasses.replace(W.CONFIGS["central"], n_hyp=2)
    d = W.generate(spec); cfg = dict(W.matcher_config(spec), x_over_x0=0.01, eloss=50.0, eloss_fluct=0.1, mass=0.13957)
    want = O.match(cfg, d)
    got = run_gpu(B, cfg, d)
    assert want["n_matched"].sum() == 0 and got["n_matched"].sum() == 0
    check_parity(got, want, cfg, d)
    assert np.all(got["x"] == 300.0)                                  # reached the first plane, stopped in its slab


def test_random_configurations(B):
    """Seeded sweep over the knobs of trd_config and of the generator (24 combinations, 3000 tracks each): every
    sub-warp width, roads, cuts, penalties, field values, spectra, measurement model, association, displaced
    chambers, bin widths, track binning."""
    rng = np.random.default_rng(20030317)
    for k in range(24):
        n_hyp = int(rng.integers(1, 9))
        spec = dataclasses.replace(
            W.CONFIGS["central"], name=f"rand{k}", number=100 + k, n_tracks=3000, n_noise=int(rng.choice([3000, 60000, 600000])),
            n_hyp=n_hyp, n_sigma_road=float(rng.choice([2.0, 3.0, 5.0])), bz=float(rng.choice([-0.5, 0.2, 0.5])),
            pt_spectrum=str(rng.choice(["loguniform", "exp"])), res_model=int(rng.integers(0, 2)),
            n_interactions=int(rng.choice([0, 0, 3, 40])), chamber_dx_sigma=float(rng.choice([0.0, 0.0, 0.2])),
            efficiency=float(rng.choice([0.6, 0.9, 1.0])), **(MATERIAL if k % 4 == 3 else {}), **(FIELD if k % 3 == 2 else {}))
        d = W.generate(spec)
        cfg = dict(W.matcher_config(spec), chi2_cut=float(rng.choice([5.0, 15.0, 30.0])),
                   chi2_penalty=float(rng.choice([5.0, 15.0, 25.0])), ybin_width=float(rng.choice([0.0, 0.0, 0.05, 2.0])),
                   track_binning=int(rng.choice([-1, 0, 1])), n_sigma_angle=float(rng.choice([3.0, 4.0])))
        want = O.match(cfg, d)
        got = run_gpu(B, cfg, d, batch=None if k % 3 else 1024)
        # north_star tolerances throughout: y and sin(phi) accumulate in double in the CUDA path
        check_parity(got, want, cfg, d)


@pytest.mark.parametrize("name,extra", [("central", {}), ("pileup", dict(res_model=1, chamber_dx_sigma=0.3)), ("central8", {}),
                                        ("pileup", MATERIAL), ("central", dict(MATERIAL, res_model=1, chamber_dx_sigma=0.3, efficiency=0.6)),
                                        ("central", FIELD), ("pileup", dict(MATERIAL, **FIELD)),
                                        ("timeframe", dict(n_tracks=200000, n_noise=800000, batch=None))])   # config 5's density, a tenth of it
def test_refit_parity(B, name, extra):
    """SURVEY.md 8(f) NEXT#4 (PAPER.md:33 step 3): the CUDA refit against the oracle's refit, both fed the SAME matched
    chains (the oracle's, cast to float32), under the north_star criteria (parameter floor 5e-5, see below)."""
    import torch
    spec = dataclasses.replace(W.CONFIGS[name], **extra)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    m = O.match(cfg, d)
    m32 = dict(idx=m["idx"], par=m["par"].astype(np.float32), cov=m["cov"].astype(np.float32), x=m["x"].astype(np.float32),
               sector=m["sector"])
    want = O.refit(cfg, d, {k: (v.astype(np.float64) if v.dtype == np.float32 else v) for k, v in m32.items()})
    h = B.trd_create(cfg)
    try:
        if "chamber_dx" in d:
            B.trd_set_chamber_dx(h, d["chamber_dx"])
        dev = B.to_device(d)
        B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"])
        got = B.to_numpy(B.trd_refit(h, {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in m32.items()}))
        # refit of the CUDA matcher's own output runs too (chains agree with the oracle's up to fragile tracks)
        own = B.to_numpy(B.trd_refit(h, B.trd_match(h, dev)))
    finally:
        B.trd_destroy(h)
    # same discrete outcome on every track (sector, tracklets used), then the north_star criteria; the absolute floor
    # of the parameters is 5e-5 here.  The refit starts from a covariance reset to variances 600 times the tracklet's, so
    # its first updates subtract nearly equal float32 numbers in the unmeasured block (covariance good to 7e-4 of
    # sqrt(C_ii C_jj) afterwards, against 3e-6 in the matcher), the gain inherits that, and the final extrapolation of
    # 53-117 cm turns it into a few 1e-5 cm of y for a curling 0.3 GeV/c track that starts at |sin(phi)| = 0.94
    # (observed: 2 of 160 000 tracks above 1e-5 cm, 1.7e-5 and 3.5e-5, the latter 4e-5 of its own sigma_y)
    same = (got["n_used"] == want["n_used"]) & (got["sector"] == want["sector"])
    assert same.all(), int((~same).sum())
    assert np.array_equal(got["x"].astype(np.float64), want["x"].astype(np.float32).astype(np.float64))
    used = want["n_used"] >= 2
    assert used.mean() > 0.9
    dp = np.abs(got["par"].astype(np.float64) - want["par"])
    tol = np.maximum(P.PAR_RTOL * np.abs(want["par"]), 5e-5)
    assert np.all(dp[:, used] <= tol[:, used]), float((dp / tol)[:, used].max())
    thru = want["n_used"] == 0
    assert np.array_equal(got["par"][:, thru], m32["par"][:, thru])               # passed through unchanged
    dc = np.abs(got["chi2"].astype(np.float64) - want["chi2"])
    assert np.all(dc[used] <= P.CHI2_RTOL * want["chi2"][used] + 1e-9)
    scale = np.sqrt(np.abs(np.stack([want["cov"][i * (i + 1) // 2 + i] * want["cov"][j * (j + 1) // 2 + j]
                                     for i in range(5) for j in range(i + 1)])))
    dcov = np.abs(got["cov"].astype(np.float64) - want["cov"])
    assert np.all(dcov[:, used] <= 2e-3 * scale[:, used])
    assert (own["n_used"] >= 2).mean() > 0.9 and np.all(own["x"][own["n_used"] >= 2] == 247.0)
