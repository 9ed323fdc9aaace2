"""trd_match_static: the entry point that allocates nothing (its scratch is a file-scope device array of the library,
include/trdmatch.h) against the existing trd_match on the same inputs.

The order in which tracks are processed changes no result, so the tolerance is the one the binning tests use
(tests/test_gpu_parity.py, test_track_binning_does_not_change_results): bit-identical outputs.  Every case makes
two calls in a row on one stream, without a synchronisation between them, on different inputs: the second call finds
the first call's records, keys, permutation and histogram in the shared array.

Collected last on purpose (file name): the suite runs with pytest -x.
"""

import numpy as np
import pytest

from paper_2003_03174_b200 import workloads as W

pytestmark = pytest.mark.gpu

KEYS = ("idx", "par", "cov", "x", "sector", "chi2", "n_matched", "n_evals")


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_03174_b200 import binding, build
    build.build()
    return binding


def part_of(dev, lo, hi):
    return dict(par=dev["par"][:, lo:hi].contiguous(), cov=dev["cov"][:, lo:hi].contiguous(),
                x=dev["x"][lo:hi].contiguous(), sector=dev["sector"][lo:hi].contiguous())


def loaded_handle(B, cfg, dev):
    h = B.trd_create(cfg)
    B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"])
    return h


def same(got, want):
    for k in KEYS:
        np.testing.assert_array_equal(got[k], want[k], err_msg=k)


@pytest.mark.parametrize("name,n_tracks,second", [
    ("pileup", 32768, (10000, 17777)),        # the maximum, then a ragged slice of other tracks (n_hyp = 4)
    ("central8", 5000, (0, 5000)),            # n_hyp = 8; the same batch twice
    ("tiny", 1000, (1, 130)),                 # n_hyp = 1: one thread per track
])
def test_two_calls_in_a_row_match_the_existing_path(B, name, n_tracks, second):
    import torch
    spec = W.scaled(W.CONFIGS[name], n_tracks) if n_tracks != W.CONFIGS[name].n_tracks else W.CONFIGS[name]
    d = W.generate(spec); cfg = W.matcher_config(spec)
    dev = B.to_device(d)
    n = d["x"].shape[0]
    assert n == n_tracks <= B.TRD_STATIC_MAX_TRACKS
    lo, hi = second
    first_in, second_in = part_of(dev, 0, n), part_of(dev, lo, hi)
    h = loaded_handle(B, cfg, dev)
    try:
        # the existing path, binning off and forced on (the instantiation the static path runs)
        want_1 = B.to_numpy(B.trd_match(h, first_in))
        want_2 = B.to_numpy(B.trd_match(h, second_in))
        out_1, out_2 = B.alloc_tracks_out(n), B.alloc_tracks_out(hi - lo)
        B.trd_match_static(h, second_in, out_2)               # warm-up: kernels loaded, symbol address resolved
        torch.cuda.synchronize()
        for o in (out_1, out_2):
            for k in o:
                o[k].fill_(-7)
        torch.cuda.synchronize()
        owned, free_before = B.trd_device_bytes(h), torch.cuda.mem_get_info()[0]
        B.trd_match_static(h, first_in, out_1)                # two calls in a row, no synchronisation between them
        B.trd_match_static(h, second_in, out_2)
        torch.cuda.synchronize()
        assert B.trd_device_bytes(h) == owned                 # nothing reserved by the handle
        assert torch.cuda.mem_get_info()[0] == free_before    # nothing allocated on the device at all
        same(B.to_numpy(out_1), want_1)
        same(B.to_numpy(out_2), want_2)
        # and the other way round: the small batch first, the large one over its remains
        B.trd_match_static(h, second_in, out_2)
        B.trd_match_static(h, first_in, out_1)
        torch.cuda.synchronize()
        same(B.to_numpy(out_1), want_1)
        same(B.to_numpy(out_2), want_2)
    finally:
        B.trd_destroy(h)
    hb = loaded_handle(B, dict(cfg, track_binning=1), dev)
    try:
        same(B.to_numpy(B.trd_match(hb, first_in)), want_1)   # the binned existing path says the same
    finally:
        B.trd_destroy(hb)


def test_two_handles_share_the_array_when_serialised(B):
    """The array belongs to the library, not to a handle: calls through different handles on one stream follow each
    other on the GPU and each finds the other's remains."""
    import torch
    spec = W.CONFIGS["central"]; d = W.generate(spec)
    cfg_1 = W.matcher_config(spec); cfg_4 = dict(cfg_1, n_hyp=4)
    dev = B.to_device(d); n = d["x"].shape[0]
    tracks = part_of(dev, 0, n)
    h1, h4 = loaded_handle(B, cfg_1, dev), loaded_handle(B, cfg_4, dev)
    try:
        want_1, want_4 = B.to_numpy(B.trd_match(h1, tracks)), B.to_numpy(B.trd_match(h4, tracks))
        o1, o4, o1b = B.alloc_tracks_out(n), B.alloc_tracks_out(n), B.alloc_tracks_out(n)
        B.trd_match_static(h1, tracks, o1)
        B.trd_match_static(h4, tracks, o4)
        B.trd_match_static(h1, tracks, o1b)
        torch.cuda.synchronize()
        same(B.to_numpy(o1), want_1); same(B.to_numpy(o4), want_4); same(B.to_numpy(o1b), want_1)
    finally:
        B.trd_destroy(h1); B.trd_destroy(h4)


def test_extended_model_through_the_static_entry_point(B):
    """The extended instantiation of the kernel (sin(phi)-dependent resolutions and pad tilt, displaced chambers,
    time-frame association with its interaction ids) behind trd_match_static, twice in a row."""
    import dataclasses
    import torch
    spec = dataclasses.replace(W.CONFIGS["pileup"], res_model=1, chamber_dx_sigma=0.3, n_interactions=5)
    d = W.generate(spec); cfg = W.matcher_config(spec)
    dev = B.to_device(d); n = d["x"].shape[0]
    tracks = dict(part_of(dev, 0, n), interaction=dev["interaction"])
    h = B.trd_create(cfg)
    try:
        B.trd_set_chamber_dx(h, np.ascontiguousarray(d["chamber_dx"], np.float32))
        B.trd_load_tracklets_tf(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"], dev["tl_interaction"],
                                d["n_interactions"])
        want = B.to_numpy(B.trd_match(h, tracks))
        o1, o2 = B.alloc_tracks_out(n), B.alloc_tracks_out(n)
        B.trd_match_static(h, tracks, o1)
        B.trd_match_static(h, tracks, o2)
        torch.cuda.synchronize()
        same(B.to_numpy(o1), want); same(B.to_numpy(o2), want)
        assert int((want["n_matched"] >= 2).sum()) > 0.8 * n
    finally:
        B.trd_destroy(h)


def test_sizes_beyond_the_maximum_are_refused(B):
    import torch
    spec = W.CONFIGS["tiny"]; d = W.generate(spec); cfg = W.matcher_config(spec)
    dev = B.to_device(d)
    h = loaded_handle(B, cfg, dev)
    try:
        n = B.TRD_STATIC_MAX_TRACKS + 1
        big = dict(par=torch.zeros(5, n, device="cuda"), cov=torch.zeros(15, n, device="cuda"),
                   x=torch.full((n,), 247.0, device="cuda"), sector=torch.zeros(n, dtype=torch.int32, device="cuda"))
        out = B.alloc_tracks_out(n)
        out["n_matched"].fill_(-7)
        with pytest.raises(B.TrdError) as err:
            B.trd_match_static(h, big, out)
        assert err.value.code == B.TRD_E_ARG
        assert "TRD_STATIC_MAX_TRACKS" in str(err.value) and str(n) in str(err.value)
        torch.cuda.synchronize()
        assert int((out["n_matched"] != -7).sum().item()) == 0          # refused before anything ran
        B.trd_match_static(h, part_of(dev, 0, 0), B.alloc_tracks_out(0))    # empty batch: accepted, nothing to do
        # and the call still works afterwards
        n0 = d["x"].shape[0]
        got = B.trd_match_static(h, part_of(dev, 0, n0), B.alloc_tracks_out(n0))
        torch.cuda.synchronize()
        same(B.to_numpy(got), B.to_numpy(B.trd_match(h, part_of(dev, 0, n0))))
    finally:
        B.trd_destroy(h)


def test_needs_a_loaded_index(B, base_cfg):
    h = B.trd_create(base_cfg)
    try:
        with pytest.raises(B.TrdError) as err:
            B.trd_match_static(h, dict(x=__import__("torch").zeros(0, device="cuda")), B.alloc_tracks_out(0))
        assert err.value.code == B.TRD_E_STATE
    finally:
        B.trd_destroy(h)
