#!/usr/bin/env python
"""bench.py -- ITS-TPC tracks matched per second through the 6 TRD layers (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload timeframe]

One "step" is one pass of the whole hot path over one synthetic time frame (BASELINE.json configs[4]:
2,000,000 tracks, ~18.8M tracklets, nHyp = 4, 3 sigma road): ONE trd_load_tracklets (key, radix sort,
gather, bin table) + FOUR trd_match calls of 500k tracks.  `value` is timed with inputs resident in HBM;
`e2e` goes through the *_host entry points of the C ABI with pinned host buffers, copies inside the timed
region.  N > 1 (torchrun): every rank runs the whole path on its own time frame, no data-path collective
(weak scaling); barrier + max over ranks.  `--impl reference` times the oracle (oracle/, double precision,
OpenMP over tracks) on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "ITS-TPC tracks matched/sec through 6 TRD layers"
UNIT = "tracks/s"

# Algorithmic flops per unit, counted from the formulas of DESIGN.md "Arithmetic" (= SURVEY.md 8(d).3):
# FMA = 2, add/mul/compare = 1, div/sqrt = 1.  Units per launch come from the oracle's counters.
FLOP = dict(n_prop=180, n_rot=60, n_road=25, n_cand=12, n_upd=110)
# Algorithmic bytes: a track in 88 B (5 + 15 floats, x, sector), out 120 B (6 indices, 5 + 15 floats, x,
# sector, chi2, n_matched), every DISTINCT tracklet found inside some road once at 12 B (y, z, dy/dx).
BYTES_TRACK_IN = 88
BYTES_TRACK_OUT = 120
BYTES_PER_CAND = 12
ORACLE_SAMPLE_TRACKS = 200_000
ORACLE_SAMPLE_TRACKS_1T = 20_000     # the one-thread leg of the oracle (Fig. 5 has both CPU curves)


def fp32_peak_tflops(sm_count: int, sm_mhz: float) -> float:
    """Plain FP32 ALUs: SMs x 128 lanes x 2 flop (FMA) x clock (B200_PROFILING.md: 148 SMs, 1965 MHz)."""
    return sm_count * 128 * 2 * sm_mhz * 1e6 / 1e12


def measured_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, uuid: str, index: int, period: float = 0.01):
        self.period, self.samples, self.mask, self.max_mhz = period, [], 0, None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.dev = pynvml.nvmlDeviceGetHandleByUUID(uuid if uuid.startswith("GPU-") else "GPU-" + uuid)
            except Exception:
                self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.dev, self.nv.NVML_CLOCK_SM)))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev))
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self) -> dict:
        if not self.samples:
            return dict(sm_mhz=None, sm_max_mhz=self.max_mhz, reasons=["unavailable"])
        return dict(sm_mhz=float(np.median(self.samples)), sm_max_mhz=self.max_mhz, n_samples=len(self.samples),
                    reasons=[name for bit, name in self.REASONS.items() if self.mask & bit])


def load_units(spec, n_batches):
    """Oracle operation counters per trd_match launch of the timeframe config (tests/golden/units_timeframe.json,
    written by tests/golden/make_units.py from the oracle alone)."""
    path = os.path.join(ROOT, "tests", "golden", "units_timeframe.json")
    if spec.name != "timeframe" or not os.path.exists(path):
        return None
    with open(path) as f:
        u = json.load(f)
    if u["n_tracks"] != spec.n_tracks or len(u["batches"]) != n_batches:
        return None
    return u["batches"]


def load_bytes_algorithmic(info: dict, n_tl: int) -> float:
    """SURVEY.md 8(d).3, tracklet load + sort + index per tracklet: 16 B in + (8 B + 8 B) per 8-bit pass over the key +
    12 B gather + 16 B out = 44 + 16 x passes (92 B at config 5, whose bin key has 24 bits)."""
    return n_tl * (44.0 + 16.0 * ((info["key_bits"] + 7) // 8))


def load_bytes_model(info: dict, n_tl: int) -> float:
    """What THIS implementation moves with the sort it used: not the roofline's numerator."""
    if info["sort_kind"] == 1:
        # key kernel 16 + 21, partition 21 + 21, placement 21 + 16, order 16 per tracklet; table: cleared, scanned (read,
        # read + write), read by the placement and by order_bins
        return n_tl * 132.0 + 24.0 * info["n_bins"]
    return n_tl * (76.0 + 20.0 * info["n_passes"])


def config_dict(spec, n_tl, world, strong=False):
    n, batch = spec.n_tracks, spec.batch or spec.n_tracks
    nb = (n + batch - 1) // batch
    return dict(workload=spec.name, n_tracks=n, n_tracklets=n_tl, n_hyp=spec.n_hyp, n_sigma_road=spec.n_sigma_road,
                batch=batch, step="1 trd_load_tracklets + %d trd_match" % nb,
                l2="inputs larger than L2 (%.0f MB tracklets + %.0f MB tracks per step)" % (16e-6 * n_tl, 88e-6 * n),
                parallelism=(f"1 time frame, tracks split over {world} ranks, index replicated, no collective" if strong else
                             f"{world} x independent time frames, no collective"))


def oracle_sample(cfg, data, n_sample, n_threads=0):
    """The oracle, as it stands, on the first n_sample tracks against ALL tracklets."""
    from oracle import oracle as O
    r = O.match(cfg, data, lo=0, hi=n_sample, n_threads=n_threads)
    cores = O.max_threads() if n_threads == 0 else n_threads
    return r, cores


def run_reference(args, spec, cfg):
    from paper_2003_03174_b200 import dist as D, workloads as W
    rank, world, _ = D.env_rank()
    if rank != 0:
        return
    data = W.generate(spec)
    n_sample = min(ORACLE_SAMPLE_TRACKS, spec.n_tracks)
    for _ in range(args.warmup):
        oracle_sample(cfg, data, n_sample)
    t0 = time.perf_counter()
    secs = []
    for _ in range(args.steps):
        r, cores = oracle_sample(cfg, data, n_sample)
        secs.append(r["seconds"])
    wall = time.perf_counter() - t0
    # whole-job estimate: one index build + the matching of all tracks at the sample's rate
    idx_s = float(np.mean([s["index"] for s in secs])); match_s = float(np.mean([s["match"] for s in secs]))
    full_s = idx_s + match_s * spec.n_tracks / n_sample
    value = spec.n_tracks / full_s
    sample = (f"{n_sample} of {spec.n_tracks} tracks against all {data['tl_y'].shape[0]} tracklets per step; "
              f"value = n_tracks / (index build {idx_s:.2f} s + match {match_s:.2f} s x {spec.n_tracks / n_sample:.0f})")
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * wall / max(args.steps, 1), higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=config_dict(spec, int(data["tl_y"].shape[0]), max(args.gpus, 1)),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


def run_ours(args, spec, cfg):
    import torch
    from paper_2003_03174_b200 import binding as B, build as Bd, dist as D, workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the TRD matcher has no CPU fallback")
    rank, world, local = D.env_rank()
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    D.init("nccl", device)
    if rank == 0:
        Bd.build()
    D.barrier()
    data = W.generate(spec)                     # every rank: its own (identically generated) time frame
    n, n_tl = spec.n_tracks, int(data["tl_y"].shape[0])
    batch = spec.batch or n
    strong = args.scaling == "strong" and world > 1
    if strong:
        # ONE frame split over the ranks: contiguous track slices, the index built on every rank
        # (replicated: 0.3 GB against 180 GB of HBM), outputs left sharded, still no data-path collective
        s_lo, s_hi = D.track_slice(n, rank, world)
        bounds = [(lo, min(s_hi, lo + batch)) for lo in range(s_lo, s_hi, batch)]
    else:
        bounds = [(lo, min(n, lo + batch)) for lo in range(0, n, batch)]
    dev = B.to_device(data, device)
    tracks = [dict(par=dev["par"][:, lo:hi].contiguous(), cov=dev["cov"][:, lo:hi].contiguous(),
                   x=dev["x"][lo:hi].contiguous(), sector=dev["sector"][lo:hi].contiguous()) for lo, hi in bounds]
    outs = [B.alloc_tracks_out(hi - lo, device) for lo, hi in bounds]
    tl = (dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"])
    n_ia = int(data.get("n_interactions", 0))
    if n_ia > 1:                                 # time-frame association variant (--interactions)
        for t, (lo, hi) in zip(tracks, bounds):
            t["interaction"] = dev["interaction"][lo:hi].contiguous()
    h = B.trd_create(cfg)
    stream = torch.cuda.current_stream()
    if "chamber_dx" in data:
        B.trd_set_chamber_dx(h, data["chamber_dx"], stream=stream)

    def load():
        if n_ia > 1:
            B.trd_load_tracklets_tf(h, *tl, dev["tl_interaction"], n_ia, stream=stream)
        else:
            B.trd_load_tracklets(h, *tl, stream=stream)

    def step(ev=None):
        if ev is not None:
            ev.append(torch.cuda.Event(enable_timing=True)); ev[-1].record(stream)
        load()
        for t, o in zip(tracks, outs):
            if ev is not None:
                ev.append(torch.cuda.Event(enable_timing=True)); ev[-1].record(stream)
            B.trd_match(h, t, o, stream=stream)
        if ev is not None:
            ev.append(torch.cuda.Event(enable_timing=True)); ev[-1].record(stream)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize(); D.barrier()
    launches0 = B.trd_kernel_launches(h)
    events = []
    with ClockSampler(str(getattr(torch.cuda.get_device_properties(local), "uuid", "")), local) as clk:
        t_start = torch.cuda.Event(enable_timing=True); t_end = torch.cuda.Event(enable_timing=True)
        t_start.record(stream)
        for _ in range(args.steps):
            ev = []; step(ev); events.append(ev)
        t_end.record(stream)
        torch.cuda.synchronize()
    D.barrier()
    launches = B.trd_kernel_launches(h) - launches0
    # the dominant kernel alone: the library records CUDA events on the launch stream around every match_kernel launch
    # (a ring of 64 pairs), so the timed region above ran without synchronisation and is read here
    kern_ms = B.trd_match_kernel_ms(h, min(64, args.steps * len(bounds)))
    # TRD-only refit of the matched chains: reported beside the step, not part of it
    r_outs = [B.trd_refit(h, o, stream=stream) for o in outs]
    torch.cuda.synchronize()
    r0 = torch.cuda.Event(enable_timing=True); r1 = torch.cuda.Event(enable_timing=True)
    r0.record(stream)
    for o, ro in zip(outs, r_outs):
        B.trd_refit(h, o, ro, stream=stream)
    r1.record(stream); torch.cuda.synchronize()
    refit_ms = r0.elapsed_time(r1)
    n_refitted = int(sum(int((ro["n_used"] >= 2).sum().item()) for ro in r_outs))
    # the same step captured once in a CUDA graph and replayed (after the warm-up the library allocates nothing): reported
    # beside the headline, which keeps plain stream launches and the library's per-kernel events
    graph_replay = None
    if world == 1:
        try:
            side = torch.cuda.Stream()
            with torch.cuda.stream(side):
                load_on = (lambda s: B.trd_load_tracklets_tf(h, *tl, dev["tl_interaction"], n_ia, stream=s)) if n_ia > 1 else \
                          (lambda s: B.trd_load_tracklets(h, *tl, stream=s))

                def step_on(s):
                    load_on(s)
                    for t, o in zip(tracks, outs):
                        B.trd_match(h, t, o, stream=s)
                step_on(side)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                step_on(side)
            for _ in range(3):
                graph.replay()
            torch.cuda.synchronize()
            g0 = torch.cuda.Event(enable_timing=True); g1 = torch.cuda.Event(enable_timing=True)
            g0.record(stream)
            for _ in range(args.steps):
                graph.replay()
            g1.record(stream); torch.cuda.synchronize()
            g_ms = g0.elapsed_time(g1) / args.steps
            graph_replay = dict(ms_per_step=g_ms, value=n / (g_ms * 1e-3), unit=UNIT, steps=args.steps,
                                note="the step (1 trd_load_tracklets + the trd_match calls) captured once with "
                                     "torch.cuda.graph and replayed; not the headline")
            del graph
        except Exception as exc:                     # noqa: BLE001 -- an extra, never the reason for a failed run
            graph_replay = dict(error=str(exc)[:200])
    total_ms = D.max_over_ranks(t_start.elapsed_time(t_end), device)
    ms_per_step = total_ms / args.steps
    n_job = n if strong else world * n            # tracks the whole job matched per step
    value = n_job / (ms_per_step * 1e-3)
    nb = len(bounds)
    load_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in events]))
    match_ms = np.array([[e[1 + k].elapsed_time(e[2 + k]) for k in range(nb)] for e in events])   # steps x batches
    n_evals = int(sum(int(o["n_evals"].sum().item()) for o in outs))
    n_ge2 = int(sum(int((o["n_matched"] >= 2).sum().item()) for o in outs))
    n_mine = sum(hi - lo for lo, hi in bounds)       # tracks this rank matched per step
    if strong:
        n_evals = int(D.sum_over_ranks(n_evals, device))

    e2e_s, e2e_steps = None, 0
    if n_ia <= 1:
        # ---- end to end through the host entry points (pinned host buffers, copies inside the timed region)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()   # noqa: E731
        h_tl = [pin(data[k]) for k in ("tl_y", "tl_z", "tl_dydx", "tl_chamber")]
        h_tracks = [dict(par=pin(data["par"][:, lo:hi]), cov=pin(data["cov"][:, lo:hi]), x=pin(data["x"][lo:hi]),
                         sector=pin(data["sector"][lo:hi])) for lo, hi in bounds]
        h_outs = [B.alloc_tracks_out_host(hi - lo, pinned=True) for lo, hi in bounds]

        def step_host():
            B.trd_load_tracklets_host(h, *h_tl, stream=stream)
            for t, o in zip(h_tracks, h_outs):
                B.trd_match_host_async(h, t, o, stream=stream)
            B.trd_wait_host(h, stream=stream)            # results of all batches are in host memory here

        for _ in range(2):
            step_host()
        torch.cuda.synchronize(); D.barrier()
        e2e_steps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step_host()                               # waits for this frame's results before the next frame
        torch.cuda.synchronize()
        e2e_sync_s = D.max_over_ranks(time.perf_counter() - t0, device) / e2e_steps
        D.barrier()

        def step_host_streaming():
            # consecutive time frames: the next frame's copy-in may start while this frame is still being matched;
            # every frame's inputs are copied in and every frame's results are copied out inside the timed region
            B.trd_load_tracklets_host(h, *h_tl, stream=stream)
            for t, o in zip(h_tracks, h_outs):
                B.trd_match_host_async(h, t, o, stream=stream)

        step_host_streaming(); B.trd_wait_host(h, stream=stream)
        torch.cuda.synchronize(); D.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step_host_streaming()
        B.trd_wait_host(h, stream=stream)                 # the last frame's results are in host memory here
        torch.cuda.synchronize()
        e2e_s = D.max_over_ranks(time.perf_counter() - t0, device) / e2e_steps
        D.barrier()
        for o, ho in zip(outs, h_outs):               # the two entry points must agree bit for bit
            assert np.array_equal(o["idx"].cpu().numpy(), ho["idx"]) and np.array_equal(o["chi2"].cpu().numpy(), ho["chi2"])
    h2d = 16 * n_tl + BYTES_TRACK_IN * n_mine
    d2h = BYTES_TRACK_OUT * n_mine
    info = B.trd_get_index_info(h)
    B.trd_destroy(h)

    if rank != 0:
        D.shutdown()
        return
    # ---- roofline of the dominant kernel: match_kernel (4 launches per step) vs the load
    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(local)
    clocks = clk.summary()
    units = load_units(spec, nb)
    match_call_ms = float(match_ms.mean())
    match_avg_ms = float(np.mean(kern_ms))
    peak_tf = fp32_peak_tflops(props.multi_processor_count, peaks["sm_max_mhz"])
    if units is not None:
        flops = float(np.mean([sum(FLOP[k] * u[k] for k in FLOP) for u in units]))
        # distinct tracklets found inside some road, counted by the oracle (each read once: SURVEY.md 8(d).3)
        cand = float(np.mean([u.get("n_distinct_cand", min(u["n_cand"], n_tl)) for u in units]))
        units_src = "tests/golden/units_timeframe.json (oracle counters per 500k-track launch; n_distinct_cand for the bytes)"
    else:                                          # other workloads: count what the GPU itself reported
        flops, cand = None, min(n_evals / nb, n_tl)
        units_src = "n_cand from the kernel's own counter (an upper bound of the distinct ones); flops not frozen for this workload"
    bytes_alg = (BYTES_TRACK_IN + BYTES_TRACK_OUT) * (n_mine / nb) + cand * BYTES_PER_CAND
    t_hbm = bytes_alg / (peaks["hbm_gbs"] * 1e9)
    t_alu = (flops / (peak_tf * 1e12)) if flops else 0.0
    if t_alu >= t_hbm:
        ach = flops / (match_avg_ms * 1e-3) / 1e12
        roof = dict(bound="alu", achieved=ach, peak=peak_tf, unit="TFLOP/s", frac=ach / peak_tf, traffic=None)
    else:
        ach = bytes_alg / (match_avg_ms * 1e-3) / 1e9
        roof = dict(bound="hbm", achieved=ach, peak=peaks["hbm_gbs"], unit="GB/s", frac=ach / peaks["hbm_gbs"], traffic=None)
    roof["bounds_ms"] = dict(t_alu=1e3 * t_alu, t_hbm=1e3 * t_hbm, binds="alu" if t_alu >= t_hbm else "hbm",
                             note="roofline time per launch = the slower of algorithmic flops at the FP32 peak and algorithmic "
                                  "bytes at the measured HBM bandwidth (SURVEY.md 8(d).3 constants)")
    roof["alu_view"] = dict(achieved_tflops=(flops / (match_avg_ms * 1e-3) / 1e12) if flops else None, peak_tflops=peak_tf)
    roof.update(kernel="match_kernel<4,BINNED>" if spec.n_hyp in (3, 4) else f"match_kernel (n_hyp={spec.n_hyp})",
                launch_ms=match_avg_ms, trd_match_call_ms=match_call_ms,
                launch_ms_note="match_kernel alone (events recorded by the library on the launch stream); trd_match_call_ms = pack + track sort + match_kernel + unpack", launches_per_step=nb, share_of_step=nb * match_avg_ms / ms_per_step, call_share_of_step=nb * match_call_ms / ms_per_step,
                algorithmic_flops_per_launch=flops, algorithmic_bytes_per_launch=bytes_alg,
                roofline_ms_per_launch=1e3 * max(t_alu, t_hbm), hbm_view_gbs=bytes_alg / (match_avg_ms * 1e-3) / 1e9,
                peak_source=f"HBM {peaks['source']} (MEASURED_PEAKS.json); FP32 = {props.multi_processor_count} SMs x 128 x 2 x "
                            f"{peaks['sm_max_mhz']:.0f} MHz", units=units_src,
                load_tracklets_ms=load_ms,
                load_algorithmic_gbs=load_bytes_algorithmic(info, n_tl) / (load_ms * 1e-3) / 1e9,
                load_frac_of_hbm=load_bytes_algorithmic(info, n_tl) / (load_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                load_model_gbs=load_bytes_model(info, n_tl) / (load_ms * 1e-3) / 1e9,
                load_io_gbs=n_tl * 32 / (load_ms * 1e-3) / 1e9,
                load_note="load_algorithmic_gbs: SURVEY.md 8(d).3 bytes (44 + 16 x passes per tracklet); load_model_gbs: the bytes "
                          "this implementation's passes move (DESIGN.md 6.1); load_io_gbs: 16 B in + 16 B out per tracklet")
    prof = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(prof) and spec.name == "timeframe":
        with open(prof) as f:
            tj = json.load(f)
        roof["traffic"] = tj.get("match_kernel_dram_bytes_per_launch")
        roof["traffic_source"] = "profiles/traffic.json (one ncu --set full capture of this kernel, NOT measured in this run): " + tj.get("source", "")
        wi = tj.get("match_kernel_warp_instructions_per_launch")
        if wi:
            issue_ms = 1e3 * wi / (props.multi_processor_count * 4 * peaks["sm_max_mhz"] * 1e6)
            roof["issue_view"] = dict(warp_instructions_per_launch=wi, issue_only_ms=issue_ms, frac_of_launch=issue_ms / match_avg_ms,
                                      note="executed warp instructions (same ncu capture) / (SMs x 4 schedulers x max clock): the time "
                                           "the kernel would take if it issued one instruction per scheduler and cycle")

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_per_step, higher_is_better=True, scaling="strong" if strong else "weak", vs_baseline=None,
                dtype="f32 (y, sin(phi) accumulated in f64)",
                data="synthetic",
                config=config_dict(spec, n_tl, world, strong),
                cand_evals_per_s=(1 if strong else world) * n_evals / (ms_per_step * 1e-3), n_cand_evals=n_evals,
                frac_tracks_ge2_tracklets=n_ge2 / max(n_mine, 1), index=dict(n_ybins=info["n_ybins"], n_zrows=info["n_zrows"],
                                                                ybin_width_cm=info["ybin_width"],
                                                                sort="counting" if info["sort_kind"] == 1 else "radix",
                                                                radix_passes=0 if info["sort_kind"] == 1 else info["n_passes"]),
                refit=dict(ms_per_time_frame=refit_ms, tracks_per_s=n_mine / (refit_ms * 1e-3), frac_refitted=n_refitted / max(n_mine, 1),
                           note="trd_refit over the matched chains of the step, device-resident, timed separately"),
                graph_replay=graph_replay, clocks=clocks, gpu_launches=int(launches),
                e2e=(dict(value=n_job / e2e_s, unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                          ms_per_step=1e3 * e2e_s, steps=e2e_steps, ms_per_step_frame_by_frame=1e3 * e2e_sync_s,
                          note="consecutive frames streamed through the host entry points (copies of frame k+1 overlap the "
                               "kernels of frame k); frame_by_frame waits for each frame's results before the next") if e2e_s else
                     dict(value=None, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0,
                          note="the host entry points do not carry interaction ids; device-resident numbers only")),
                roofline=roof)
    if world == 1 and not args.no_cpu_baseline:
        n_sample = min(ORACLE_SAMPLE_TRACKS, n)
        r, cores = oracle_sample(cfg, data, n_sample)
        full_s = r["seconds"]["index"] + r["seconds"]["match"] * n / n_sample
        n_1t = min(ORACLE_SAMPLE_TRACKS_1T, n)
        r1, _ = oracle_sample(cfg, data, n_1t, n_threads=1)
        full_1t = r1["seconds"]["index"] + r1["seconds"]["match"] * n / n_1t
        line["cpu_baseline"] = dict(
            value=n / full_s, unit=UNIT, cores=cores, kind="oracle (unoptimised: plain double-precision checker, its index is one "
                                                            "y-sorted list per (sector, layer) without z binning)",
            value_1t=n / full_1t,
            scanned_per_in_road_candidate=r["counters"]["n_scanned"] / max(r["counters"]["n_cand"], 1),
            sample=(f"first {n_sample} of {n} tracks against all {n_tl} tracklets: index build {r['seconds']['index']:.2f} s + "
                    f"match {r['seconds']['match']:.2f} s; value = n_tracks / (index + match x {n / n_sample:.0f}); value_1t: the same "
                    f"with one thread on the first {n_1t} tracks (index {r1['seconds']['index']:.2f} s + match {r1['seconds']['match']:.2f} s)"))
    print(json.dumps(line), flush=True)
    D.shutdown()


def run_sweep(args):
    """`--sweep`: the three curves of the paper's benchmark (Fig. 5: time per event against
    the number of tracks for the CPU with one thread, the CPU with all cores and the GPU) on the five configs of
    BASELINE.json.  GPU: one step = trd_load_tracklets + trd_match over all batches, device-resident, CUDA events.
    CPU: the oracle as it stands (index build + matching), on a bounded sample for config 5.  One JSON line per config
    and a markdown table at the end."""
    import torch
    from paper_2003_03174_b200 import binding as B, build as Bd, workloads as W
    from oracle import oracle as O
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the TRD matcher has no CPU fallback")
    Bd.build()
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    cores = O.max_threads()                     # before any one-thread call (the OpenMP setting sticks)
    rows = []
    for name in ("tiny", "central", "central8", "pileup", "timeframe"):
        spec = W.CONFIGS[name]; data = W.generate(spec); cfg = W.matcher_config(spec)
        n, n_tl = spec.n_tracks, int(data["tl_y"].shape[0])
        batch = spec.batch or n
        bounds = [(lo, min(n, lo + batch)) for lo in range(0, n, batch)]
        dev = B.to_device(data, torch.device("cuda", 0))
        tracks = [dict(par=dev["par"][:, lo:hi].contiguous(), cov=dev["cov"][:, lo:hi].contiguous(),
                       x=dev["x"][lo:hi].contiguous(), sector=dev["sector"][lo:hi].contiguous()) for lo, hi in bounds]
        outs = [B.alloc_tracks_out(hi - lo, torch.device("cuda", 0)) for lo, hi in bounds]
        h = B.trd_create(cfg)

        def step(s=stream):
            B.trd_load_tracklets(h, dev["tl_y"], dev["tl_z"], dev["tl_dydx"], dev["tl_chamber"], stream=s)
            for t, o in zip(tracks, outs):
                B.trd_match(h, t, o, stream=s)

        steps = args.steps if name == "timeframe" else max(args.steps, 50)
        for _ in range(5):
            step()
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            step()
        e1.record(stream); torch.cuda.synchronize()
        gpu_ms = e0.elapsed_time(e1) / steps
        # the same step captured once in a CUDA graph and replayed (after the warm-up the library allocates nothing, so its
        # calls can be captured): what a caller who processes event after event with fixed buffers would do
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            step(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            step(side)
        graph.replay(); torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(steps):
            graph.replay()
        e1.record(stream); torch.cuda.synchronize()
        graph_ms = e0.elapsed_time(e1) / steps
        del graph
        B.trd_destroy(h)
        n_all = min(ORACLE_SAMPLE_TRACKS, n); n_1t = min(ORACLE_SAMPLE_TRACKS_1T, n)
        ra = O.match(cfg, data, lo=0, hi=n_all, n_threads=cores)
        r1 = O.match(cfg, data, lo=0, hi=n_1t, n_threads=1)
        cpu_all_ms = 1e3 * (ra["seconds"]["index"] + ra["seconds"]["match"] * n / n_all)
        cpu_1t_ms = 1e3 * (r1["seconds"]["index"] + r1["seconds"]["match"] * n / n_1t)
        row = dict(sweep=name, n_tracks=n, n_tracklets=n_tl, n_hyp=spec.n_hyp, n_sigma_road=spec.n_sigma_road,
                   gpu_ms_per_step=gpu_ms, gpu_tracks_per_s=n / (gpu_ms * 1e-3), gpu_steps=steps,
                   gpu_graph_replay_ms_per_step=graph_ms,
                   oracle_cores=cores, oracle_all_cores_ms=cpu_all_ms, oracle_1_thread_ms=cpu_1t_ms,
                   oracle_sample_tracks=[n_all, n_1t], unit="ms per step (load + match of the whole config)")
        rows.append(row)
        print(json.dumps(row), flush=True)
        del dev, tracks, outs
        torch.cuda.empty_cache()
    print("\n| config | tracks | tracklets | nHyp | oracle, 1 thread | oracle, %d threads | GPU (B200) | GPU, step replayed as a CUDA graph | GPU tracks/s |" % rows[0]["oracle_cores"])
    print("|---|---|---|---|---|---|---|---|---|")
    for r in rows:
        print("| %s | %d | %d | %d | %.1f ms | %.1f ms | %.3f ms | %.3f ms | %.3g |" % (
            r["sweep"], r["n_tracks"], r["n_tracklets"], r["n_hyp"], r["oracle_1_thread_ms"], r["oracle_all_cores_ms"],
            r["gpu_ms_per_step"], r["gpu_graph_replay_ms_per_step"], r["gpu_tracks_per_s"]))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="timeframe")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one time frame per rank (default); strong = one frame, its tracks split over the ranks")
    ap.add_argument("--tracks", type=int, default=0, help="scale the workload to this many tracks (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs 1-5: oracle with one thread, oracle with all cores, GPU (PAPER.md Fig. 5)")
    ap.add_argument("--interactions", type=int, default=0,
                    help="> 1: time-frame association with this many interactions (SURVEY.md 8(f) NEXT#2)")
    ap.add_argument("--ybin-width", type=float, default=0.0, help="local-y bin width of the index in cm (0 = chosen by the library)")
    ap.add_argument("--chamber-dx", type=float, default=0.0,
                    help="> 0: chambers displaced radially by N(0, this) cm, two-stage propagation (SURVEY.md 8(f) NEXT#3)")
    ap.add_argument("--material", action="store_true",
                    help="a slab of material in front of every layer: multiple scattering and energy loss (SURVEY.md 8(f) NEXT#3)")
    ap.add_argument("--field", action="store_true",
                    help="inhomogeneous field Bz (1 + bz_r2 r^2 + bz_z2 z^2), true particles integrated numerically (SURVEY.md 8(f) NEXT#3)")
    ap.add_argument("--res-model", type=int, default=0, choices=[0, 1],
                    help="1: inputs and matcher with the sin(phi)-dependent resolutions and pad tilt (SURVEY.md 8(f) NEXT#1)")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
        return
    from paper_2003_03174_b200 import workloads as W
    spec = W.CONFIGS[args.workload]
    if args.tracks:
        spec = W.scaled(spec, args.tracks)
    import dataclasses
    if args.res_model:
        spec = dataclasses.replace(spec, res_model=1, name=spec.name + "_res1")
    if args.interactions > 1:
        spec = dataclasses.replace(spec, n_interactions=args.interactions, name=spec.name + f"_tf{args.interactions}")
    if args.chamber_dx > 0.0:
        spec = dataclasses.replace(spec, chamber_dx_sigma=args.chamber_dx, name=spec.name + "_dx")
    if args.material:
        spec = dataclasses.replace(spec, x_over_x0=W.X_OVER_X0, eloss=W.ELOSS, eloss_fluct=W.ELOSS_FLUCT, name=spec.name + "_mat")
    if args.field:
        spec = dataclasses.replace(spec, bz_r2=W.BZ_R2, bz_z2=W.BZ_Z2, name=spec.name + "_field")
    cfg = W.matcher_config(spec)
    if args.ybin_width > 0.0:
        cfg["ybin_width"] = args.ybin_width
    if args.impl == "reference":
        run_reference(args, spec, cfg)
    else:
        run_ours(args, spec, cfg)


if __name__ == "__main__":
    main()
