#!/usr/bin/env python
"""bench.py -- photons propagated / s on the DARWIN-scale TPC (BASELINE.json configs[2]) on N B200s.

A "step" is one pass of the whole hot path (photon claim -> Philox -> BVH first hit -> bulk / surface physics ->
fates and per-PMT / arrival-time reductions) over one batch of 1e7 synthetic photons resident in HBM.
    python bench.py --gpus N --steps K --warmup W            # this library (one rank per GPU under torchrun)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on a bounded sample (rank 0 only)
Prints ONE JSON line (see DESIGN.md "Measurement" for every field).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "photons propagated/sec on 1 B200 (DARWIN-scale TPC); % of propagation roofline"
UNIT = "photons/s"
# Algorithmic work per photon-step at C2: the ideal path of an 8-wide BVH
# over T = 113 280 triangles with 4-triangle leaves = ceil(log8(T/4)) = 5 nodes x 125 lane-instructions
# + 4 triangles x 45 + 250 for the physics of the step = 1055 lane-instructions; 5 x 80 B + 4 x 48 B = 592 B.
def algorithmic_work(n_tri):
    """(lane-instructions, bytes) per photon-step of the ideal 8-wide path over n_tri triangles with 4-triangle leaves."""
    import math
    levels = max(1, math.ceil(math.log(max(n_tri, 8) / 4.0) / math.log(8.0)))
    return levels * 125 + 4 * 45 + 250, levels * 80 + 4 * 48


ALG_LANE_INSTR_PER_STEP, ALG_BYTES_PER_STEP = algorithmic_work(113_280)     # C2: 5 levels -> 1055 lane-instr, 592 B
ALG_STATE_BYTES_PER_PHOTON = 44 + 32          # eleven fp32 words in, eight 4-byte result words out (what dw_propagate is handed)
SM_COUNT, LANES_PER_SM = 148, 128


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=float(d.get("hbm_gbs", 6650.0)), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (pynvml; nvidia-smi as a fallback)."""

    def __init__(self, index: int, period_s: float = 0.02):
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self._proc = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                     0x80: "hw_power_brake_slowdown"}

            def loop():
                while not self._stop.is_set():
                    try:
                        self.samples.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                        r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                        for bit, nm in names.items():
                            if r & bit:
                                self.reasons.add(nm)
                    except Exception:
                        pass
                    time.sleep(self.period)
            self._thr = threading.Thread(target=loop, daemon=True)
            self._thr.start()
        except Exception:
            q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                 "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
            try:
                self._proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "100",
                                               "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            except Exception:
                self._proc = None
        return self

    def stop(self) -> dict:
        self._stop.set()
        if self._thr:
            self._thr.join(timeout=1.0)
        if self._proc:
            self._proc.terminate()
            try:
                out, _ = self._proc.communicate(timeout=2.0)
            except Exception:
                out = ""
            for line in out.splitlines():
                f = [x.strip() for x in line.split(",")]
                if len(f) >= 6:
                    try:
                        self.samples.append(float(f[0]))
                        self.max_mhz = float(f[1])
                    except ValueError:
                        continue
                    for nm, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                        if v.lower().startswith("active"):
                            self.reasons.add(nm)
        med = float(np.median(self.samples)) if self.samples else None
        return dict(sm_mhz=med, sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons), samples=len(self.samples))


def workload(args):
    from paper_2203_14354_b200 import synth
    c = synth.config_design(args.design, 2) if getattr(args, "design", "") else synth.config(args.config)
    n = args.photons or c.n_photons
    return c, n


def synth_source(cfg):
    from paper_2203_14354_b200 import synth
    return synth.source_for(cfg)


def emit_args(dw, source):
    import ctypes
    src = dw.Source(shape=int(source["shape"]), centre=(ctypes.c_float * 3)(*source["centre"]), radius=source["radius"], z0=source["z0"],
                    z1=source["z1"], lambda_mean=source["lambda_mean"], lambda_sigma=source["lambda_sigma"], t_start=source["t_start"],
                    tau1=source["tau1"], tau3=source["tau3"], f_singlet=source["f_singlet"])
    return (ctypes.byref(src),)


def cpu_baseline(c, n_sample, id_base=0, threads=None):
    """The oracle, as it stands, on the first n_sample photons of the workload's batch."""
    from oracle import oracle as orc
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    cores = threads or orc.hardware_threads()
    ph = c.make_photons(n_sample, id_base)
    t0 = time.perf_counter()
    out = o.propagate(ph, c.seed, c.max_steps, n_bins=2000, dt=1.0, full=False, nthreads=cores)
    dt = time.perf_counter() - t0
    return dict(value=n_sample / dt, unit=UNIT, cores=cores, kind="oracle",
                sample=f"first {n_sample} photons of the {c.name} batch, all {cores} host threads, {dt:.2f} s",
                photon_steps_per_s=float(out["total_steps"][0]) / dt, seconds=dt,
                detected_fraction=float(out["fate_count"][0]) / n_sample), o


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c, n_full = workload(args)
    n_sample = args.ref_sample
    from oracle import oracle as orc
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    cores = orc.hardware_threads()
    times, steps_total = [], 0
    for it in range(args.warmup + args.steps):
        ph = c.make_photons(n_sample, it * n_sample)
        t0 = time.perf_counter()
        out = o.propagate(ph, c.seed, c.max_steps, n_bins=2000, dt=1.0, full=False, nthreads=cores)
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt)
            steps_total += int(out["total_steps"][0])
    total = sum(times)
    value = n_sample * args.steps / total
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * total / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=dict(workload=c.name, photons_per_step=n_sample, full_batch=n_full, max_steps=c.max_steps,
                                              triangles=c.geometry.n_tri),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle",
                                  sample=f"{n_sample} photons of the {c.name} batch per step, {cores} host threads"),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                photon_steps_per_s=steps_total / total, gpu_launches=0)
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2: DARWIN-scale TPC)")
    ap.add_argument("--photons", type=int, default=0, help="photons per step per GPU (default: the config's batch)")
    ap.add_argument("--ref-sample", type=int, default=2_000_000, help="photons per step of the oracle (--impl reference / cpu_baseline): "
                    "about 10 s of work on 16 host threads at C2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--literal", action="store_true", help="DW_PROP_UNBOUNDED_QUERY (the oracle's literal loop)")
    ap.add_argument("--max-leaf", type=int, default=0, help="triangles per BVH leaf (0 = library default)")
    ap.add_argument("--ploc-radius", type=int, default=0, help="search radius of the BVH clustering rounds (0 = library default)")
    ap.add_argument("--split-div", type=int, default=0, help="split triangles longer than scene extent / this (0 = default, -1 = never)")
    ap.add_argument("--grid-res", type=int, default=0, help="cells per axis of the empty-space grid (0 = default, -1 = none)")
    ap.add_argument("--design", default="", choices=["", "baseline", "detailed_pmt", "side_sensors", "both"],
                    help="run on synth.config_design(VARIANT) at C2 size instead of a BASELINE.json config (SURVEY 8(f) f4, diagnostic)")
    ap.add_argument("--move", default="", choices=["", "affine", "component", "jitter"], help="run on synth.moved(geometry, KIND) (diagnostic)")
    ap.add_argument("--refit", action="store_true", help="with --move: build the tree on the original geometry and move it with dw_refit_bvh "
                    "instead of building on the moved one (diagnostic: cost and quality of a refit)")
    ap.add_argument("--render", type=int, default=0, help="also time dw_render on an N x N image of the detector seen from outside and from "
                    "inside (diagnostic: the first-hit query on coherent rays; reported in config.render)")
    ap.add_argument("--pipeline", action="store_true", help="also time the same K steps issued alternately on two streams, so that the drain "
                    "of one batch (its longest-lived photons) overlaps the start of the next (diagnostic, reported in config.pipelined; "
                    "the headline value stays the serial one)")
    ap.add_argument("--no-skip", action="store_true", help="DW_PROP_NO_EMPTY_SKIP (traverse every query, diagnostic)")
    ap.add_argument("--emit", action="store_true", help="generate each step's photons on the device with dw_emit inside the timed step "
                    "(SURVEY 8(f) f1; C1-C4 only) instead of propagating a resident batch")
    ap.add_argument("--legacy", action="store_true", help="DW_PROP_LEGACY_SCHEDULER (first-generation kernel, diagnostic)")
    ap.add_argument("--th-phys", type=int, default=0, help="phase-scheduling threshold (0 = library default)")
    ap.add_argument("--th-leaf", type=int, default=0, help="phase-scheduling threshold (0 = library default)")
    ap.add_argument("--sweep", action="store_true", help="with --config 4: also run BASELINE.json configs[4] as written (PTFE reflectivity 0.90 / 0.95 / "
                    "0.99, 10 batches of 1e7 photons each with photon_id_base = b * 1e7, only dw_set_surfaces between them) and report the wall "
                    "time of the sweep, the hit map totals and the arrival-time histogram per reflectivity in config.sweep")
    ap.add_argument("--design-study", type=int, default=0, help="also time dw_design_study (ONE library call: emit, propagate, tally, LCE and "
                    "t90) for this many point sources on a Z x R^2 grid of the config's liquid volume (the paper's LCE map has ~2500), "
                    "--study-photons each; reported in config.design_study (SURVEY 8(f) f3, diagnostic)")
    ap.add_argument("--study-photons", type=int, default=1_000_000, help="photons per source of --design-study (the paper: 1e6)")
    ap.add_argument("--no-counters", action="store_true", help="skip the run of the counting instantiation (roofline.implementation_counters)")
    ap.add_argument("--counter-sample", type=int, default=0,
                    help="photons of the batch that the counting instantiation runs over (0 = the whole batch: a short sample is mostly the "
                         "tail of its warps and under-reports the lanes per iteration)")
    ap.add_argument("--block", type=int, default=0, help="threads per block (0 = library default)")
    ap.add_argument("--blocks-per-sm", type=int, default=0, help="cap on resident blocks per SM (0 = occupancy limit)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2203_14354_b200 import binding as dw
    from paper_2203_14354_b200 import dist as dwdist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU path")
    rank, world, local = dwdist.init_from_env()
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    c, n = workload(args)
    ctx = dw.Context(local)
    ctx.set_optics(c.optics)
    from paper_2203_14354_b200 import synth as _synth
    geom = c.geometry if (not args.move or args.refit) else _synth.moved(c.geometry, args.move)
    ctx.set_geometry(geom)
    stats = ctx.build_bvh(args.max_leaf, ploc_radius=args.ploc_radius, grid_res=args.grid_res, split_div=args.split_div)
    # the first build of a context also grows its memory pool (one-off); a rebuild of the same geometry is what a sweep of variants pays
    rebuild_ms = ctx.build_bvh(args.max_leaf, ploc_radius=args.ploc_radius, grid_res=args.grid_res, split_div=args.split_div)["build_ms"]
    refit_info = None
    if args.move and args.refit:
        rs = ctx.refit(_synth.moved(c.geometry, args.move).xyz)
        refit_info = dict(refit_ms=rs["refit_ms"], loose_tris=rs["n_loose_tris"], levels=rs["n_levels"], area_ratio=rs["area_ratio"])
    render_info = None
    if args.render > 0:
        import numpy as _np
        lo, hi = geom.xyz.min(0).astype(float), geom.xyz.max(0).astype(float)
        mid, size = (lo + hi) / 2, float((hi - lo).max())
        render_info = {}
        for name, v in (("outside", dict(eye=mid + _np.array([1.3, 0.8, 0.9]) * size, forward=[-1.3, -0.8, -0.9], up=[0, 0, 1], fov_y_deg=40.0)),
                        ("inside", dict(eye=mid + _np.array([0.1, -0.05, -0.25]) * size, forward=[0.4, 0.3, 0.85], up=[0, 0, 1], fov_y_deg=80.0))):
            best = float("inf")
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                tri_img, _, _ = ctx.render(width=args.render, height=args.render, device=dev, **v)
                e1.record()
                torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1))
            render_info[name] = dict(ms=best, mrays_per_s=args.render ** 2 / best / 1e3, hit_fraction=float((tri_img >= 0).float().mean()))
    id_base, _ = dwdist.shard_ids(n, rank, world, weak=True)
    ph = c.make_photons(n, id_base)
    d_ph = dw.DevicePhotons(ph, dev)
    out = dw.DeviceResults(n, ("flags", "channel", "t", "steps", "last_tri", "x", "y", "z"), dev)   # 32 B / photon
    hist = dw.DeviceHists(ctx.n_chan, 2000, 0.0, 1.0, dev)
    stream = torch.cuda.current_stream()
    flags = (dw.PROP_UNBOUNDED_QUERY if args.literal else 0) | (dw.PROP_LEGACY_SCHEDULER if args.legacy else 0) | (dw.PROP_NO_EMPTY_SKIP if args.no_skip else 0)

    source = synth_source(args.config) if args.emit else None
    state = dict(d_ph=d_ph, k=0)

    def step():
        if source is not None:                  # a new batch of ids every step, written by dw_emit on the same stream
            state["d_ph"] = ctx.emit(source, c.seed, n, id_base=id_base + state["k"] * n * world, device=dev, stream=stream)
            state["k"] += 1
        ctx.propagate(state["d_ph"], c.seed, c.max_steps, out, hist, flags=flags, stream=stream, th_phys=args.th_phys,
                      th_leaf=args.th_leaf, block_threads=args.block, blocks_per_sm=args.blocks_per_sm)
        if world > 1:
            dwdist.merge_hists(hist)        # the only exchange: tens of kB of integer histograms

    sampler = ClockSampler(local).start()            # NVML is initialised here, before the warm-up: its first calls take driver locks
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    hist.zero_()
    dwdist.barrier()
    torch.cuda.synchronize()
    launches0 = ctx.last_launch()["n_launches"]
    sampler.samples.clear()                          # only the samples of the timed region count
    sampler.reasons.clear()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for i in range(args.steps):
        step()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    dwdist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    per_step_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[-1])
    total_ms = dwdist.max_over_ranks(total_ms)
    launches = ctx.last_launch()["n_launches"] - launches0
    h = hist.numpy()                                # this rank's reductions over the K timed steps
    local_steps = int(h["total_steps"][0])
    total_steps = dwdist.sum_over_ranks(local_steps)
    fate = h["fate_count"].astype(np.int64)
    n_all = n * world
    value = n_all * args.steps / (total_ms * 1e-3)

    pipelined = None
    if args.pipeline and not args.emit and world == 1:
        out2 = dw.DeviceResults(n, ("flags", "channel", "t", "steps", "last_tri", "x", "y", "z"), dev)
        lanes = [(torch.cuda.Stream(device=dev), out), (torch.cuda.Stream(device=dev), out2)]
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for rep in range(2):                                   # first pass warms the second stream up
            e0.record(lanes[0][0])
            lanes[1][0].wait_event(e0)
            for i in range(args.steps):
                st_i, out_i = lanes[i % 2]
                ctx.propagate(d_ph, c.seed, c.max_steps, out_i, hist, flags=flags, stream=st_i, th_phys=args.th_phys, th_leaf=args.th_leaf,
                              block_threads=args.block, blocks_per_sm=args.blocks_per_sm)
            done = torch.cuda.Event()
            done.record(lanes[1][0])
            lanes[0][0].wait_event(done)
            e1.record(lanes[0][0])
            torch.cuda.synchronize()
        pms = e0.elapsed_time(e1)
        pipelined = dict(value=n * args.steps / (pms * 1e-3), ms_per_step=pms / args.steps, streams=2,
                         note="same K steps, alternating streams; results of the two lanes go to separate buffers")

    emit_info = None
    if args.emit:
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        keep = ctx.emit(source, c.seed, n, device=dev, stream=stream)          # warm-up and allocation
        reps = 20
        evs[0].record(stream)
        for r in range(reps):
            ctx.L.dw_emit(ctx.h, *emit_args(dw, source), int(c.seed), __import__("ctypes").byref(keep.c), dw._stream_ptr(stream))
        evs[1].record(stream)
        torch.cuda.synchronize()
        ems = evs[0].elapsed_time(evs[1]) / reps
        peaks0 = measured_peaks()
        emit_info = dict(kernel="emit_kernel", ms=ems, photons_per_s=n / (ems * 1e-3), bytes_per_photon=44,
                         achieved_gbs=44.0 * n / (ems * 1e-3) / 1e9, hbm_peak_gbs=peaks0["hbm_gbs"],
                         frac_of_hbm=44.0 * n / (ems * 1e-3) / 1e9 / peaks0["hbm_gbs"])

    study_info = None
    if args.design_study > 0 and world == 1 and args.config in (1, 2, 3):
        g = geom
        R, zl = (250.0, 495.0) if args.config == 1 else (1300.0, 2600.0)
        nz = max(1, int(round(np.sqrt(args.design_study * 2))))         # twice as many heights as radii, as in the paper's maps
        nr = max(1, -(-args.design_study // nz))
        srcs = [_synth.source(_synth.SHAPE_POINT, (float(np.sqrt((j + 0.5) / nr) * (R - 20.0)), 0.0, float(10.0 + (i + 0.5) / nz * (zl - 20.0))))
                for i in range(nz) for j in range(nr)][: args.design_study]
        group = np.where(np.arange(g.n_channels) < g.n_channels // 2, 0, 1).astype(np.int32)
        comp = (np.asarray(g.surface) + 1).astype(np.int32)
        spb = max(1, (1 << 25) // args.study_photons)
        torch.cuda.synchronize()
        t0 = time.perf_counter()                                        # one batch first: the context's pool grows to the batch buffers (one-off)
        ctx.design_study(srcs[:spb], args.study_photons, c.seed, c.max_steps, group, 2, comp, int(comp.max()) + 1, n_bins=1000, dt=1.0,
                         sources_per_batch=spb, device=dev)
        dt_first = time.perf_counter() - t0
        t0 = time.perf_counter()
        res = ctx.design_study(srcs, args.study_photons, c.seed, c.max_steps, group, 2, comp, int(comp.max()) + 1, n_bins=1000, dt=1.0,
                               sources_per_batch=spb, device=dev)
        dt = time.perf_counter() - t0
        lce = res["lce"].sum(1)
        study_info = dict(sources=len(srcs), photons_per_source=args.study_photons, seconds=dt, photons_per_s=len(srcs) * args.study_photons / dt,
                          first_batch_call_seconds=dt_first, api="dw_design_study (one call, after one call over the first batch of sources)", lce_min=float(lce.min()), lce_max=float(lce.max()),
                          t90_min_ns=float(np.nanmin(res["t90"])), t90_max_ns=float(np.nanmax(res["t90"])),
                          absorbed_by_component=[int(v) for v in res["absorbed_by_component"]])

    sweep_info = None
    if args.sweep and args.config == 4 and world == 1 and not args.emit:
        nb, nbp = 10, 10_000_000                                                             # BASELINE.json: 1e8 photons in batches of 1e7
        batches = [dw.DevicePhotons(c.make_photons(nbp, b * nbp), dev) for b in range(nb)]   # 10 x 440 MB resident; generation is not timed
        out_b = dw.DeviceResults(nbp, ("flags", "channel", "t", "steps", "last_tri", "x", "y", "z"), dev)
        sweep_info, t_all = {}, 0.0
        for rho in (0.90, 0.95, 0.99):
            o4 = _synth.config(4, ptfe_reflectivity=rho).optics
            hs = dw.DeviceHists(ctx.n_chan, 2000, 0.0, 1.0, dev)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ctx.set_surfaces(o4.detect, o4.reflect_diffuse, o4.reflect_specular, o4.transmit)    # the only thing that changes: no BVH rebuild
            for b in range(nb):
                ctx.propagate(batches[b], c.seed, c.max_steps, out_b, hs, flags=flags, stream=stream)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            t_all += dt
            hh = hs.numpy()
            det = int(hh["fate_count"][0])
            th = hh["time_hist"].astype(np.int64)
            cum = np.cumsum(th)
            nch = ctx.n_chan // 2
            sweep_info[f"rho_{rho:.2f}"] = dict(seconds=dt, photons=nbp * nb, photons_per_s=nbp * nb / dt, detected=det, lce=det / (nbp * nb),
                                                hits_bottom_array=int(hh["chan_count"][:nch].sum()), hits_top_array=int(hh["chan_count"][nch:].sum()),
                                                max_hits_one_pmt=int(hh["chan_count"].max()), escaped=int(hh["fate_count"][3]),
                                                arrival_hist_peak_bin_ns=int(th.argmax()), arrival_hist_overflow=int(th[-1]),
                                                bin_holding_90_percent_ns=int(np.searchsorted(cum, 0.9 * cum[-1])),
                                                steps_per_photon=int(hh["total_steps"][0]) / (nbp * nb))
        sweep_info["wall_seconds_3_reflectivities"] = t_all
        o4 = c.optics
        ctx.set_surfaces(o4.detect, o4.reflect_diffuse, o4.reflect_specular, o4.transmit)
        del batches

    # ---- end to end through the host-buffer entry (pinned host memory, H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e and not args.emit:
        hp = dw.HostPhotons(ph)
        hout = dw.HostResults(n, ("flags", "channel", "t"))
        hh = dw.HostHists(ctx.n_chan, 2000, 0.0, 1.0)
        ctx.propagate_host(hp, c.seed, c.max_steps, hout, hh, flags=flags)      # warm-up (allocates staging)
        dwdist.barrier()
        t0 = time.perf_counter()
        reps = max(1, min(args.steps, 3))
        each = []
        for _ in range(reps):
            t1 = time.perf_counter()
            ctx.propagate_host(hp, c.seed, c.max_steps, hout, hh, flags=flags)      # synchronous: returns when the host buffers are complete
            each.append(1e3 * (time.perf_counter() - t1))
        torch.cuda.synchronize()
        dt = dwdist.max_over_ranks(time.perf_counter() - t0)
        e2e = dict(value=n_all * reps / dt, unit=UNIT, h2d_bytes_per_step=int(hp.nbytes), d2h_bytes_per_step=int(hout.nbytes + hh.nbytes),
                   ms_per_step=1e3 * dt / reps, ms_each=each, api="dw_propagate_host (pinned host buffers, chunked copies overlapped with propagation)",
                   h2d="11 fp32 arrays (44 B / photon)", d2h="flags, channel, t (12 B / photon) + the four reductions")

    if rank != 0:
        dwdist.finalize()
        return 0

    peaks = measured_peaks()
    alg_instr, alg_step_bytes = algorithmic_work(c.geometry.n_tri)
    kernel_ms = float(np.mean(per_step_ms))
    kernel_s = kernel_ms * 1e-3
    steps_per_launch = local_steps / args.steps
    peak_lane = SM_COUNT * LANES_PER_SM * peaks["sm_max_mhz"] * 1e6          # lane-instructions / s
    achieved_lane = steps_per_launch * alg_instr / kernel_s
    tree_bytes = steps_per_launch * alg_step_bytes                              # BVH bytes of the ideal path: L2-resident tree (C0-C2) or L2 + HBM
    state_bytes = n * ALG_STATE_BYTES_PER_PHOTON                                # photon state in and results out: HBM
    # the derived ALU peak against what this device issues in register-only streams, and the L2 read bandwidth (dw_probe_peaks:
    # ~0.1 s, outside the timed region)
    probe = None
    try:
        pk = ctx.probe_peaks()
        probe = dict(fma_tlane_instr_s=pk["fma_lane_instr_per_s"] / 1e12, alu_tlane_instr_s=pk["alu_lane_instr_per_s"] / 1e12,
                     mix_tlane_instr_s=pk["mix_lane_instr_per_s"] / 1e12, l2_read_gbs=pk["l2_read_bytes_per_s"] / 1e9,
                     note="dw_probe_peaks in this run: pure FP32 FMA / pure integer ALU / even mix in lane-instructions per second, and the read "
                          "bandwidth of a 32 MiB buffer resident in L2 (the denominator of frac_l2)")
    except Exception as ex:                      # the probe is context, never a reason to lose the line
        probe = dict(error=str(ex))
    l2_gbs = probe.get("l2_read_gbs") if probe else None
    # T_roof = max(B_L2 / BW_L2, B_HBM / BW_HBM, F / P_FP32); each term as a fraction of the measured time
    frac_alu = achieved_lane / peak_lane
    frac_l2 = (tree_bytes / kernel_s / 1e9) / l2_gbs if l2_gbs else None
    tree_total = float(stats["node_bytes"] + stats["tri_bytes"])
    tree_in_l2 = tree_total < 100e6
    hbm_bytes = state_bytes + tree_total                                         # the state once, and one compulsory pass over the tree
    frac_hbm = (hbm_bytes / kernel_s / 1e9) / peaks["hbm_gbs"]
    terms = dict(alu=frac_alu, l2=frac_l2 or 0.0, hbm=frac_hbm)
    binding = max(terms, key=terms.get)
    roofline = dict(bound="alu", achieved=achieved_lane / 1e12, peak=peak_lane / 1e12, unit="Tlane-instr/s",
                    frac=frac_alu, traffic=None,
                    frac_alu=frac_alu, frac_l2=frac_l2, frac_hbm=frac_hbm, binding_term=binding, frac_of_t_roof=terms[binding],
                    frac_note="frac = frac_alu, the conservative (smaller) of the two terms that matter; T_roof of SURVEY.md 8(d) is the max of the "
                              "three terms, i.e. binding_term / frac_of_t_roof",
                    kernel="propagate_kernel" if args.legacy else "propagate_pool_kernel", kernel_ms=kernel_ms,
                    photon_steps_per_launch=steps_per_launch,
                    algorithmic_lane_instr_per_photon_step=alg_instr, algorithmic_tree_bytes_per_photon_step=alg_step_bytes,
                    algorithmic_state_bytes_per_photon=ALG_STATE_BYTES_PER_PHOTON,
                    algorithmic_bytes_per_launch=tree_bytes + state_bytes,
                    l2_side=dict(achieved_gbs=tree_bytes / kernel_s / 1e9, peak_gbs=l2_gbs, peak_source="dw_probe_peaks, this run",
                                 tree_bytes=int(stats["node_bytes"] + stats["tri_bytes"]), tree_resident_in_l2=bool(tree_in_l2)),
                    hbm_side=dict(achieved_gbs=hbm_bytes / kernel_s / 1e9, peak_gbs=peaks["hbm_gbs"], peak_source=peaks["source"]),
                    peak_derivation=f"{SM_COUNT} SMs x {LANES_PER_SM} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz ({peaks['source']} max SM clock)",
                    issue_probe=probe)
    # what the kernel actually does per photon-step: the counting instantiation, once over a sample, outside the timed region
    if not args.legacy and not args.literal and not args.no_counters:
        try:
            ns = min(n, args.counter_sample) if args.counter_sample > 0 else n
            hs = dw.DeviceHists(ctx.n_chan, 0, 0.0, 1.0, dev)
            ps = dw.DevicePhotons(ph.slice(0, ns), dev)
            ctx.propagate(ps, c.seed, c.max_steps, None, hs, flags=flags, stream=stream)
            torch.cuda.synchronize()
            S = float(hs.numpy()["total_steps"][0])
            k = ctx.propagate_counters(ps, c.seed, c.max_steps, flags=flags)
            q = max(k["queries_traced"], 1)
            roofline["implementation_counters"] = dict(
                sample_photons=ns, photon_steps=S,
                node_visits_per_step=k["node_visits"] / S, tri_tests_per_step=k["tri_tests"] / S,
                node_visits_per_traced_query=k["node_visits"] / q, tri_tests_per_traced_query=k["tri_tests"] / q,
                queries_traced_per_step=k["queries_traced"] / S, queries_skipped_share=k["queries_skipped"] / max(k["queries_skipped"] + k["queries_traced"], 1),
                tree_bytes_per_step=(k["node_visits"] * 112 + k["tri_tests"] * 48) / S,
                lanes_per_node_iteration=k["lanes_node"] / max(k["iters_node"], 1), lanes_per_triangle_iteration=k["lanes_leaf"] / max(k["iters_leaf"], 1),
                node_iterations_per_step=k["iters_node"] / S, triangle_iterations_per_step=k["iters_leaf"] / S,
                slots_per_physics_phase=(k["lanes_physics"] + k["lanes_fresh"]) / max(k["physics_phases"], 1),
                physics_phases_per_step=k["physics_phases"] / S,
                note="dw_propagate_counters (counting instantiation of the same kernel) over the first sample_photons of the batch; 112 B are "
                     "read per node visit and 48 B per triangle test; lanes per executed instruction and pipe utilisation need ncu: profiles/")
        except Exception as ex:
            roofline["implementation_counters"] = dict(error=str(ex))
    # measured DRAM traffic per launch of the dominant kernel, from the ncu capture named in the file (null if none for this workload)
    traffic_file = ROOT / "profiles" / "traffic.csv"
    if traffic_file.exists() and n == c.n_photons and not args.legacy:
        try:
            import csv
            for row in csv.DictReader(traffic_file.open()):
                if row["config"] == f"C{args.config}":
                    roofline["traffic"] = int(row["dram_bytes_per_launch"])
                    roofline["traffic_source"] = "NOT measured in this run: " + row["source"]
        except Exception:
            pass

    # what ncu measured for this kernel on this workload (issue slots, lanes per instruction, L1 / L2 throughput), beside the model
    cap_file = ROOT / "profiles" / "capture_metrics.csv"
    if cap_file.exists() and n == c.n_photons and not args.legacy:
        try:
            import csv
            rows = [r for r in csv.DictReader(cap_file.open()) if r["config"] == f"C{args.config}"]
            if rows:
                cap = {r["metric"]: float(r["value"]) for r in rows}
                cap["warp_instructions_per_photon_step"] = cap["smsp__inst_executed.sum"] / steps_per_launch if steps_per_launch else None
                cap["source"] = "NOT measured in this run: one ncu --set full capture of the same kernel and workload, profiles/capture_metrics.md"
                roofline["ncu_capture"] = cap
        except Exception:
            pass

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu, _ = cpu_baseline(c, args.ref_sample)

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=total_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                data="synthetic",
                config=dict(workload=c.name, photons_per_step_per_gpu=n, triangles=c.geometry.n_tri, max_steps=c.max_steps,
                            seed=c.seed, l2="inputs larger than L2 (440 MB photon state in, 320 MB results out per step)",
                            mode="literal" if args.literal else "bounded rays",
                            inputs="dw_emit on the device, a new batch of photon ids every step" if args.emit else "resident batch, same photons every step",
                            scheduler="legacy" if args.legacy else "pool", bvh_nodes=stats["n_nodes"],
                            bvh_build_ms=stats["build_ms"], bvh_rebuild_ms=rebuild_ms, bvh_leaves=stats["n_leaves"], bvh_depth=stats["max_depth"], grid_res=stats["grid_res"], bvh_refs=stats["n_refs"], split_div=stats["split_div"],
                            grid_free_cells=stats["grid_free_cells"], empty_skip=not args.no_skip and not args.legacy, launch=ctx.last_launch(),
                            **({"moved": args.move, "refit": refit_info} if args.move else {}),
                            **({"render": render_info} if render_info else {}),
                            **({"pipelined": pipelined} if pipelined else {}),
                            **({"sweep": sweep_info} if sweep_info else {}),
                            **({"design_study": study_info} if study_info else {})),
                photon_steps_per_s=total_steps / (total_ms * 1e-3),
                steps_per_photon=total_steps / (n_all * args.steps),
                fates={k: int(v) for k, v in zip(dw.FATE_NAMES, fate[:6])},
                clocks=clocks, ms_each=[round(v, 3) for v in per_step_ms], e2e=e2e, emission=emit_info, gpu_launches=int(launches) * (2 if args.emit else 1), roofline=roofline, cpu_baseline=cpu)
    print(json.dumps(line))
    dwdist.finalize()
    return 0


if __name__ == "__main__":
    sys.exit(main())
