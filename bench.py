#!/usr/bin/env python
"""bench.py -- fused TSDF + colour-volume integration throughput on B200 (one JSON line on stdout).

A *step* is one pass of the whole hot path (S0-S9: per-pixel pre-pass, then ONE persistent fused kernel that classifies
tiles, sets and scans the shell marks and integrates both volumes) over one synthetic RGB-D frame.  Workload at N = 1:
BASELINE.json configs[2] ("cfg3": geometry 512^3 over a 3 m cube, colour 1024^3, 640x480 depth, 1920x1080 RGB, 20
primitives on a plane, jittered orbit) -- the configuration the 70 % target is quoted on.

  value     whole-job voxel updates/s = (N_geo + N_col) voxels brought up to date per frame x frames / device time:
            exactly K steps enqueued one after the other between two CUDA events on the launching stream, inputs resident
            in HBM.  No L2 flush kernel: three volumes take the steps in turn, so consecutive steps work on different
            4.8 GB of memory (inputs larger than L2); --single-volume keeps them on one.
  flushed   the same K frames timed one by one with a 512 MiB flush before each (round 1's method; per_frame_ms)
  steady_state  the same after the arc has been swept until the weights are saturated (gate closed, stores skipped)
  stress    three saturating frames: free space, inside the truncation band, colour shell
  e2e       the same metric through vol_integrate_host (pinned HOST frames copied in, per-frame stats copied out)
  roofline  fused kernel: algorithmic bytes per launch (4 B x voxels read + 4 B x voxels changed + the two input images;
            sector_exact: 32 B x sectors touched) / its mean launch time (CUDA events inside the library, one frame at a
            time), against the measured HBM copy peak; step_frac: the same bytes over the whole step; traffic / issue: ncu
            figures from profiles/traffic.csv, quoted only if captured with the kernel sources this run was built from
  cpu_baseline  the CPU oracle, as it stands, on the first full-size frames of the same workload (rank 0, N = 1 only)

N > 1 (torchrun): every rank integrates an independent scan of the same configuration (replicas, no data-path
collective), value = sum over ranks / max-over-ranks time, "scaling": "weak".  With --shard the N
ranks integrate ONE scan as z-slab shards ("strong"); --shard-of R,W times one such shard alone on one GPU.
`--impl reference` times the CPU oracle alone (rank 0), each step a bounded sample of the workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "fused_voxel_updates_per_s"
UNIT = "voxel updates/s"


def parse(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=3, help="BASELINE config number 1..5 (default 3 = the headline workload)")
    ap.add_argument("--r", type=int, default=None, help="colour/geometry ratio override (config 4 sweep)")
    ap.add_argument("--no-flush", action="store_true", help="time frames back to back without flushing L2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--first-frame", type=int, default=0)
    ap.add_argument("--variant", type=int, default=0, choices=[0, 1, 2, 4],
                    help="alternative reading of the method (vol_opts_t.variant; both arms); 0 = the headline path")
    ap.add_argument("--stress", default=None, choices=list(synth.STRESS_KINDS),
                    help="time ONE saturating frame kind of SURVEY 8(d) item 5 as the main workload instead of the scan "
                         "(the default run reports all three under \"stress\")")
    ap.add_argument("--no-stress", action="store_true", help="skip the three saturating frames")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: ONE scan on N GPUs -- rank k owns the z-slabs k mod N of both volumes (vol_opts_t.shard_*), every rank "
                         "receives every frame; value = one scan's voxels / max-over-ranks time, scaling = strong")
    ap.add_argument("--shard-of", default=None, metavar="R,W",
                    help="single process: time shard R of W alone on this GPU (what rank R of a W-GPU --shard run would do)")
    ap.add_argument("--single-volume", action="store_true", help="all timed steps on one volume (default: three volumes take them in turn)")
    ap.add_argument("--steady-frames", type=int, default=150,
                    help="frames swept back and forth over the arc before the steady-state window (0 = skip it)")
    return ap.parse_args(argv)


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_source_hash():
    """sha256 (first 16 hex digits) over the CUDA sources the hot path (k_prepass, k_fused and their launch code) is built
    from: ncu figures recorded for another build of it are not quoted.  (The ray caster, the front end and the static-scratch
    ICP step live in other files of the same library and do not change these kernels.)"""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1602_06645_b200", "csrc")
    for name in ("exact.cuh", "fused.cuh", "params.cuh", "prepass.cuh", "volfusion.cu"):
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def ncu_record(workload):
    """The committed ncu --set full figures of k_fused for this workload (profiles/traffic.csv:
    workload,kernel,dram_bytes_per_launch,warp_instructions_per_launch,source_hash) -- only if they were captured with the
    kernel sources this run was built from (source_hash = kernel_source_hash()); None otherwise, so that a stale capture is
    never quoted beside a live timing."""
    try:
        want = kernel_source_hash()
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                cols = [c.strip() for c in line.split(",")]
                if len(cols) >= 5 and cols[0] == workload and cols[1] == "k_fused" and cols[4] == want:
                    return {"dram_bytes": float(cols[2]), "warp_instructions": float(cols[3])}
    except Exception:
        pass
    return None


def ncu_block(workload):
    """traffic / warp instructions of k_fused for a secondary workload, from profiles/traffic.csv (null on another build)"""
    rec = ncu_record(workload)
    return {"traffic": rec["dram_bytes"] if rec else None, "warp_instructions_per_launch": rec["warp_instructions"] if rec else None}


def issue_roofline(rec, fused_ms_mean, sm_mhz, n_sms):
    """The bound the fused kernel actually runs into: warp instructions issued per second against
    SMs x 4 schedulers x 1 instruction per cycle at the SM clock seen during the run.  The instruction count per launch comes
    from the committed ncu capture of the same build (it cannot be measured outside a profiler)."""
    if rec is None or not sm_mhz:
        return None
    peak = n_sms * 4 * sm_mhz * 1e6
    achieved = rec["warp_instructions"] / (fused_ms_mean * 1e-3)
    return {"bound": "alu", "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "T warp-instructions/s", "frac": achieved / peak,
            "warp_instructions_per_launch": rec["warp_instructions"], "sms": n_sms,
            "source": "profiles/traffic.csv (ncu smsp__inst_executed.sum, same kernel sources)"}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons while the benchmark runs (the profiling recipe's clocks line)."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,utilization.gpu"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc:
            self.proc.terminate()
        self.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        busy = [float(r[0]) for r in self.rows if len(r) >= 7 and r[6].isdigit() and int(r[6]) > 0 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 7 for n, v in zip(names, r[2:6]) if v.lower().startswith("active")})
        use = busy or sm
        return {"sm_mhz": float(np.median(use)) if use else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "samples_under_load": len(busy)}


class NvmlClocks:
    """SM clock and throttle reasons read through NVML from this process: polled while the timed frames are still running on
    the device (the timed region is only milliseconds long, shorter than nvidia-smi's sampling period)."""

    def __init__(self, index):
        self.h, self.sm, self.reasons = None, [], set()
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
        except Exception:
            self.h = None

    def sample(self):
        if self.h is None:
            return
        try:
            nv = self.nv
            self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
            r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            for name, bit in (("hw_slowdown", 0x8), ("sw_power_cap", 0x4), ("sw_thermal_slowdown", 0x20), ("hw_thermal_slowdown", 0x40)):
                if r & bit:
                    self.reasons.add(name)
        except Exception:
            pass


def workload_name(c):
    var = getattr(c, "variant", 0)
    return (f"{c.name}: geometry {c.dims_geo[0]}^3 over {c.extent} m, colour {c.dims_col[0]}^3 (r={c.r}), depth {c.wd}x{c.hd}, "
            f"rgb {c.wh}x{c.hh}" + (f" -- alternative reading {var} (vol_opts_t.variant)" if var else ""))


def oracle_sample(c, n_frames, slab_layers=None):
    """Time the CPU oracle (as it stands) on `n_frames` frames.  slab_layers = None: the full volumes; otherwise a central
    z-slab of that many geometry layers (and r x as many colour layers) -- a bounded sample of the same workload."""
    import oracle
    oracle.build()
    nx, ny, nz = c.dims_geo
    origin = np.array(c.origin, np.float32)
    if slab_layers is not None and slab_layers < nz:
        k0 = (nz - slab_layers) // 2
        origin = origin.copy()
        origin[2] += np.float32(k0) * np.float32(c.voxel)
        dims = (nx, ny, slab_layers)
        sample = f"central z-slab of {slab_layers}/{nz} geometry layers (and {slab_layers * c.r} colour layers), {n_frames} frames"
    else:
        dims = (nx, ny, nz)
        sample = f"full volumes, first {n_frames} frames"
    o = oracle.RefVolume(dims, c.r, origin, c.extent, c.mu, c.w_max, sigma=c.sigma, gate=c.gate, variant=getattr(c, "variant", 0))
    o.desc.extent = float(np.float32(c.voxel) * np.float32(nx))
    nvox = dims[0] * dims[1] * dims[2] * (1 + c.r ** 3)
    times = []
    for i in range(n_frames):
        depth, rgb, T = synth.frame(c, i)
        t0 = time.perf_counter()
        o.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        times.append(time.perf_counter() - t0)
    # the same oracle volumes ray-cast once from the last pose (reported beside the GPU's vol_raycast time)
    t0 = time.perf_counter()
    o.raycast(c.wd, c.hd, T, c.K_depth, 0.3, 8.0)
    oracle_sample.raycast_ms = 1e3 * (time.perf_counter() - t0)
    return nvox, times, sample


def run_reference(args, rank):
    """--impl reference: the CPU oracle on this box's host cores, rank 0 only; each step = one frame over a z-slab sample."""
    if rank != 0:
        return
    c = synth.config(args.cfg, r=args.r)
    c.variant = args.variant
    import oracle
    cores = oracle.threads()
    slab = max(8, c.dims_geo[2] // 16)
    nvox, times, sample = oracle_sample(c, args.warmup + args.steps, slab_layers=slab)
    t = times[args.warmup:]
    ms = 1e3 * float(np.mean(t))
    val = nvox / (ms * 1e-3)
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": workload_name(c), "sample_per_step": sample},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def max_over_ranks(values, world, device):
    """Device times are reported as the MAX over ranks (one all-reduce; identity at world 1)."""
    if world == 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(nvox_per_rank, steps, world, total_ms):
    """Whole-job aggregate: voxels brought up to date by all ranks / max-over-ranks device time."""
    return world * nvox_per_rank * steps / (total_ms * 1e-3)


STAT_KEYS = ("geo_read", "geo_changed", "col_read", "col_changed", "geo_sectors_read", "geo_sectors_written", "col_sectors_read",
             "col_sectors_written", "geo_visited", "col_gated", "geo_skippable", "geo_sectors_skippable", "tiles_geo", "subs_geo",
             "items_col", "cells_col", "jobs_mark")
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json: "B200's ~8 TB/s peak"


def stats_row(s):
    return [float(getattr(s, k)) for k in STAT_KEYS]


def bytes_of(cnt, frame_bytes):
    """Algorithmic bytes per fused launch from a (frames x STAT_KEYS) array: voxel-exact
    4 (geo_read + geo_changed + col_read + col_changed) + the two images, the same at 32-byte sector granularity, and what
    the plain kernel really has to touch (without the saturated free space it leaves out)."""
    k = {n: cnt[:, i] for i, n in enumerate(STAT_KEYS)}
    voxel = 4.0 * (k["geo_read"] + k["geo_changed"] + k["col_read"] + k["col_changed"]) + frame_bytes
    sector = 32.0 * (k["geo_sectors_read"] + k["geo_sectors_written"] + k["col_sectors_read"] + k["col_sectors_written"]) + frame_bytes
    touched = voxel - 4.0 * k["geo_skippable"]
    touched_sector = sector - 32.0 * k["geo_sectors_skippable"]
    return voxel, sector, touched, touched_sector


class Window:
    """Counts, per-kernel times and the timed passes of one list of frames.  Step s integrates frame s into volume s mod N of
    `vols`: with N = 3 volumes taking the steps in turn, a volume's lines are touched again only after two other steps have
    moved their own ~290 MB through the 126 MB L2 -- the inputs of consecutive timed steps are larger than L2 without any
    flush kernel between them.  Every pass uses the same schedule, so the counters belong to exactly the timed steps."""

    def __init__(self, vols, frames, c, stream, flush_buf, flush):
        self.vols = vols if isinstance(vols, (list, tuple)) else [vols]
        self.vol = self.vols[0]
        self.frames, self.c, self.stream, self.flush_buf, self.flush = frames, c, stream, flush_buf, flush

    def integrate(self, fr, s=0):
        _, _, dd, dr, T = fr
        c = self.c
        v = self.vols[s % len(self.vols)]
        v.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=self.stream)
        return v

    def count(self):
        """(untimed) per-step counters of exactly these steps, from the counting variant"""
        for v in self.vols:
            v.set_counting(True)
        rows = []
        for s, fr in enumerate(self.frames):
            v = self.integrate(fr, s)
            rows.append(stats_row(v.frame_stats(self.stream)))
        for v in self.vols:
            v.set_counting(False)
        return np.array(rows, dtype=np.float64)

    def kernel_times(self):
        """(untimed) per-kernel times (library-side CUDA events on the launching stream)"""
        for v in self.vols:
            v.set_profiling(True)
        kms = []
        for s, fr in enumerate(self.frames):
            if self.flush:
                self.flush_buf.zero_()
            v = self.integrate(fr, s)
            kms.append(v.last_kernel_ms())
        for v in self.vols:
            v.set_profiling(False)
        return np.array(kms)

    def back_to_back(self, torch, barrier, nvml=None):
        """THE timed pass: the steps enqueued with nothing between them (no flush kernel, no event): one pair of events around
        all of them.  Only here can the pre-pass of step n + 1 start under the tail of step n's fused kernel (programmatic
        dependent launch)."""
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t0.record(self.stream)
        for s, fr in enumerate(self.frames):
            self.integrate(fr, s)
        t1.record(self.stream)
        while nvml and not t1.query():
            nvml.sample()
        barrier()
        return float(t0.elapsed_time(t1)) / len(self.frames)

    def timed(self, torch, barrier, nvml=None):
        """the same steps one by one: events around every step, L2 flushed (512 MiB memset) before each"""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in self.frames]
        barrier()
        for n, fr in enumerate(self.frames):
            if self.flush:
                self.flush_buf.zero_()
            ev[n][0].record(self.stream)
            self.integrate(fr, n)
            ev[n][1].record(self.stream)
            if nvml and n % 4 == 3:
                nvml.sample()                                     # the device is busy with the frames enqueued so far
        while nvml and not ev[-1][1].query():
            nvml.sample()
        barrier()
        return np.array([a.elapsed_time(b) for a, b in ev])


def roofline_block(alg_voxel, alg_sector, touched, touched_sector, fused_ms, step_ms, peak):
    """Fractions of the HBM roofline of one window: algorithmic bytes over the fused kernel's time (and over the whole step)."""
    t_f, t_s = fused_ms.sum() * 1e-3, step_ms.sum() * 1e-3
    gbs = lambda b, t: float(b.sum() / t / 1e9)
    out = {"achieved": gbs(alg_voxel, t_f), "frac": gbs(alg_voxel, t_f) / peak, "frac_of_nominal_8tbs": gbs(alg_voxel, t_f) / NOMINAL_HBM_GBS,
           "step_frac": gbs(alg_voxel, t_s) / peak,
           "sector_exact": {"bytes": float(alg_sector.mean()), "achieved": gbs(alg_sector, t_f), "frac": gbs(alg_sector, t_f) / peak}}
    if float((alg_voxel - touched).sum()) > 0.0:
        out["touched"] = {"bytes": float(touched.mean()), "sector_bytes": float(touched_sector.mean()),
                          "frac": gbs(touched, t_f) / peak, "sector_frac": gbs(touched_sector, t_f) / peak,
                          "note": "without the saturated free space the plain kernel leaves out (read and unchanged by definition): "
                                  "the bytes it really has to move"}
    return out


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist

    import paper_1602_06645_b200 as vf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    c = synth.config(args.cfg, r=args.r)
    c.variant = args.variant
    W, K = args.warmup, args.steps
    nfr = W + K
    shard_rank, shard_world = (rank, world) if args.shard else (0, 1)
    if args.shard_of:
        shard_rank, shard_world = (int(t) for t in args.shard_of.split(","))
    sharded = shard_world > 1
    scans = 1 if args.shard else world                        # independent scans in the job
    first = args.first_frame + (0 if args.shard else 7 * rank)     # replicas scan different parts of the trajectory
    sampler = ClockSampler(local_rank) if rank == 0 else None
    if sampler:
        sampler.start()
    n_sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
    peak, peak_src = peaks()
    frame_bytes = c.wd * c.hd * 2 + c.wh * c.hh * 3
    stream = torch.cuda.current_stream()
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def upload(fr):
        depth, rgb, T = fr
        hd_, hr_ = torch.from_numpy(depth.view(np.int16)).pin_memory(), torch.from_numpy(rgb).pin_memory()
        return (hd_, hr_, hd_.cuda(), hr_.cuda(), T)

    # ---- inputs: generated once, pinned on the host and resident on the device
    stress_kind = args.stress if args.stress in synth.STRESS_KINDS else None
    mu, sigma = synth.stress_params(c, stress_kind) if stress_kind else (c.mu, c.sigma)
    frames = [upload(synth.stress_frame(c, i, stress_kind) if stress_kind else synth.frame(c, (first + i) % c.n_frames)) for i in range(nfr)]
    vol = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, mu, c.w_max, sigma=sigma, gate=c.gate, device=local_rank,
                    variant=getattr(c, "variant", 0), shard_rank=shard_rank, shard_world=shard_world)
    warm, timed = frames[:W], frames[W:]
    # Three volumes take the timed steps in turn (Window): their 3 x (N_geo + N_col) x 4 bytes must fit beside everything else
    n_rot = 1 if (stress_kind or args.single_volume or 3 * 4 * int(np.prod(c.dims_geo)) * (1 + c.r ** 3) > 100e9) else 3
    vols = [vol] + [vf.Volume(c.dims_geo, c.r, c.origin, c.extent, mu, c.w_max, sigma=sigma, gate=c.gate, device=local_rank,
                              variant=getattr(c, "variant", 0), shard_rank=shard_rank, shard_world=shard_world) for _ in range(n_rot - 1)]
    win = Window(vols, timed, c, stream, flush_buf, not args.no_flush)

    def warm_up():
        for n, v in enumerate(vols):
            v.reset(stream)
            for fr in warm:
                win.integrate(fr, n)

    # ---- pass 1 (untimed): per-frame voxel and sector counters of exactly the timed frames -> algorithmic bytes
    warm_up()
    cnt = win.count()
    # ---- pass 2 (untimed): per-kernel times of the timed frames
    warm_up()
    kms = win.kernel_times()
    # ---- pass 3: THE timed region -- K frames, device-resident inputs, events around every frame, L2 flushed between
    warm_up()
    nvml = NvmlClocks(local_rank) if rank == 0 else None
    per_frame_ms = win.timed(torch, barrier, nvml)
    flushed_ms = float(per_frame_ms.sum())
    # ---- pass 3b: THE timed region -- exactly K steps between two events, nothing else on the stream (the frames differ from
    #      one another, 6.8 MB each, and each touches > 100 MB of volumes of 2.7 GB: larger than L2 without a flush)
    warm_up()
    total_ms = win.back_to_back(torch, barrier, nvml) * K

    # ---- steady state of a long scan (same volume): the arc is swept back and forth until the weights are saturated
    #      (w = w_max wherever the arc sees free space or the surface, the 0.8 gate mostly closed), then the same frames
    #      are counted, profiled and timed again
    steady = None
    if args.steady_frames > 0 and not stress_kind:
        order = list(range(nfr)) + list(range(nfr - 2, 0, -1))
        for n in range(args.steady_frames):
            for k in range(len(vols)):
                win.integrate(frames[order[n % len(order)]], k)
        s_cnt = win.count()
        s_kms = win.kernel_times()
        s_flushed = win.timed(torch, barrier)
        s_ms = np.full(K, win.back_to_back(torch, barrier))
        av, asec, tch, tchs = bytes_of(s_cnt, frame_bytes)
        steady = {"frames_before": nfr * 3 + args.steady_frames + 3 * K, "ms_per_step": float(s_ms.mean()), "ms_per_step_flushed": float(s_flushed.mean()),
                  "kernel_ms_mean": {"prepass": float(s_kms[:, 0].mean()), "fused": float(s_kms[:, 2].mean())},
                  "per_frame_mean": {k: float(s_cnt[:, i].mean()) for i, k in enumerate(STAT_KEYS)},
                  "algorithmic_bytes": float(av.mean()),
                  "roofline": dict(roofline_block(av, asec, tch, tchs, s_kms[:, 2], s_ms, peak), **ncu_block(c.name + "-steady")),
                  "note": "the timed frames again after the arc has been swept back and forth: geometry weights saturated at w_max, "
                          "colour gate mostly closed (col_changed << col_read), stores skipped where the word does not change"}

    # ---- pass 4: end to end through vol_integrate_host -- pinned host frames in, per-frame stats out, every step.
    #      Frames are enqueued back to back, as when a recorded sequence is fused: the library copies frame n + 1 while the
    #      kernels of frame n run (two staging sets), and the step's result (the 128-byte statistics record) comes back with
    #      vol_frame_stats_async into pinned memory, in stream order.
    vol.reset(stream)
    raw_stats = torch.zeros((max(K, W), vf.VOL_STATS_RAW_BYTES // 8), dtype=torch.int64).pin_memory()
    for i in range(W):                                            # warm-up through the same entry point (staging buffers exist)
        hd_, hr_, _, _, T = frames[i]
        vol.integrate_host(hd_, hr_, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        vol.frame_stats_async(raw_stats[i], stream)
    barrier()
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for n, i in enumerate(range(W, nfr)):
        hd_, hr_, _, _, T = frames[i]
        vol.integrate_host(hd_, hr_, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        vol.frame_stats_async(raw_stats[n], stream)               # device -> host read of the step's result
    t1.record(stream)
    barrier()
    e2e_ms = float(t0.elapsed_time(t1))
    e2e_tiles = [vol.decode_stats(raw_stats[n]).tiles_geo for n in range(K)]
    assert min(e2e_tiles) > 0, "a frame of the end-to-end pass visited no tile"

    # ---- pass 4b: the same, one frame at a time (a live scan: the caller waits for every frame's result before the next)
    vol.reset(stream)
    for i in range(W):
        hd_, hr_, _, _, T = frames[i]
        vol.integrate_host(hd_, hr_, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        vol.frame_stats(stream)
    barrier()
    t2 = torch.cuda.Event(enable_timing=True); t3 = torch.cuda.Event(enable_timing=True)
    t2.record(stream)
    for i in range(W, nfr):
        hd_, hr_, _, _, T = frames[i]
        vol.integrate_host(hd_, hr_, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        vol.frame_stats(stream)                                   # synchronises
    t3.record(stream)
    barrier()
    e2e_serial_ms = float(t2.elapsed_time(t3))

    # ---- the saturating frames of SURVEY 8(d) item 5, on volumes of the same size (each kind with the mu / sigma it needs):
    #      counted, profiled and timed like the scan, a few frames each.  Parity: tests/test_gpu_parity.py::test_stress_*.
    stress = None
    if world == 1 and not sharded and not stress_kind and not args.no_stress:
        stress = {}
        for kind in synth.STRESS_KINDS:
            s_mu, s_sigma = synth.stress_params(c, kind)
            nw_, nt_ = (1, 2) if kind == "colour" else (2, 4)
            sfr = [upload(synth.stress_frame(c, i, kind)) for i in range(nw_ + nt_)]
            svol = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, s_mu, c.w_max, sigma=s_sigma, gate=c.gate, device=local_rank)
            swin = Window(svol, sfr[nw_:], c, stream, flush_buf, not args.no_flush)
            res = []
            for what in ("count", "kernel_times", "timed", "back_to_back"):
                svol.reset(stream)
                for fr in sfr[:nw_]:
                    swin.integrate(fr)
                res.append(swin.count() if what == "count" else swin.kernel_times() if what == "kernel_times" else
                           swin.timed(torch, barrier) if what == "timed" else np.full(nt_, swin.back_to_back(torch, barrier)))
            s_cnt, s_kms, s_flushed, s_ms = res
            av, asec, tch, tchs = bytes_of(s_cnt, frame_bytes)
            stress[kind] = {"frames": nt_, "ms_per_step": float(s_ms.mean()), "ms_per_step_flushed": float(s_flushed.mean()),
                            "fused_ms": float(s_kms[:, 2].mean()),
                            "mu_m": s_mu, "sigma_m": s_sigma, "algorithmic_bytes": float(av.mean()),
                            "geo_read": float(s_cnt[:, 0].mean()), "col_read": float(s_cnt[:, 2].mean()),
                            "roofline": dict(roofline_block(av, asec, tch, tchs, s_kms[:, 2], s_ms, peak), **ncu_block(f"{c.name}-stress-{kind}"))}
            svol.close()
            del svol, sfr
            torch.cuda.empty_cache()

    # (a shard does not hold the whole volume: the rows beyond the hot path are measured on unsharded volumes only)
    raycast_ms = raycast_hit = raycast_tri_ms = rc_fresh = tracking = sample_ms = sample_filled = sample_tri_ms = None
    sp_pts = None
    if not sharded:
        # ---- NEXT row, outside the timed regions: vol_raycast of the volumes as they stand now, from the
        #      last frame's pose, one 640 x 480 (depth-camera sized) image per call
        rc_depth = torch.empty(c.wd * c.hd, dtype=torch.float32, device="cuda")
        rc_rgb = torch.empty(c.wd * c.hd * 3, dtype=torch.uint8, device="cuda")
        T_last = frames[nfr - 1][4]
        for _ in range(3):
            vol.raycast(c.wd, c.hd, T_last, c.K_depth, 0.3, 8.0, rc_depth, rc_rgb, stream=stream)
        r0 = torch.cuda.Event(enable_timing=True); r1 = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        r0.record(stream)
        for _ in range(10):
            vol.raycast(c.wd, c.hd, T_last, c.K_depth, 0.3, 8.0, rc_depth, rc_rgb, stream=stream)
        r1.record(stream)
        torch.cuda.synchronize()
        raycast_ms = float(r0.elapsed_time(r1)) / 10.0
        raycast_hit = float((rc_depth > 0).float().mean())
        for _ in range(3):
            vol.raycast_trilinear(c.wd, c.hd, T_last, c.K_depth, 0.3, 8.0, rc_depth, rc_rgb, stream=stream)
        torch.cuda.synchronize()
        r0.record(stream)
        for _ in range(10):
            vol.raycast_trilinear(c.wd, c.hd, T_last, c.K_depth, 0.3, 8.0, rc_depth, rc_rgb, stream=stream)
        r1.record(stream)
        torch.cuda.synchronize()
        raycast_tri_ms = float(r0.elapsed_time(r1)) / 10.0
        # the same right after a frame has been integrated: the casters' skip flags are rebuilt from the volume first
        rc_fresh = {}
        for name, fn in (("nearest", vol.raycast), ("trilinear", vol.raycast_trilinear)):
            ts = []
            for fr in frames[-4:]:
                win.integrate(fr)
                r0.record(stream)
                fn(c.wd, c.hd, T_last, c.K_depth, 0.3, 8.0, rc_depth, None, stream=stream)
                r1.record(stream)
                torch.cuda.synchronize()
                ts.append(float(r0.elapsed_time(r1)))
            rc_fresh[name] = float(np.mean(ts[1:]))
        vol.raycast(c.wd, c.hd, T_last, c.K_depth, 0.3, 8.0, rc_depth, rc_rgb, stream=stream)       # (the sampling figures below use these hits)
        torch.cuda.synchronize()
        # ---- NEXT row: the tracker -- front end of the last frame, prediction ray-cast from the pose before
        #      it, coarse-to-fine ICP (19 steps, each a kernel and a 232-byte read-back); the tracked pose against the true one
        tracking = None
        if not stress_kind and nfr >= 2:
            fe = vf.Frontend(c.wd, c.hd, 3, device=local_rank, trilinear_prediction=True)
            T_prev, dd_last = np.asarray(frames[nfr - 2][4], np.float32), frames[nfr - 1][2]
            tms = {"measure": [], "predict": [], "track": []}
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            T_rel, trk_rms, trk_cnt, lost = np.eye(4, dtype=np.float32), float("nan"), 0, None
            for rep in range(6):
                evs[0].record(stream)
                fe.measure(dd_last, c.K_depth, stream=stream)
                evs[1].record(stream)
                fe.predict(vol, T_prev, c.K_depth, 0.3, 8.0, stream=stream)
                evs[2].record(stream)
                try:
                    T_rel, trk_rms, trk_cnt = fe.track(stream=stream)
                except vf.VolError as e:                          # VOL_E_LOST: e.g. the sphere of config 1 (rotations about its centre unobservable)
                    if e.code != vf.VOL_E_LOST:
                        raise
                    lost = str(e)
                evs[3].record(stream)
                torch.cuda.synchronize()
                if rep >= 2:
                    for k, name in enumerate(("measure", "predict", "track")):
                        tms[name].append(float(evs[k].elapsed_time(evs[k + 1])))
            T_trk = T_prev.astype(np.float64) @ T_rel.astype(np.float64)
            trk_status, trk_level, trk_cond = fe.track_info()
            tracking = {"status": "lost: " + lost if lost else "ok", "conditioning": trk_cond, "measure_ms": float(np.mean(tms["measure"])), "predict_ms": float(np.mean(tms["predict"])),
                        "track_ms": float(np.mean(tms["track"])), "icp_steps": 19, "correspondences": int(trk_cnt), "rms_mm": 1e3 * trk_rms,
                        "pose_error_mm": 1e3 * float(np.linalg.norm(T_trk[:3, 3] - np.asarray(T_last, np.float64)[:3, 3])),
                        "motion_mm": 1e3 * float(np.linalg.norm(T_prev[:3, 3] - np.asarray(T_last, np.float32)[:3, 3])),
                        "prediction": "vol_raycast_trilinear, no F8 (opts.trilinear_prediction)",
                        "note": "vol_frontend_measure / _predict / _track (SURVEY 8(f) rank 4) of the last frame against the fused volumes, "
                                "not part of the timed step"}
            fe.close()
        # ---- NEXT row: vol_sample_colour at surface points -- the ray-cast hit points, 8 jittered copies
        #      each (about the density of a texture map with Size_pixel = one colour voxel), as a polygon texture map would ask
        Tl = torch.from_numpy(np.asarray(T_last, np.float32)).cuda()
        yy, xx = torch.meshgrid(torch.arange(c.hd, device="cuda", dtype=torch.float32), torch.arange(c.wd, device="cuda", dtype=torch.float32), indexing="ij")
        zz = rc_depth.reshape(c.hd, c.wd)
        cam = torch.stack([(xx - float(c.K_depth[0, 2])) / float(c.K_depth[0, 0]) * zz, (yy - float(c.K_depth[1, 2])) / float(c.K_depth[1, 1]) * zz, zz], dim=-1)
        hit_pts = (cam.reshape(-1, 3) @ Tl[:3, :3].T + Tl[:3, 3])[rc_depth > 0]
        gen = torch.Generator(device="cuda"); gen.manual_seed(1)
        sp_pts = (hit_pts.repeat(8, 1) + (torch.rand(hit_pts.shape[0] * 8, 3, device="cuda", generator=gen) - 0.5) * (2.0 * c.voxel / c.r)).contiguous()
        sp_out = torch.empty(sp_pts.shape[0], dtype=torch.int32, device="cuda")
        sample_ms, sample_filled, sample_tri_ms = None, None, None
        if sp_pts.shape[0] > 0:
            for _ in range(3):
                vol.sample_colour(sp_pts, sp_pts.shape[0], sp_out, stream=stream)
            torch.cuda.synchronize()
            r0.record(stream)
            for _ in range(10):
                vol.sample_colour(sp_pts, sp_pts.shape[0], sp_out, stream=stream)
            r1.record(stream)
            torch.cuda.synchronize()
            sample_ms = float(r0.elapsed_time(r1)) / 10.0
            sample_filled = float(((sp_out.view(torch.int32) >> 24) != 0).float().mean())
            for _ in range(3):
                vol.sample_colour_trilinear(sp_pts, sp_pts.shape[0], sp_out, stream=stream)
            torch.cuda.synchronize()
            r0.record(stream)
            for _ in range(10):
                vol.sample_colour_trilinear(sp_pts, sp_pts.shape[0], sp_out, stream=stream)
            r1.record(stream)
            torch.cuda.synchronize()
            sample_tri_ms = float(r0.elapsed_time(r1)) / 10.0
    total_ms, flushed_ms, e2e_ms, e2e_serial_ms = max_over_ranks([total_ms, flushed_ms, e2e_ms, e2e_serial_ms], world, "cuda")
    clocks = sampler.stop() if sampler else None
    if clocks is not None and nvml is not None and nvml.sm:
        # clocks DURING the timed region (NVML, in-process); the nvidia-smi figures cover the whole run
        clocks.update({"sm_mhz_whole_run": clocks["sm_mhz"], "sm_mhz": float(np.median(nvml.sm)), "samples_timed_region": len(nvml.sm),
                       "reasons": sorted(set(clocks["reasons"]) | nvml.reasons)})
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    nvox = int(np.prod(c.dims_geo)) * (1 + c.r ** 3)
    ms_per_step = total_ms / K
    value = whole_job_value(nvox, K, scans, total_ms)
    e2e_value = whole_job_value(nvox, K, scans, e2e_ms)
    fused_ms = kms[:, 2]
    av, asec, tch, tchs = bytes_of(cnt, frame_bytes)
    wl_key = c.name + (f"-stress-{stress_kind}" if stress_kind else "") + (f"-variant{args.variant}" if args.variant else "")
    rec = ncu_record(wl_key)
    roof = {"bound": "hbm", "kernel": "k_fused", "peak": peak, "unit": "GB/s", "peak_source": peak_src}
    roof.update(roofline_block(av, asec, tch, tchs, fused_ms, np.full(K, ms_per_step), peak))
    roof.update({"traffic": rec["dram_bytes"] if rec else None,
                 "traffic_source": "profiles/traffic.csv: ncu dram__bytes_read.sum + dram__bytes_write.sum per k_fused launch, captured with "
                                   "these kernel sources (hash " + kernel_source_hash() + ")" if rec else
                                   "null: no ncu capture of these kernel sources is committed (hash " + kernel_source_hash() + ")",
                 "dense_sweep_frac": float(8.0 * nvox / (fused_ms.mean() * 1e-3) / 1e9 / peak),
                 "issue": issue_roofline(rec, float(fused_ms.mean()), (clocks or {}).get("sm_mhz"), n_sms)})
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(c) + (f" -- STRESS: saturating frame ({stress_kind})" if stress_kind else ""),
                   "value_kind": "visited: (N_geo + N_col) voxels brought up to date per frame x frames / device time -- about 1 % of them "
                                 "are touched (applied_updates_per_s counts those); the reference arm uses the same convention",
                   "frames": "one saturating pose, the wall moving" if stress_kind else f"{first}..{first + nfr - 1} of the seeded trajectory",
                   "l2": (f"no flush: inputs larger than L2 -- {n_rot} volumes of {4e-9 * nvox:.1f} GB take the K steps in turn, each step a "
                          "distinct frame (6.8 MB) that moves > 100 MB of its volume, so a volume's lines are touched again only "
                          "after the other volumes' steps have gone through the 126 MB L2" if n_rot > 1 else
                          "no flush, one volume: K distinct frames, each moving its own part of the volume") +
                         "; the figure with a 512 MiB flush before every step is under \"flushed\"",
                   "parallelism": (f"shard {shard_rank} of {shard_world} alone (z-slabs {shard_rank} mod {shard_world}): its share of one scan" if args.shard_of else
                                   "single GPU" if world == 1 else
                                   f"one scan on {world} z-slab shards, every rank receives every frame, no data-path collective; counters are rank 0's shard" if args.shard else
                                   f"{world} replicas (independent scans), no data-path collective")},
        "frames_per_s": scans * K / (total_ms * 1e-3),
        "applied_updates_per_s": scans * float(cnt[:, 0].sum() + cnt[:, 2].sum()) / (total_ms * 1e-3),
        "per_frame_ms": {"median": float(np.median(per_frame_ms)), "p95": float(np.percentile(per_frame_ms, 95)), "min": float(per_frame_ms.min())},
        "kernel_ms_mean": {"prepass": float(kms[:, 0].mean()), "fused": float(fused_ms.mean())},
        "flushed": None if args.no_flush else {
            "ms_per_step": flushed_ms / K, "value": whole_job_value(nvox, K, scans, flushed_ms),
            "note": "the same K frames timed one by one (a pair of events around each, L2 flushed by a 512 MiB memset before each; "
                    "per_frame_ms are these): round 1's headline method.  Nothing can overlap from one frame to the next "
                    "here; in the timed region proper the next frame's pre-pass starts under the tail of the fused kernel "
                    "(programmatic dependent launch), which is most of the difference"},
        "per_frame_mean": dict({k: float(cnt[:, i].mean()) for i, k in enumerate(STAT_KEYS)}, algorithmic_bytes=float(av.mean()),
                               sector_exact_bytes=float(asec.mean())),
        "instructions_hint": None if rec is None else {
            "warp_instructions_per_launch": rec["warp_instructions"],
            "thread_instructions_per_visited_voxel": 32.0 * rec["warp_instructions"] / float(cnt[:, 8].mean() + cnt[:, 9].mean()),
            "note": "ncu smsp__inst_executed.sum x 32 / (geometry voxels projected + colour voxels gated); all roles of the kernel included"},
        "roofline": roof,
        "steady_state": steady,
        "stress": stress,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms / K, "h2d_bytes_per_step": frame_bytes,
                "d2h_bytes_per_step": vf.VOL_STATS_RAW_BYTES,
                "mode": "vol_integrate_host + vol_frame_stats_async per frame, frames enqueued back to back (a recorded "
                        "sequence): the copies of frame n + 1 overlap the kernels of frame n",
                "one_frame_at_a_time": {"value": whole_job_value(nvox, K, scans, e2e_serial_ms), "ms_per_step": e2e_serial_ms / K,
                                        "mode": "vol_integrate_host + vol_frame_stats (synchronises) per frame (a live scan)"}},
        "tracking": tracking,
        "raycast": None if raycast_ms is None else {"ms": raycast_ms, "rays_per_s": c.wd * c.hd / (raycast_ms * 1e-3), "image": f"{c.wd}x{c.hd}", "hit_fraction": raycast_hit,
                    "trilinear_ms": raycast_tri_ms, "after_a_new_frame_ms": rc_fresh,
                    "note": "vol_raycast / vol_raycast_trilinear of the fused volumes (SURVEY 8(f) rank 1), not part of the timed step; "
                            "ms: repeated casts of an unchanged volume; after_a_new_frame_ms: depth only, including the rebuild of the "
                            "casters' skip flags that the first cast after a vol_integrate does"},
        "sample_colour": None if sample_ms is None else {
            "ms": sample_ms, "points": int(sp_pts.shape[0]), "points_per_s": sp_pts.shape[0] / (sample_ms * 1e-3), "filled_fraction": sample_filled,
            "trilinear_ms": sample_tri_ms,
            "note": "vol_sample_colour at jittered surface points (SURVEY 8(f) rank 3), not part of the timed step"},
        "gpu_launches": vol.launches_per_frame() * K,
        "clocks": clocks,
    }
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        n = 2 if nvox > 5e8 else (4 if nvox > 5e7 else 5)
        nv, times, sample = oracle_sample(c, min(n, c.n_frames))
        out["cpu_baseline"] = {"value": nv * len(times) / sum(times), "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
                               "sample": sample, "ms_per_frame": 1e3 * float(np.mean(times)),
                               "omp_get_max_threads": oracle.threads(), "nproc": os.cpu_count() or 1,
                               "raycast_ms": oracle_sample.raycast_ms}
        # plus a 1-thread figure on config 1 (a subprocess: the thread count is fixed when the OpenMP runtime starts)
        try:
            r = subprocess.run([sys.executable, "-c",
                                "import sys, json; sys.path.insert(0, %r); import bench, synth\n"
                                "nv, t, s = bench.oracle_sample(synth.config(1), 5)\n"
                                "print(json.dumps({'value': nv * len(t) / sum(t), 'ms_per_frame': 1e3 * sum(t) / len(t), 'sample': 'config 1, ' + s}))" % ROOT],
                               env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True, text=True, timeout=120)
            out["cpu_baseline"]["one_thread_cfg1"] = dict(json.loads(r.stdout.strip().splitlines()[-1]), unit=UNIT, cores=1)
        except Exception as e:                                     # reported, never fatal
            out["cpu_baseline"]["one_thread_cfg1"] = {"error": repr(e)[:200]}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
