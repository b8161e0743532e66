#!/usr/bin/env python
"""bench.py — throughput of the D(q,tau) hot path on synthetic stacks shaped like BASELINE.json's configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One "step" = one pass of the whole hot path (frame sums, normalise, 2-D R2C FFT, HBM ring, lag
accumulation, azimuthal binning) over one whole synthetic stack: reset -> nfs_push_frames -> nfs_finalize.
`value` = frames/s with the uint16 stack already resident in HBM; `e2e` = the same through the C-ABI
with the stack in pinned HOST memory (chunked H2D copies overlapped with compute, result D2H), both timed
with CUDA events / synchronised wall clock.  Prints ONE JSON line (rank 0).
Multi-GPU: replicas only: every rank analyses its own stack, no data-path collective.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

SM_COUNT = 148
FP32_LANES_PER_SM = 128
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "lag_traffic.csv")
LAG_SOURCES = ["paper_1209_3362_b200/csrc/nfs_lag.cu", "paper_1209_3362_b200/csrc/nfs_common.cuh"]


def lag_source_sha():
    """SHA-256 (16 hex digits) of the lag kernel's sources: the key under which an ncu traffic figure is valid."""
    import hashlib

    h = hashlib.sha256()
    for f in LAG_SOURCES:
        h.update(open(os.path.join(ROOT, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_lag_traffic(workload, batch, frames):
    """DRAM bytes (read + write) per k_lag_tiled launch from the committed `ncu --set full` capture
    (profiles/lag_traffic.csv: workload,batch,frames,source_sha16,bytes_per_launch,capture).  Returned only if the
    capture was taken from the kernel sources of this tree; otherwise null with the reason."""
    if not os.path.exists(TRAFFIC_CSV):
        return None, "no profiles/lag_traffic.csv"
    sha = lag_source_sha()
    stale = False
    for line in open(TRAFFIC_CSV):
        f = [x.strip() for x in line.split(",")]
        if len(f) < 6 or f[0] == "workload":
            continue
        if (f[0], f[1], f[2]) == (workload, str(batch), str(frames)):
            if f[3] == sha:
                return float(f[4]), "ncu --set full dram__bytes_read.sum + dram__bytes_write.sum per launch, profiles/" + f[5]
            stale = True
    return None, ("the ncu capture in profiles/lag_traffic.csv is of other kernel sources (sha16 now %s)" % sha) if stale else \
        "no ncu capture of this workload"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region: an NVML polling thread (every ~2 ms),
    falling back to an `nvidia-smi -lms` child process where NVML cannot be loaded."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index, uuid=None):
        self.index, self.uuid = index, uuid
        self.sm, self.mx, self.reasons, self.power = [], [], set(), []
        self.proc, self.thread, self.run, self.how = None, None, False, None

    def _nvml_handle(self):
        import pynvml

        pynvml.nvmlInit()
        if self.uuid:
            try:
                return pynvml, pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(self.uuid)).encode())
            except Exception:
                pass
        return pynvml, pynvml.nvmlDeviceGetHandleByIndex(self.index)

    def start(self):
        try:
            nv, h = self._nvml_handle()
            mx = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            bits = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                    "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}

            def poll():
                while self.run:
                    try:
                        self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                        self.mx.append(mx)
                        r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                        for nm, bit in bits.items():
                            if r & bit:
                                self.reasons.add(nm)
                        self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    except Exception:
                        pass
                    time.sleep(0.002)

            self.run, self.how = True, "nvml"
            self.thread = threading.Thread(target=poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.how = "nvidia-smi"
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            try:
                self.sm.append(float(r[0]))
                self.mx.append(float(r[1]))
                self.power.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        self.reasons.add(nm)
            except Exception:
                pass

    def stop(self):
        if self.thread is not None:
            self.run = False
            self.thread.join(timeout=1.0)
        elif self.proc is not None:
            time.sleep(0.05)
            self.proc.terminate()
        else:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no NVML, no nvidia-smi"], samples=0)
        sm, mx = self.sm, self.mx
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_min_mhz=min(sm) if sm else None,
                    sm_max_mhz=max(mx) if mx else None, reasons=sorted(self.reasons), samples=len(sm),
                    power_w_max=max(self.power) if self.power else None, how=self.how)


def workload_counts(cfg):
    P = cfg.H * (cfg.W // 2 + 1)
    pairs = sum(max(0, cfg.N - t) for t in cfg.lags)
    return P, pairs


def lag_algorithmic_work(cfg, binding):
    """FP32 work of the lag accumulation per Fourier pixel and time step (all pairs present), from the lag plan
    (DESIGN.md 7.2): a run of c consecutive lags costs one complex increment (2 lane-instructions, 2 flops), the direct
    update of its smallest lag (2 SUB + 2 FMA = 4 lane-instructions, 6 flops) and one complex FMA per further lag
    (2 lane-instructions, 4 flops); an isolated lag costs the direct update.  -> (lane-instructions, flops)."""
    plan = binding.nfs_plan_lags(cfg.lags, cfg.H * (cfg.W // 2 + 1))
    inst = flop = 0
    for t in plan["tasks"]:
        c = t["cnt"]
        if c == 0:
            continue
        if (t["kind"] & 1) == 0:
            inst += 2 + 4 + 2 * (c - 1)
            flop += 2 + 6 + 4 * (c - 1)
        else:
            inst += 4 * c
            flop += 6 * c
    return inst, flop, plan


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample_frames(cfg):
    """Frames of the bounded oracle sample: about 10-30 s of CPU work on the box's host cores."""
    return min(cfg.N, 128 if cfg.W >= 2048 else (400 if cfg.W >= 1024 else (1000 if cfg.W >= 512 else cfg.N)))


def oracle_sample(cfg, stack_np_fn):
    """The oracle, as it stands, on a bounded sample of the workload -> (frames/s, seconds, description, cores)."""
    from oracle import nfs_oracle as orc

    n_s = oracle_sample_frames(cfg)
    fr = stack_np_fn(n_s)
    t = time.time()
    orc.structure_function(fr, cfg.lags, cfg.n_qbins)
    dt = time.time() - t
    pairs_s = sum(max(0, n_s - t) for t in cfg.lags)
    pairs_full = sum(max(0, cfg.N - t) for t in cfg.lags)
    desc = ("first %d frames of the %dx%d stack, all %d lags, full-plane fp64 oracle (oracle/nfs_oracle.c: it evaluates "
            "both halves of the Hermitian plane, twice the pixels the kernels touch); the sample has %.1f frame pairs per "
            "frame, the full stack %.1f" % (n_s, cfg.W, cfg.H, len(cfg.lags), pairs_s / n_s, pairs_full / cfg.N))
    fft_s, pair_s = orc.last_stage_seconds()
    extra = dict(cpu_model=cpu_model(), fft_stage_seconds=fft_s, pair_stage_seconds=pair_s,
                 frame_pairs_per_s=pairs_s / dt, pixel_pair_updates_per_s=pairs_s * cfg.W * cfg.H / dt)
    return n_s / dt, dt, desc, orc.num_threads(), extra


def run_reference(args, cfg):
    """--impl reference: the CPU oracle on the box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import synth

    gen = synth.SynthStack(cfg, "cpu")
    n_s = oracle_sample_frames(cfg)
    frames = gen.next_frames(n_s).numpy()
    times = []
    desc, cores, extra = "", 0, {}
    for i in range(args.warmup + args.steps):
        v, dt, desc, cores, extra = oracle_sample(cfg, lambda n: frames[:n])
        if i >= args.warmup:
            times.append(dt)
    T = sum(times) / len(times)
    val = n_s / T
    out = dict(metric="frames_per_s", value=val, unit="frames/s", n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
               ms_per_step=T * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
               impl="reference",
               config=dict(workload="%s: %dx%d uint16, %d lags, %d |q| bins (bounded sample: %d of %d frames)" % (
                   cfg.name, cfg.W, cfg.H, len(cfg.lags), cfg.n_qbins, n_s, cfg.N)),
               cpu_baseline=dict(value=val, unit="frames/s", cores=cores, kind="oracle", sample=desc, **extra),
               e2e=dict(value=val, unit="frames/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2: 1024^2 x 2000, 100 lags); "
                    "5 = the workload of the paper's own timing (512^2 x 2048, all 2047 lags, PAPER.md:L39)")
    ap.add_argument("--frames", type=int, default=0, help="override the number of frames (debug)")
    ap.add_argument("--batch", type=int, default=0, help="internal batch size (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-hbm-regime", action="store_true", help="skip the small-batch run of the lag kernel")
    ap.add_argument("--mode", default="path", choices=["path", "bin-only", "banded", "fit"],
                    help="path: the headline line (default).  Secondary measurements of the SURVEY 8(f) rows, one JSON line each, "
                         "single GPU: bin-only (NFS_FLAG_BIN_ONLY against the 2-D mode), banded (out-of-core band schedule "
                         "against the in-memory one; --bands sets alpha), fit (k_fit_eq1 device time)")
    ap.add_argument("--bands", type=int, default=3, help="--mode banded: number of lag bands alpha the ring cap forces")
    ap.add_argument("--sharding", default="replicas", choices=["replicas", "time"],
                    help="N > 1: 'replicas' = every rank analyses its own stack (weak scaling, the default); 'time' = ONE "
                         "stack cut into time chunks with halos, one NCCL all-reduce of the partial sums (strong scaling, "
                         "SURVEY.md 8(e))")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    import synth

    cfg = synth.config(args.config)
    if args.frames:
        cfg.N = args.frames
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.mode != "path":
        return run_mode(args, cfg)
    run_ours(args, cfg)


def run_mode(args, cfg):
    """Secondary measurements: one GPU, stack resident in HBM, CUDA events on the library's
    stream, W warm-up and K timed steps; one JSON line (not the headline line: `metric` names what is measured)."""
    import numpy as np
    import torch
    import synth
    from paper_1209_3362_b200 import binding

    binding.use_dev_library()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(0)
    dev = "cuda:0"
    stack = synth.make_stack(cfg, dev)
    stream = torch.cuda.Stream(device=dev)
    chunk = cfg.chunk or cfg.N

    def timed(nfs, after=None):
        def step():
            nfs.reset()
            for i in range(0, cfg.N, chunk):
                nfs.push(stack[i:i + chunk])
            return nfs.finalize()
        for _ in range(max(args.warmup, 1)):
            out = step()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            out = step()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps, out

    base = dict(n_gpus=1, steps=args.steps, warmup=args.warmup, dtype="f32", data="synthetic",
                config=dict(workload=cfg.name, W=cfg.W, H=cfg.H, frames=cfg.N, n_lags=len(cfg.lags), lag_max=cfg.lags[-1],
                            n_qbins=cfg.n_qbins, inputs="stack resident in HBM, larger than L2"))
    if args.mode == "bin-only":
        full = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=stream, batch_frames=args.batch)
        ms_full, (D_full, I_full, _) = timed(full)
        bytes_full = full.device_bytes
        full.close()
        bo = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=stream, batch_frames=args.batch, bin_only=True)
        ms_bo, (D_bo, I_bo, cnt) = timed(bo)
        bytes_bo = bo.device_bytes
        bo.close()
        nz = cnt > 0
        out = dict(base, metric="ms per stack, NFS_FLAG_BIN_ONLY (PAPER.md:L41)", value=ms_bo, unit="ms", higher_is_better=False,
                   two_d_mode_ms=ms_full, slowdown_vs_2d=ms_bo / ms_full, device_bytes=bytes_bo, device_bytes_2d=bytes_full,
                   max_rel_diff_binned_D_vs_2d=float(np.max(np.abs(D_bo[:, nz] - D_full[:, nz]) / D_full[:, nz])))
    elif args.mode == "banded":
        alpha = max(2, args.bands)
        b = args.batch or 128
        nstar = (cfg.lags[-1] + alpha - 1) // alpha
        cap = nstar + 2 * b
        mem = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=stream, batch_frames=b)
        ms_mem, (D_mem, _, cnt) = timed(mem)
        mem.close()
        bd = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=stream, batch_frames=b, ring_frames_cap=cap, max_frames=cfg.N)
        ms_bd, (D_bd, _, _) = timed(bd)
        tc = bd.transfer_counts()   # of the last step (reset clears them)
        ring = bd.ring_capacity
        bd.close()
        plan = binding.nfs_band_plan(cfg.N, cfg.lags, cap, b)
        a = tc["bands"]
        nz = cnt > 0
        out = dict(base, metric="ms per stack, out-of-core band schedule (PAPER.md:L33, Fig. 2(b))", value=ms_bd, unit="ms",
                   higher_is_better=False, in_memory_ms=ms_mem, slowdown_vs_in_memory=ms_bd / ms_mem, bands=a,
                   band_width=tc["band_width"], batch=b, ring_frames_cap=cap, ring_frames=ring,
                   fourier_frames_uploaded=tc["h2d_frames"], fourier_frames_downloaded=tc["d2h_frames"],
                   band_plan_uploads=plan["old_uploads"] + plan["new_uploads"],
                   paper_N_FFT=cfg.N * (2 * a - 3 + 2.0 / a),
                   max_rel_diff_binned_D_vs_in_memory=float(np.max(np.abs(D_bd[:, nz] - D_mem[:, nz]) / D_mem[:, nz])))
    else:  # fit
        nfs = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=stream, batch_frames=args.batch)
        for i in range(0, cfg.N, chunk):
            nfs.push(stack[i:i + chunk])
        nfs.finalize()
        nfs.set_profiling(True)
        for _ in range(max(args.warmup, 1)):
            nfs.fit_eq1(), nfs.variance()
        nfs.kernel_times()
        for _ in range(args.steps):
            nfs.variance()               # k_bin alone
        ms_bin = nfs.kernel_times()["bin"][0] / args.steps
        t0 = time.time()
        for _ in range(args.steps):
            A, Cq, G, chi2 = nfs.fit_eq1()  # k_bin + k_fit_eq1
        call_ms = (time.time() - t0) / args.steps * 1e3
        ms_both = nfs.kernel_times()["bin"][0] / args.steps
        nfs.close()
        out = dict(base, metric="k_fit_eq1 device time (PAPER.md:L23-25, Eq. 1; per-|q| fit of A, C, Gamma)", value=(ms_both - ms_bin) * 1e3,
                   unit="us", higher_is_better=False, k_bin_us=ms_bin * 1e3, nfs_fit_eq1_call_ms=call_ms,
                   bins_fitted=int((G > 0).sum()))
    print(json.dumps(out), flush=True)


def run_ours(args, cfg):
    import torch
    import synth
    from paper_1209_3362_b200 import binding

    binding.use_dev_library()  # per-kernel timing, launch counts, the traffic probe: include/nfs_dev.h (same kernels)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --impl ours needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    peaks = load_peaks()
    P, pairs = workload_counts(cfg)
    updates = pairs * P

    from paper_1209_3362_b200 import replicas

    from paper_1209_3362_b200 import sharding

    time_sharded = args.sharding == "time"
    # replicas: every rank analyses its own stack (seed differs per rank); time sharding: the same stack everywhere,
    # each rank feeds its context the halo and the own frames of its time chunk
    stack = synth.make_stack(cfg if time_sharded else replicas.rank_config(cfg, rank), dev)
    stream = torch.cuda.Stream(device=dev)
    nfs = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=stream, batch_frames=args.batch)
    torch.cuda.synchronize()
    shard = sharding.shard_plan(cfg.N, world, cfg.lags[-1])[rank] if time_sharded else None
    merge_bytes = 0

    def step():
        nonlocal merge_bytes
        nfs.reset()
        if time_sharded:
            sharding.push_shard(nfs, stack, shard)
            merge_bytes = sharding.merge(nfs, dist)   # the path's one collective: all-reduce of the fp64 partial sums
        else:
            nfs.push(stack)
        return nfs.finalize()

    for _ in range(max(args.warmup, 1) if args.warmup else 0):
        step()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local, getattr(torch.cuda.get_device_properties(local), "uuid", None))
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall = time.time()
    e0.record(stream)
    n_launch = 0
    for _ in range(args.steps):
        step()
        n_launch += nfs.num_launches
    e1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t_wall = time.time() - t_wall
    clocks = sampler.stop() if rank == 0 else None
    ms_total = replicas.max_over_ranks(e0.elapsed_time(e1), dist, dev)
    ms_step = ms_total / args.steps
    # per-kernel durations: the same K steps once more with a CUDA event pair around every launch on the library's
    # stream (kept out of the headline region: the event records cost a little host and device time)
    nfs.set_profiling(True)
    nfs.kernel_times()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record(stream)
    for _ in range(args.steps):
        step()
    e3.record(stream)
    torch.cuda.synchronize()
    ktimes = nfs.kernel_times()
    nfs.set_profiling(False)
    ms_step_profiled = e2.elapsed_time(e3) / args.steps
    value = (1 if time_sharded else world) * cfg.N / (ms_step * 1e-3)   # time sharding: ONE stack over all ranks

    # ---- end to end through the C-ABI with the stack in pinned HOST memory ----
    e2e = None
    if not args.no_e2e and not time_sharded:
        e2e = run_e2e(torch, nfs, stack, cfg, stream, dev, args, dist, world)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (lag accumulation, k_lag_tiled) ----
    # Algorithmic work per launch: FP32 lane-instructions of the neighbouring-lag recurrence for the
    # lag plan of this workload x the frame pairs x pixels one launch processes; the kernel's average launch duration
    # comes from CUDA events recorded around every launch on the library's stream (nfs_set_profiling).
    lag_ms, lag_n = ktimes["lag_accum"]
    lag_s_per_launch = lag_ms * 1e-3 / max(lag_n, 1)
    upd_per_launch = updates / (world if time_sharded else 1) * args.steps / max(lag_n, 1)   # this rank's share
    inst_step, flop_step, plan = lag_algorithmic_work(cfg, binding)
    n_l = len(cfg.lags)
    inst_per_update, flop_per_update = inst_step / n_l, flop_step / n_l   # averaged over the lags of the plan
    lane_rate_peak = SM_COUNT * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6
    peak_tflops = lane_rate_peak * (flop_per_update / inst_per_update) / 1e12
    ach_tflops = upd_per_launch * flop_per_update / lag_s_per_launch / 1e12
    B = nfs.ring_capacity - cfg.lags[-1]  # the library's internal batch (frames)
    nb = (cfg.N + B - 1) // B
    # algorithmic HBM bytes of the accumulation: 8*U/B + 16*n_l/B per pixel and new frame
    lag_bytes = P * (8.0 * (cfg.N + nb * cfg.lags[-1]) + 16.0 * len(cfg.lags) * nb)
    traffic, traffic_source = ncu_lag_traffic(cfg.name, B, cfg.N)
    roofline = dict(bound="alu", kernel="k_lag_tiled", achieved=ach_tflops, peak=peak_tflops, unit="TFLOP/s",
                    frac=ach_tflops / peak_tflops, traffic=traffic, traffic_source=traffic_source,
                    peak_source="derived (DESIGN.md §7.2): 148 SM x 128 FP32 lanes x %.0f MHz (clocks.max.sm, %s) = %.3g "
                                "lane-instructions/s x %.3f flop per lane-instruction of this lag plan (%.2f lane-instructions, "
                                "%.2f flops per pair update: one direct update per run of lags, one complex FMA per further lag)"
                                % (peaks["sm_max_mhz"], peaks["source"], lane_rate_peak, flop_per_update / inst_per_update,
                                   inst_per_update, flop_per_update),
                    lane_instructions_per_pair_update=inst_per_update, flops_per_pair_update=flop_per_update,
                    direct_form=dict(note="the plain per-pair form |F_s - F_{s-tau}|^2 (4 lane-instructions, 6 flops per pair "
                                          "update, round 1's kernel) would need this fraction of the same peak",
                                     frac=upd_per_launch * 4.0 / lag_s_per_launch / lane_rate_peak),
                    pair_updates_per_s=upd_per_launch / lag_s_per_launch, ms_per_launch=lag_s_per_launch * 1e3,
                    ms_per_step=lag_ms / args.steps, launches_per_step=lag_n / args.steps,
                    tile_px=plan["tile_px"], task_slots=plan["slots"], lag_groups=len(plan["groups"]),
                    hbm=dict(algorithmic_gb_per_step=lag_bytes / 1e9, achieved_gbs=lag_bytes / (lag_ms * 1e-3 / args.steps) / 1e9,
                             peak_gbs=peaks["hbm_gbs"], frac=lag_bytes / (lag_ms * 1e-3 / args.steps) / 1e9 / peaks["hbm_gbs"],
                             note="of measured copy peak; HBM is not the binding roofline for dense lags (DESIGN.md §7.2)"))
    if world == 1 and not args.no_hbm_regime and not args.batch:
        roofline["hbm_bound_regime"] = run_hbm_regime(torch, binding, stack, cfg, P, peaks, inst_per_update)
    fft_ms = ktimes["fft"][0]
    fft_bytes = (2.0 * cfg.W * cfg.H + 24.0 * P) * cfg.N      # one round trip between the passes
    fft_bytes_min = (2.0 * cfg.W * cfg.H + 8.0 * P) * cfg.N   # intermediate kept in L2 (what k_fft does)
    fft_s = fft_ms / args.steps * 1e-3
    fft = dict(bound="hbm", kernel="k_fft", ms_per_step=fft_ms / args.steps, algorithmic_gb_per_step=fft_bytes_min / 1e9,
               achieved_gbs=fft_bytes_min / fft_s / 1e9, peak_gbs=peaks["hbm_gbs"], frac=fft_bytes_min / fft_s / 1e9 / peaks["hbm_gbs"],
               bytes_note="2WH + 8P bytes per frame: the uint16 frame in, the Fourier frame out; the row-pass intermediate "
                          "stays in L2",
               round_trip_gb_per_step=fft_bytes / 1e9, round_trip_frac=fft_bytes / fft_s / 1e9 / peaks["hbm_gbs"],
               round_trip_note="SURVEY.md 8(d)'s figure with one HBM round trip between the passes (2WH + 24P)",
               us_per_frame=fft_s / cfg.N * 1e6)
    kernels = {k: dict(ms_per_step=v[0] / args.steps, launches_per_step=v[1] / args.steps) for k, v in ktimes.items()
               if k != "unused"}

    # BASELINE.md holds a paper number only for the paper's own workload (512^2 x 2048, all lags): total time
    # "< 2 min" on a Tesla C2050, i.e. > 17.07 frames/s (another machine's: context, not the target)
    vs_baseline = value / (2048.0 / 120.0) if (cfg.name == "paper-fig3" and world == 1) else None
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, dt, desc, cores, extra = oracle_sample(cfg, lambda n: stack[:n].cpu().numpy())
        cpu = dict(value=v, unit="frames/s", cores=cores, kind="oracle", sample=desc, seconds=dt, **extra)

    out = dict(metric="frames_per_s", value=value, unit="frames/s", n_gpus=world, steps=args.steps, warmup=args.warmup,
               ms_per_step=ms_step, higher_is_better=True, scaling="strong" if time_sharded else "weak", vs_baseline=vs_baseline,
               dtype="f32", data="synthetic",
               config=dict(workload="%s: %dx%d uint16 x %d frames, %d lags (max %d), %d |q| bins" % (
                   cfg.name, cfg.W, cfg.H, cfg.N, len(cfg.lags), cfg.lags[-1], cfg.n_qbins),
                   parallelism=("time chunks x%d, halo %d frames, one all-reduce of %.1f MB" % (world, cfg.lags[-1], merge_bytes / 1e6))
                   if time_sharded else "replicas x%d" % world, internal_batch=B,
                   l2_policy="inputs larger than L2 (%.2f GB stack streamed from HBM every step)" % (stack.numel() * 2 / 1e9)),
               frame_pairs_per_s=(1 if time_sharded else world) * pairs / (ms_step * 1e-3),
               pair_updates_per_s=(1 if time_sharded else world) * updates / (ms_step * 1e-3),
               wall_s_per_step=t_wall / args.steps, ms_per_step_with_kernel_events=ms_step_profiled, gpu_launches=n_launch,
               clocks=clocks, e2e=e2e, roofline=roofline,
               fft=fft, kernels=kernels, cpu_baseline=cpu)
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_hbm_regime(torch, binding, stack, cfg, P, peaks, inst_per_update):
    """The same lag kernel where HBM is its binding roofline (BASELINE.json metric: "lag-accumulation HBM GB/s"):
    batches of one 26-step chunk, so that every launch re-reads the whole lag window and touches the fp64 totals
    once per 26 frames.  Algorithmic bytes per launch = P (8 (b + Lmax) + 16 n_lags); time = CUDA
    events around every k_lag_tiled launch on the library's stream, one warm-up stack then two timed."""
    B = 26
    st = torch.cuda.Stream(device=stack.device)
    h = binding.NFS(cfg.W, cfg.H, cfg.lags, cfg.n_qbins, stream=st, batch_frames=B)
    h.set_profiling(True)
    steps = 2
    for i in range(1 + steps):
        h.reset()
        h.push(stack)
        h.finalize()
        if i == 0:
            h.kernel_times()
    ms, n = h.kernel_times()["lag_accum"]
    probe_ms, probe_bytes = h.probe_lag_traffic(B, 20)
    h.close()
    nb = (cfg.N + B - 1) // B
    alg = P * (8.0 * (cfg.N + nb * cfg.lags[-1]) + 16.0 * len(cfg.lags) * nb)  # bytes per stack
    ach = alg / (ms / steps * 1e-3) / 1e9
    return dict(internal_batch=B, launches_per_step=n / steps, ms_per_step=ms / steps, algorithmic_gb_per_step=alg / 1e9,
                achieved_gbs=ach, peak_gbs=peaks["hbm_gbs"], frac=ach / peaks["hbm_gbs"],
                alu_floor_ms=(sum(max(0, cfg.N - t) for t in cfg.lags) * P * inst_per_update) / (SM_COUNT * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6) * 1e3,
                note="same kernel and stack, batches of 26 frames: algorithmic HBM time exceeds the ALU floor, HBM is the bound",
                access_pattern_probe=dict(ms_per_launch=probe_ms, algorithmic_gb_per_launch=probe_bytes / 1e9,
                                          achieved_gbs=probe_bytes / (probe_ms * 1e-3) / 1e9,
                                          frac_of_copy_peak=probe_bytes / (probe_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                          kernel_ms_per_launch=ms / max(n, 1),
                                          note="nfs_probe_lag_traffic: the same TMA box copies and fp64 reductions per launch, no "
                                               "arithmetic — what this access pattern reaches on this device"))


def run_e2e(torch, nfs, stack, cfg, stream, dev, args, dist, world):
    """Stack in pinned host memory; chunks of `chunk` frames go through a ring of device staging buffers on a
    copy stream (enough of them to keep copying while a lag kernel of a whole batch runs: a staging buffer is
    free again only when the work enqueued by its push has finished), are pushed through the C-ABI, and the
    result is read back by nfs_finalize."""
    chunk = cfg.chunk or 256
    chunk = min(chunk, cfg.N)
    host = torch.empty(stack.shape, dtype=torch.uint16, pin_memory=True)
    host.copy_(stack)
    torch.cuda.synchronize()
    n_stage = max(2, min(6, (cfg.N + chunk - 1) // chunk))
    stage = [torch.empty((chunk, cfg.H, cfg.W), dtype=torch.uint16, device=dev) for _ in range(n_stage)]
    copy_stream = torch.cuda.Stream(device=dev)
    copied = [torch.cuda.Event() for _ in range(n_stage)]
    consumed = [torch.cuda.Event() for _ in range(n_stage)]

    def step():
        nfs.reset()
        i, k = 0, 0
        while i < cfg.N:
            m = min(chunk, cfg.N - i)
            b = k % n_stage
            with torch.cuda.stream(copy_stream):
                if k >= n_stage:
                    copy_stream.wait_event(consumed[b])
                stage[b][:m].copy_(host[i:i + m], non_blocking=True)
                copied[b].record(copy_stream)
            stream.wait_event(copied[b])
            nfs.push_ptr(stage[b].data_ptr(), m)
            consumed[b].record(stream)
            i += m
            k += 1
        return nfs.finalize()

    step()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    steps = max(1, args.steps)  # the same number of steps as the device-timed headline
    t = time.time()
    for _ in range(steps):
        D, I, cnt = step()
    torch.cuda.synchronize()
    dt = (time.time() - t) / steps
    from paper_1209_3362_b200 import replicas

    dt = replicas.max_over_ranks(dt, dist, dev)
    del host
    return dict(value=world * cfg.N / dt, unit="frames/s", h2d_bytes_per_step=int(stack.numel() * 2),
                d2h_bytes_per_step=int(D.nbytes + I.nbytes + 4), ms_per_step=dt * 1e3, chunk_frames=chunk,
                staging_buffers=n_stage,
                note="pinned host stack -> ring of device staging buffers (copy stream) -> nfs_push_frames -> nfs_finalize")


if __name__ == "__main__":
    main()
