#!/usr/bin/env python
"""bench.py -- headline benchmark of libtnlm on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Metric (BASELINE.json): TNLM Gauss-Jacobi pixel-updates/s (px x phase x iter).  Workload at
N=1: BASELINE.json configs[1] ("TNLM step alone": 256x256 fp32 x 10 cyclic phases, window 11,
patch 5, h=0.008, mu=0.1, 10 Gauss-Jacobi sweeps, seed 1).  One step = one
tnlm_regularize_step call (weights + 10 sweeps + clip) on one slice per GPU, as the library ships it:
10 launches of gj_sweep_kernel<.,.,false>, every one computing the weights of g in fp32 (ALU bound).
The opt-in stored-weight path (option weight_cache_mb > 0: 1 launch of gj_sweep_kernel<.,.,true> that also
stores the weights as bf16, then 9 launches of gj_apply3_kernel streaming them, HBM bound) is timed beside it
and reported under "value_stored_bf16"; it is not the headline because it can miss the 1e-4 bar (tnlm.h).

--gpus N > 1: when not already under torchrun, bench.py re-executes itself under
`python -m torch.distributed.run --nproc-per-node N` (one rank per GPU, NCCL for the barrier and
the max-over-ranks of the timings only).  Every rank runs its own slice(s): slices are
independent, no collective on the data path, weak scaling for the headline;
the 64-slice batch of configs[4] ("recon_batch") is sharded by paper_1009_1351_b200.sharding.

Timed region: K steps, each bracketed by CUDA events on the launching stream; L2 is flushed
(a 256 MiB device buffer is rewritten) between steps, outside the event brackets; a barrier and
torch.cuda.synchronize() on both sides; the max over ranks is taken.  The second half of the
metric ("s per 10-phase slice recon") is reported under "recon" (configs[3]), "recon_low_mas"
(configs[2]), "recon_tiny" (configs[0]) and "recon_batch" (configs[4], 64 slices).

--impl reference times the CPU oracle (oracle/, plain C fp64) on the host cores, on a bounded
sample of the same workload.  Only that leg and the `cpu_baseline*` legs touch oracle/.
"""
import argparse
import json
import os
import socket
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "TNLM Gauss-Jacobi pixel-updates/s (px x phase x iter)"
UNIT = "px-updates/s"
FP32_LANES_PER_SM = 128          # CUDA cores per SM (sm_100)
N_SM = 148
DTYPE = "f32"


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ---- algorithmic work per unit -----------------------
def flops_per_px_update(window, patch):
    """One Gauss-Jacobi pixel update with the weights computed on the fly, separable box-sum form:
    2 neighbours x W^2 offsets x (2d+4) flops."""
    return 2 * window * window * (2 * patch + 4)


def flops_per_px_update_symmetric(window, patch):
    """The same with the pair distance shared by the two directions: (2d+1)/2 + 3 per
    directed evaluation.  Reported beside the unsymmetric count so the fraction is not padded."""
    return 2 * window * window * ((2 * patch + 1) / 2.0 + 3)


def bytes_per_px_update_stored(window):
    """One Gauss-Jacobi pixel update from stored weights: 2 neighbours x W^2 bf16 weights + g, u read
    and u' written once (3 x 4 bytes)."""
    return 2 * window * window * 2 + 12


def kernel_source_sha256():
    """Hash of the TNLM kernel source the stored ncu traffic figures (profiles/traffic.json) belong to."""
    import hashlib
    with open(os.path.join(ROOT, "paper_1009_1351_b200", "csrc", "regularize.cuh"), "rb") as f:
        return hashlib.sha256(f.read()).hexdigest()


def projector_work(cfg, n_slices):
    """Algorithmic work of ONE application of P or P^T to n_slices slices:
    forward ~10 flop per ray segment, 1.3 L segments per ray; gather backprojection ~76 flop per
    pixel-view; bytes = image + sinogram once (4 L^2 + 4 V B per phase).  The slices of a batch share the
    geometry, so the library evaluates the ray walk (6 of the 10 flops of a segment) once per group of 4 slices
    and the candidate geometry (66 of the 76 flops of a pixel-view) once per group of 16: the *_shared counts are
    the flops that formulation needs, reported beside the per-slice counts so that no fraction is padded."""
    n = n_slices * cfg.N
    gf = 4 if n_slices >= 4 else 1          # slices per forward group (project_il_kernel)
    gb = 16 if n_slices >= 16 else (8 if n_slices >= 8 else (4 if n_slices >= 4 else (2 if n_slices >= 2 else 1)))
    return {"project_flops": n * cfg.V * cfg.B * 1.3 * cfg.L * 10.0,
            "project_flops_shared": n * cfg.V * cfg.B * 1.3 * cfg.L * (6.0 / gf + 4.0),
            "backproject_flops": n * cfg.L * cfg.L * cfg.V * 76.0,
            "backproject_flops_shared": n * cfg.L * cfg.L * cfg.V * (66.0 / gb + 10.0),
            "bytes": n * 4.0 * (cfg.L * cfg.L + cfg.V * cfg.B)}


class ClockSampler:
    """Samples SM clock and throttle reasons (NVML) in a thread while the timed region runs."""

    def __init__(self, torch_device_index, period=0.002):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.period = period
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(torch_device_index).uuid)
                self.dev = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.dev = pynvml.nvmlDeviceGetHandleByIndex(torch_device_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)))
                bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev))
                for k, b in names.items():
                    if bits & b:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def cfg2_input(seed):
    cfg = workloads.config(2, seed=seed)
    return cfg, workloads.make_inputs(cfg)["g"].astype(np.float32)          # [1][N][L][L]


# ----------------------------------------------------------------------------------- reference arm
def time_oracle(cfg, g, budget_s):
    """The oracle as it stands on the host cores: whole Gauss-Jacobi sweeps of the workload
    (naive O(W^2 d^2) fp64 loop, weights recomputed per sweep, as oracle_regularize_step does)
    until ~budget_s is spent."""
    import oracle
    n_px = g[0].size
    t0 = time.perf_counter()
    sweeps = 0
    while True:
        oracle.regularize_step(g[0], cfg.window, cfg.patch, cfg.h, cfg.mu, 1)
        sweeps += 1
        dt = time.perf_counter() - t0
        if dt >= budget_s or sweeps >= cfg.m2:
            break
    return sweeps * n_px / dt, sweeps, dt, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, g = cfg2_input(1)
    for _ in range(min(args.warmup, 1)):
        time_oracle(cfg, g, 0.0)
    vals, secs, sweeps_tot, cores = [], 0.0, 0, 1
    per_step_budget = max(1.0, min(10.0, 60.0 / max(args.steps, 1)))
    for _ in range(args.steps):
        v, sweeps, dt, cores = time_oracle(cfg, g, per_step_budget)
        vals.append(v); secs += dt; sweeps_tot += sweeps
    value = sweeps_tot * g[0].size / secs
    sample = (f"{sweeps_tot} whole Gauss-Jacobi sweeps (naive fp64 weights + update, recomputed every sweep) "
              f"of cfg2 256x256x10 in {secs:.1f} s")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(cfg, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(cfg, n_gpus):
    return {"workload": "BASELINE.json configs[1]: TNLM step alone", "image": f"{cfg.L}x{cfg.L}",
            "n_phase": cfg.N, "window": cfg.window, "patch": cfg.patch, "h": cfg.h, "mu": cfg.mu,
            "gauss_jacobi_sweeps": cfg.m2, "slices_per_gpu": 1, "seed": cfg.seed,
            "parallelism": f"slice-sharded x{n_gpus}, no collective",
            "l2": "flushed between timed steps (256 MiB rewrite outside the event brackets)"}


# ------------------------------------------------------------------------------- multi-GPU plumbing
def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` (N > 1) outside torchrun: start N ranks, one per GPU."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this node has {have}")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def sharded_batch(n_slices, world, rank, dist, run_local, device="cpu"):
    """The N>1 path of the 64-slice batch: contiguous slice ranges per rank
    (sharding.slice_range), every rank runs `run_local(slices) -> (per-slice result tensor, device
    seconds)` on its own share with no exchange, the time is the max over ranks and the per-slice
    results are gathered once at the end in slice order.  tests/test_sharding_gloo.py runs exactly this
    function on world_size-2 gloo with a CPU stand-in for the library call."""
    from paper_1009_1351_b200.sharding import gather_slices, max_over_ranks, slice_range
    mine = slice_range(n_slices, world, rank)
    local, seconds = run_local(mine)
    seconds = max_over_ranks(seconds, dist if world > 1 else None, device)
    full = gather_slices(local, n_slices, dist if world > 1 else None)
    return full, seconds, mine


# ---------------------------------------------------------------------------------------- our arm
def kernel_table(tn, h, steps_done, step_us):
    """{kind: (launches per step, mean us per launch)} from the library's event pairs."""
    acc = {}
    for kind, kms in tn.kernel_times(h):
        acc.setdefault(kind, []).append(kms)
    return {k: (len(v) / steps_done, 1e3 * float(np.mean(v))) for k, v in acc.items()}


def run_ours(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch one rank per GPU")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libtnlm has no CPU fallback")
    if local >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: LOCAL_RANK {local} but only {torch.cuda.device_count()} CUDA devices")
    if local == 0:
        from paper_1009_1351_b200 import build
        build.build()                # no-op when libtnlm.so is newer than its sources
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()                                        # (local rank 0 may just have built the library)
    import paper_1009_1351_b200 as tn
    from paper_1009_1351_b200.sharding import max_over_ranks
    cfg, g_np = cfg2_input(1 + rank)                 # one independent slice per rank
    n_px_step = g_np.size * cfg.m2                   # pixel updates of one step on this rank
    h = tn.create(None, cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch, cfg.h, cfg.mu)
    tn.reserve(h, 1, 0, cfg.m2, True)
    g = torch.from_numpy(g_np).cuda()
    f = torch.empty_like(g)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        tn.regularize_step(h, g, cfg.m2, f, stream)

    def timed_steps(n):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        barrier()
        for a, b in ev:
            flush.fill_(1)
            a.record(stream); step(); b.record(stream)
        barrier()
        return sum(a.elapsed_time(b) for a, b in ev)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        flush.fill_(1); step()
    barrier()
    n0 = h.launch_count
    with ClockSampler(torch.cuda.current_device()) as cs:
        ms = timed_steps(args.steps)
    launches = h.launch_count - n0
    ms_total = max_over_ranks(ms, dist, "cuda")
    ms_per_step = ms_total / args.steps
    value = world * n_px_step / (ms_per_step * 1e-3)

    # ---- the same call with the opt-in stored weights (sweeps 2..10 stream bf16 weights instead of computing them)
    tn.set_option(h, "weight_cache_mb", 16384)
    tn.reserve(h, 1, 0, cfg.m2, True)
    for _ in range(3):
        flush.fill_(1); step()
    n_st = max(3, min(args.steps, 20))
    ms_st = max_over_ranks(timed_steps(n_st), dist, "cuda") / n_st
    tn.profile_kernels(h, True)
    for _ in range(3):
        flush.fill_(1); step()
    kern_st = kernel_table(tn, h, 3, ms_st * 1e3)
    tn.profile_kernels(h, False)
    tn.set_option(h, "weight_cache_mb", 0)
    value_st = world * n_px_step / (ms_st * 1e-3)

    # ---- per-kernel durations: the same K steps again with the library's event pair around every
    # launch (CUDA events on the launching stream; a separately instrumented pass, kept out of the
    # headline region above, so the shares can sum to slightly more than 1)
    step(); torch.cuda.synchronize()
    tn.profile_kernels(h, True)
    for _ in range(args.steps):
        flush.fill_(1); step()
    kern = kernel_table(tn, h, args.steps, ms_per_step * 1e3)
    tn.profile_kernels(h, False)
    torch.cuda.synchronize()

    # ---- end to end: host buffers through the C ABI, copies inside the timed region
    gh = torch.from_numpy(g_np).pin_memory()
    fh = torch.empty_like(gh).pin_memory()
    for _ in range(3):
        tn.regularize_step_host(h, gh, cfg.m2, fh, stream)
    barrier()
    n_e2e = max(3, min(args.steps, 50))
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        tn.regularize_step_host(h, gh, cfg.m2, fh, stream)      # synchronises the stream itself
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
    e2e_value = world * n_px_step * n_e2e / e2e_s
    checksum = float(fh.double().sum().item())

    peaks, peak_src = measured_peaks()
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    peak_tf_derived = N_SM * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12
    peak_tf = tn.fma_peak(stream)               # FFMA-chain probe of the library, same run, same box
    ctx = {"tn": tn, "torch": torch, "dist": dist, "world": world, "rank": rank, "args": args,
           "peak_tf": peak_tf, "hbm_gbs": hbm_gbs, "barrier": barrier}

    # ---- the 64-slice batch (configs[4]) sharded over the ranks: every rank takes part
    batch = None if args.no_batch else time_recon_batch(ctx)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    n_px = g_np.size
    traffic = {}
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_file):
        try:
            traffic = json.load(open(traffic_file))
        except Exception:
            traffic = {}
    # the stored ncu figures describe the kernels of regularize.cuh as they were when captured: stale once it changes
    traffic_stale = traffic.get("kernel_source_sha256") != kernel_source_sha256()
    names = {"sweep": "gj_sweep_kernel<PB,RB,false> (weights on the fly + sweep)",
             "sweep_store": "gj_sweep_kernel<PB,RB,true> (weights on the fly + sweep, stores bf16 weights)",
             "apply": "gj_apply3_kernel (sweep from stored bf16 weights: one CTA per band, per-warp cp.async rings)"}

    def tnlm_entry(kind, per_step, us, step_us_):
        k = {"kernel": names[kind], "launches_per_step": per_step, "us_per_launch": us,
             "share_of_step": per_step * us / step_us_}
        if kind == "apply":
            gbs = bytes_per_px_update_stored(cfg.window) * n_px / (us * 1e-6) / 1e9
            k.update({"bound": "hbm", "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs,
                      "traffic": traffic.get("gj_apply_cfg2_dram_bytes_per_launch"),
                      "algorithmic_bytes_per_px_update": bytes_per_px_update_stored(cfg.window)})
        else:
            fl, fls = flops_per_px_update(cfg.window, cfg.patch), flops_per_px_update_symmetric(cfg.window, cfg.patch)
            tf = fl * n_px / (us * 1e-6) / 1e12
            k.update({"bound": "alu", "achieved": tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": tf / peak_tf,
                      "frac_symmetric_flop_count": tf * fls / fl / peak_tf,
                      "traffic": traffic.get("gj_%s_cfg2_dram_bytes_per_launch" % kind),
                      "algorithmic_flops_per_px_update": fl})
        return k

    step_us = ms_per_step * 1e3
    kernels = [tnlm_entry(kind, per_step, us, step_us) for kind, (per_step, us) in sorted(kern.items())]
    dominant = max(kernels, key=lambda k: k["share_of_step"]) if kernels else {}
    roofline = {key: dominant.get(key) for key in ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic",
                                                   "us_per_launch", "launches_per_step", "share_of_step")}
    roofline["traffic_source"] = traffic.get("source", "none: no ncu capture recorded in profiles/traffic.json")
    roofline["traffic_stale"] = bool(traffic_stale)
    # SURVEY.md section 8(d)'s own accounting of the whole step, whatever the kernels do inside: 2 W^2 (2d+4) flops
    # and 12 bytes (g, u read, u' written) per pixel update
    survey_flops = flops_per_px_update(cfg.window, cfg.patch)
    survey_bytes_launch = 12.0 * n_px
    roofline["survey_flops_per_px_update"] = survey_flops
    roofline["step_tflops"] = survey_flops * n_px_step / (ms_per_step * 1e-3) / 1e12
    roofline["step_frac_of_fp32_peak"] = roofline["step_tflops"] / peak_tf
    roofline["survey_bytes_per_launch"] = survey_bytes_launch
    roofline["traffic_over_survey_bytes"] = (dominant["traffic"] / survey_bytes_launch) if dominant.get("traffic") else None
    roofline["peak_source"] = (
        f"{peak_src} MEASURED_PEAKS.json hbm_gbs (burst copy figure)" if dominant.get("bound") == "hbm" else
        "measured in this run by tnlm_fma_peak (8-chain FFMA kernel)")
    roofline["share_note"] = ("us_per_launch and share_of_step come from a separately instrumented pass (an event pair "
                              "around every launch), so the shares can sum to slightly more than 1")
    roofline["kernels"] = kernels
    roofline["fp32_peak_tflops_measured"] = peak_tf
    roofline["fp32_peak_tflops_derived"] = peak_tf_derived

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warm, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
            "config": workload_config(cfg, world), "clocks": cs.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(g_np.nbytes),
                    "d2h_bytes_per_step": int(g_np.nbytes), "calls": n_e2e, "checksum": checksum},
            "gpu_launches": int(launches), "roofline": roofline,
            "value_stored_bf16": {"value": value_st, "unit": UNIT, "ms_per_step": ms_st,
                                  "step_frac_of_fp32_peak": survey_flops * n_px_step / (ms_st * 1e-3) / 1e12 / peak_tf,
                                  "what": "NOT the default: the same call with option weight_cache_mb = 16384, i.e. sweep 1 "
                                          "also stores the weights as bf16 and sweeps 2..10 stream them (fp32 accumulation); "
                                          "2e-6 vs the oracle on this workload, but up to 2e-4 on binary high-contrast "
                                          "images with mu >= 2 (include/tnlm.h), so it is opt-in",
                                  "kernels": [tnlm_entry(kind, per_step, us, ms_st * 1e3)
                                              for kind, (per_step, us) in sorted(kern_st.items())]}}

    if batch is not None:
        line["recon_batch"] = batch
    if world == 1 and not args.no_recon:
        line["recon"] = time_recon(ctx, 4)
        if "fbp_start" in line["recon"]:
            line["recon_fbp_start"] = line["recon"].pop("fbp_start")
        line["recon_low_mas"] = time_recon(ctx, 3)
        line["recon_tiny"] = time_recon(ctx, 1)
    if world == 1 and not args.no_cpu:
        v, sweeps, dt, cores = time_oracle(cfg, g_np.astype(np.float64), args.cpu_budget)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{sweeps} whole Gauss-Jacobi sweep(s) of the same cfg2 slice "
                                          f"(of {cfg.m2}) in {dt:.1f} s; the oracle is the naive fp64 O(W^2 d^2) "
                                          f"loop and computes the weights in every sweep, as the timed GPU path does"}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def recon_kernel_entries(cfg, n_slices, table, total_us, peak_tf, hbm_gbs):
    """roofline.kernels[] of a reconstruction: per kernel kind, launches and us per outer iteration, the
    algorithmic flop rate against the measured FP32 peak and the algorithmic byte rate against HBM."""
    work = projector_work(cfg, n_slices)
    n_img = n_slices * cfg.N * cfg.L * cfg.L
    n_sino = n_slices * cfg.N * cfg.V * cfg.B
    out = []
    for kind, (per_it, us) in sorted(table.items()):
        e = {"kernel": kind, "launches_per_outer_iteration": per_it, "us_per_launch": us,
             "share_of_outer_iteration": per_it * us / total_us}
        sec = us * 1e-6
        if kind == "project":
            e.update({"bound": "l1tex (gathers)" if n_slices >= 4 else "alu", "algorithmic_tflops": work["project_flops_shared"] / sec / 1e12,
                      "algorithmic_tflops_per_slice_geometry": work["project_flops"] / sec / 1e12,
                      "algorithmic_gbs": work["bytes"] / sec / 1e9})
        elif kind == "backproject":
            e.update({"bound": "alu", "algorithmic_tflops": work["backproject_flops_shared"] / sec / 1e12,
                      "algorithmic_tflops_per_slice_geometry": work["backproject_flops"] / sec / 1e12,
                      "algorithmic_gbs": work["bytes"] / sec / 1e9})
        elif kind in ("sweep", "sweep_store"):
            fl = flops_per_px_update(cfg.window, cfg.patch) * n_img
            e.update({"bound": "alu", "algorithmic_tflops": fl / sec / 1e12, "algorithmic_gbs": 12.0 * n_img / sec / 1e9,
                      "frac_symmetric_flop_count": flops_per_px_update_symmetric(cfg.window, cfg.patch) * n_img / sec / 1e12 / peak_tf})
        elif kind == "transpose":
            # the copies the forward projector reads: one transposed image (read 4 B, write 4 B per pixel), or, for
            # groups of four slices of a batch, the two interleaved copies (read 4 B, write 8 B per pixel)
            e.update({"bound": "hbm", "algorithmic_gbs": (12.0 if n_slices >= 4 else 8.0) * n_img / sec / 1e9})
        elif kind == "cgls_vector":
            # mean over its launches: r update (16 B per ray), fused u/s update (28 B per pixel), last u update (12 B)
            e.update({"bound": "hbm", "algorithmic_gbs": None})
        if e.get("algorithmic_tflops") is not None:
            e["frac_of_fp32_peak"] = e["algorithmic_tflops"] / peak_tf
        if e.get("algorithmic_gbs") is not None:
            e["frac_of_hbm_peak"] = e["algorithmic_gbs"] / hbm_gbs
        out.append(e)
    _ = n_sino
    return out


def time_recon(ctx, which):
    """Second half of BASELINE.json's metric: seconds per 10-phase slice reconstruction (tnlm_reconstruct),
    on configs[3] (which=4: 512x512x10, 60 views, W=15, d=7, 30 outer), configs[2] (which=3: 360 views,
    W=11, d=5, 20 outer, 5 CGLS steps) or configs[0] (which=1: 64x64).  Single slice: the working set is L2
    resident by construction (the same slice is iterated K times), so L2 is not flushed between iterations."""
    tn, torch = ctx["tn"], ctx["torch"]
    cfg = workloads.config(which)
    inp = workloads.make_inputs(cfg)
    h = tn.create(tn.Geometry(**workloads.geometry_kwargs(cfg)), cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch,
                  cfg.h, cfg.mu)
    tn.reserve(h, 1, cfg.m1, cfg.m2, False)
    y = torch.from_numpy(inp["y"].astype(np.float32)).cuda()
    w = torch.from_numpy(inp["w"].astype(np.float32)).cuda()
    out = torch.empty(1, cfg.N, cfg.L, cfg.L, device="cuda")
    st = torch.cuda.current_stream()
    tn.reconstruct(h, y, w, None, 2, cfg.m1, cfg.m2, out, st)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, n0 = (1 if which == 3 else 3), h.launch_count
    a.record(st)
    for _ in range(reps):
        tn.reconstruct(h, y, w, None, cfg.K, cfg.m1, cfg.m2, out, st)
    b.record(st)
    torch.cuda.synchronize()
    s = a.elapsed_time(b) * 1e-3 / reps
    launches = int((h.launch_count - n0) // reps)
    ph = torch.from_numpy(inp["phantom"].astype(np.float32)).cuda()
    err = float(((out - ph).norm() / ph.norm()).item())
    res = {"metric": "s per 10-phase slice recon", "value": s, "unit": "s", "higher_is_better": False,
           "workload": f"BASELINE.json configs[{which - 1}]: {cfg.L}x{cfg.L}x{cfg.N}, {cfg.V} views x {cfg.B} bins, "
                       f"W={cfg.window} d={cfg.patch}, K={cfg.K} m1={cfg.m1} m2={cfg.m2}, f0=0",
           "gpu_launches": launches, "rel_l2_to_phantom": err,
           "paper_context": "40-90 s per 10-phase slice on a Tesla C1060 (PAPER.md:L15), other workload"}
    # per-kernel split of one outer iteration (library event pairs), with the algorithmic rates
    k_prof = 3
    tn.profile_kernels(h, True)
    tn.reconstruct(h, y, w, None, k_prof, cfg.m1, cfg.m2, out, st)
    table = kernel_table(tn, h, k_prof, 1.0)
    tn.profile_kernels(h, False)
    res["kernels"] = recon_kernel_entries(cfg, 1, table, 1e6 * s / cfg.K, ctx["peak_tf"], ctx["hbm_gbs"])
    if which != 1:
        # quality figures of the paper's section 3 on the synthetic phantom (Eq. 10, Eq. 11): TNLM result vs the
        # all-phase FBP image (step 1 of the algorithm, tnlm_fbp_init), mean over the phases
        from workloads import quality
        tn.reconstruct(h, y, w, None, cfg.K, cfg.m1, cfg.m2, out, st)
        fbp = torch.empty_like(out)
        tn.fbp_init(h, y, fbp, st)
        torch.cuda.synchronize()
        truth = inp["phantom"][0]

        def figures(img_dev, tag, q):
            img = img_dev[0].cpu().numpy()
            q["snr_db_" + tag] = q["cnr_tumour_" + tag] = 0.0
            for i in range(cfg.N):
                sig, bg = quality.tumour_rois(truth[i])
                q["snr_db_" + tag] += quality.snr_db(img[i], truth[i]) / cfg.N
                q["cnr_tumour_" + tag] += quality.cnr(img[i], sig, bg) / cfg.N
            return q

        res["quality"] = figures(fbp, "fbp_all_phases", figures(out, "tnlm", {}))
        if which == 4:
            # the paper's own start (TNLM Algorithm step 1): f^(0) = FBP of all projections of all
            # phases (tnlm_fbp_init), then the K outer iterations -- both inside the timed region
            out2 = torch.empty_like(out)
            tn.fbp_init(h, y, fbp, st)
            tn.reconstruct(h, y, w, fbp, 1, cfg.m1, cfg.m2, out2, st)
            torch.cuda.synchronize()
            n0 = h.launch_count
            a.record(st)
            for _ in range(reps):
                tn.fbp_init(h, y, fbp, st)
                tn.reconstruct(h, y, w, fbp, cfg.K, cfg.m1, cfg.m2, out2, st)
            b.record(st)
            torch.cuda.synchronize()
            res["fbp_start"] = {
                "metric": "s per 10-phase slice recon", "value": a.elapsed_time(b) * 1e-3 / reps, "unit": "s",
                "higher_is_better": False, "workload": res["workload"].replace("f0=0", "f0=FBP of all phases (tnlm_fbp_init, timed)"),
                "gpu_launches": int((h.launch_count - n0) // reps),
                "rel_l2_to_phantom": float(((out2 - ph).norm() / ph.norm()).item()),
                "quality": figures(out2, "tnlm_fbp_start", {"snr_db_tnlm_zero_start": res["quality"]["snr_db_tnlm"],
                                                            "cnr_tumour_tnlm_zero_start": res["quality"]["cnr_tumour_tnlm"]})}
    if not ctx["args"].no_cpu:
        # the oracle on the host cores for the same config, bounded: K_o outer iterations (all K for the tiny
        # config), with the GPU result of the same K_o compared element by element (parity at this size)
        import oracle
        k_o = cfg.K if which == 1 else 1
        og = oracle.Geometry(**workloads.geometry_kwargs(cfg))
        y64, w64 = inp["y"][0].astype(np.float32), inp["w"][0].astype(np.float32)
        t0 = time.perf_counter()
        want = oracle.reconstruct(og, y64, w64, None, cfg.L, cfg.L, cfg.window, cfg.patch, cfg.h, cfg.mu, k_o, cfg.m1, cfg.m2)
        dt = time.perf_counter() - t0
        tn.reconstruct(h, y, w, None, k_o, cfg.m1, cfg.m2, out, st)
        got = out[0].cpu().numpy().astype(np.float64)
        res["parity"] = {"outer_iterations": k_o,
                         "rel_l2_vs_oracle": float(np.linalg.norm(got - want) / np.linalg.norm(want))}
        res["cpu_baseline"] = {"value": dt * cfg.K / k_o, "unit": "s", "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": f"{k_o} of {cfg.K} outer iterations in {dt:.1f} s"
                                         + ("" if k_o == cfg.K else f", scaled x{cfg.K}/{k_o} (extrapolated)")}
    h.close()
    return res


def time_recon_batch(ctx):
    """BASELINE.json configs[4]: 64 independent slices of 512x512x10, 60 views x 888 bins, W=15, d=7, 20 outer
    iterations, sharded contiguously over the ranks (sharding.slice_range), each rank one tnlm_reconstruct call
    over its share.  671 MB per image buffer at S=64: the only config whose working set leaves L2."""
    tn, torch, dist, world, rank, args = (ctx[k] for k in ("tn", "torch", "dist", "world", "rank", "args"))
    cfg = workloads.config(5)
    K = cfg.K if args.batch_outer is None else args.batch_outer
    # every rank builds only its own slices on the host (slice s of the sample equals slice s of the full config)
    from paper_1009_1351_b200.sharding import slice_range
    own = slice_range(cfg.S, world, rank)
    full = workloads.make_inputs(cfg, slices=list(own), phantom=False) if len(own) else {}
    h = tn.create(tn.Geometry(**workloads.geometry_kwargs(cfg)), cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch,
                  cfg.h, cfg.mu)
    st = torch.cuda.current_stream()
    state = {}

    def run_local(mine):
        S = len(mine)
        if S == 0:
            return torch.zeros(0, cfg.N, 2, device="cuda"), 0.0
        tn.reserve(h, S, cfg.m1, cfg.m2, False)
        assert (mine.start, mine.stop) == (own.start, own.stop)
        y = torch.from_numpy(full["y"].astype(np.float32)).cuda()
        w = torch.from_numpy(full["w"].astype(np.float32)).cuda()
        out = torch.empty(S, cfg.N, cfg.L, cfg.L, device="cuda")
        tn.reconstruct(h, y, w, None, 1, cfg.m1, cfg.m2, out, st)          # warm-up: one outer iteration
        ctx["barrier"]()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n0 = h.launch_count
        a.record(st)
        tn.reconstruct(h, y, w, None, K, cfg.m1, cfg.m2, out, st)
        b.record(st)
        ctx["barrier"]()
        state.update(y=y, w=w, out=out, S=S, launches=h.launch_count - n0)
        digest = torch.stack([out.mean(dim=(2, 3)), out.square().sum(dim=(2, 3)).sqrt()], dim=2)   # [S][N][2]
        return digest, a.elapsed_time(b) * 1e-3

    digest, seconds, mine = sharded_batch(cfg.S, world, rank, dist, run_local, "cuda")
    res = None
    if rank == 0:
        S = state["S"]
        res = {"metric": "s per 10-phase slice recon", "value": seconds / cfg.S, "unit": "s",
               "higher_is_better": False, "slices_per_s": cfg.S / seconds, "batch_seconds": seconds,
               "workload": f"BASELINE.json configs[4]: {cfg.S} slices x {cfg.L}x{cfg.L}x{cfg.N}, {cfg.V} views x "
                           f"{cfg.B} bins, W={cfg.window} d={cfg.patch}, K={K} m1={cfg.m1} m2={cfg.m2}, f0=0",
               "sharding": f"{world} rank(s), contiguous slice ranges, rank 0 holds slices {mine.start}..{mine.stop - 1}; "
                           f"no collective on the data path",
               "gpu_launches": int(state["launches"]),
               "digest_all_finite": bool(torch.isfinite(digest).all().item()), "digest_slices": int(digest.shape[0]),
               "l2": "working set (0.67 GB per image buffer, 136 MB per sinogram buffer per 64 slices) exceeds L2"}
        k_prof = 1
        tn.profile_kernels(h, True)
        tn.reconstruct(h, state["y"], state["w"], None, k_prof, cfg.m1, cfg.m2, state["out"], st)
        table = kernel_table(tn, h, k_prof, 1.0)
        tn.profile_kernels(h, False)
        res["kernels"] = recon_kernel_entries(cfg, S, table, 1e6 * seconds / K, ctx["peak_tf"], ctx["hbm_gbs"])
        if world == 1 and not args.no_cpu:
            # parity at S = 64 and the oracle's time: slices 0, 31, 63 after one outer iteration, scaled x64/3 x K
            import oracle
            pick = [0, 31, 63]
            og = oracle.Geometry(**workloads.geometry_kwargs(cfg))
            y3, w3 = full["y"][pick].astype(np.float32), full["w"][pick].astype(np.float32)
            t0 = time.perf_counter()
            want = oracle.reconstruct(og, y3, w3, None, cfg.L, cfg.L, cfg.window, cfg.patch, cfg.h, cfg.mu, 1, cfg.m1, cfg.m2)
            dt = time.perf_counter() - t0
            tn.reconstruct(h, state["y"], state["w"], None, 1, cfg.m1, cfg.m2, state["out"], st)
            got = state["out"][pick].cpu().numpy().astype(np.float64)
            res["parity"] = {"outer_iterations": 1, "slices": pick,
                             "rel_l2_vs_oracle": [float(np.linalg.norm(got[a] - want[a]) / np.linalg.norm(want[a])) for a in range(3)]}
            res["cpu_baseline"] = {"value": dt * (cfg.S / 3.0) * K / cfg.S, "unit": "s", "cores": oracle.num_threads(),
                                   "kind": "oracle",
                                   "sample": f"slices 0, 31, 63, one outer iteration, in {dt:.1f} s; per-slice figure scaled "
                                             f"x{K} outer iterations (extrapolated: slices and iterations cost the same)"}
    state.clear()
    h.close()
    torch.cuda.empty_cache()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline legs and the oracle parity figures")
    ap.add_argument("--no-recon", action="store_true", help="skip the single-slice reconstruction timings")
    ap.add_argument("--no-batch", action="store_true", help="skip the 64-slice batch (configs[4])")
    ap.add_argument("--batch-outer", type=int, default=None, help="outer iterations of the 64-slice batch (default: the config's 20)")
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 5 if args.impl == "reference" else 200
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args)
    run_ours(args)


if __name__ == "__main__":
    main()
