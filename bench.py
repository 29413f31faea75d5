#!/usr/bin/env python
"""bench.py -- headline benchmark of libtnlm on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Metric (BASELINE.json): TNLM Gauss-Jacobi pixel-updates/s (px x phase x iter).  Workload at
N=1: BASELINE.json configs[1] ("TNLM step alone": 256x256 fp32 x 10 cyclic phases, window 11,
patch 5, h=0.008, mu=0.1, 10 Gauss-Jacobi sweeps, seed 1).  One step = one
tnlm_regularize_step call (weights + 10 sweeps + clip) on one slice per GPU: 1 launch of
gj_sweep_kernel<.,.,true> (weights of g, sweep 1, stores the weights as bf16) and 9 launches of
gj_apply_kernel (sweeps 2..10 from the stored weights, HBM bound).  With N>1 every
rank runs its own slice (slices are independent: no collective on the data path; weak scaling).

Timed region: K steps, each bracketed by CUDA events on the launching stream; L2 is flushed
(a 256 MiB device buffer is rewritten) between steps, outside the event brackets; a barrier and
torch.cuda.synchronize() on both sides; the max over ranks is taken.  The second half of the
metric ("s per 10-phase slice recon") is reported under "recon" for BASELINE.json configs[3].

--impl reference times the CPU oracle (oracle/, plain C fp64) on the host cores, on a bounded
sample of the same workload.  Only that leg and `cpu_baseline` touch oracle/.
"""
import argparse
import json
import os
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


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def flops_per_px_update(window, patch):
    """Algorithmic flops of one Gauss-Jacobi pixel update with the weights computed on the fly, in the
    separable box-sum form: 2 neighbours x W^2 offsets x (2d+4) flops."""
    return 2 * window * window * (2 * patch + 4)


def bytes_per_px_update_stored(window):
    """Algorithmic HBM bytes of one Gauss-Jacobi pixel update from stored weights:
    2 neighbours x W^2 bf16 weights + g, u read and u' written once (3 x 4 bytes)."""
    return 2 * window * window * 2 + 12


class ClockSampler:
    """Samples SM clock and throttle reasons (NVML) in a thread while the timed region runs."""

    def __init__(self, torch_device_index, period=0.05):
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
    (weights recomputed per sweep, as oracle_regularize_step does) until ~budget_s is spent."""
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
    sample = f"{sweeps_tot} whole Gauss-Jacobi sweeps (weights + update) of cfg2 256x256x10 in {secs:.1f} s"
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


# ---------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if local == 0:
        from paper_1009_1351_b200 import build
        build.build()                # no-op when libtnlm.so is newer than its sources
    import paper_1009_1351_b200 as tn
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libtnlm has no CPU fallback")
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
    cfg, g_np = cfg2_input(1 + rank)                 # one independent slice per rank
    n_px_step = g_np.size * cfg.m2                   # pixel updates of one step on this rank
    h = tn.create(None, cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch, cfg.h, cfg.mu)
    g = torch.from_numpy(g_np).cuda()
    f = torch.empty_like(g)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        tn.regularize_step(h, g, cfg.m2, f, stream)

    for _ in range(max(args.warmup, 3)):
        flush.fill_(1); step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    n0 = h.launch_count
    with ClockSampler(torch.cuda.current_device()) as cs:
        barrier()
        for a, b in ev:
            flush.fill_(1)
            a.record(stream); step(); b.record(stream)
        barrier()
    launches = h.launch_count - n0
    ms = sum(a.elapsed_time(b) for a, b in ev)

    # ---- per-kernel durations: the same K steps again with the library's event pair around every
    # launch (CUDA events on the launching stream; kept out of the headline region above)
    tn.profile_sweeps(h, True)
    kern = {}
    for _ in range(args.steps):
        flush.fill_(1); step()
        for kind, kms in tn.sweep_times(h):
            kern.setdefault(kind, []).append(kms)
    tn.profile_sweeps(h, False)
    torch.cuda.synchronize()
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_per_step = ms_total / args.steps
    value = world * n_px_step / (ms_per_step * 1e-3)

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
    e2e_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = world * n_px_step * n_e2e / float(te.item())
    checksum = float(fh.double().sum().item())

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peaks, peak_src = measured_peaks()
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    peak_tf_derived = N_SM * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12
    peak_tf = tn.fma_peak(stream)               # FFMA-chain probe of the library, same run, same box
    n_px = g_np.size
    traffic = {}
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_file):
        try:
            traffic = json.load(open(traffic_file))
        except Exception:
            traffic = {}
    kernels = []
    step_us = ms_per_step * 1e3
    for kind, vals in sorted(kern.items()):
        us = 1e3 * float(np.mean(vals))
        per_step = len(vals) / args.steps
        k = {"kernel": {"sweep": "gj_sweep_kernel<PB,RB,false> (weights on the fly + sweep)",
                        "sweep_store": "gj_sweep_kernel<PB,RB,true> (weights on the fly + sweep, stores bf16 weights)",
                        "apply": "gj_apply_kernel (sweep from stored bf16 weights)"}[kind],
             "launches_per_step": per_step, "us_per_launch": us, "share_of_step": per_step * us / step_us}
        if kind == "apply":
            gbs = bytes_per_px_update_stored(cfg.window) * n_px / (us * 1e-6) / 1e9
            k.update({"bound": "hbm", "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs,
                      "traffic": traffic.get("gj_apply_cfg2_dram_bytes_per_launch"),
                      "algorithmic_bytes_per_px_update": bytes_per_px_update_stored(cfg.window)})
        else:
            tf = flops_per_px_update(cfg.window, cfg.patch) * n_px / (us * 1e-6) / 1e12
            k.update({"bound": "alu", "achieved": tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": tf / peak_tf,
                      "traffic": traffic.get("gj_%s_cfg2_dram_bytes_per_launch" % kind),
                      "algorithmic_flops_per_px_update": flops_per_px_update(cfg.window, cfg.patch)})
        kernels.append(k)
    dominant = max(kernels, key=lambda k: k["share_of_step"]) if kernels else {}
    roofline = {key: dominant.get(key) for key in ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic",
                                                   "us_per_launch", "launches_per_step", "share_of_step")}
    roofline["peak_source"] = (
        f"{peak_src} MEASURED_PEAKS.json hbm_gbs (burst copy figure)" if dominant.get("bound") == "hbm" else
        "measured in this run by tnlm_fma_peak (8-chain FFMA kernel)")
    roofline["kernels"] = kernels
    roofline["fp32_peak_tflops_measured"] = peak_tf
    roofline["fp32_peak_tflops_derived"] = peak_tf_derived

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(cfg, world), "clocks": cs.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(g_np.nbytes),
                    "d2h_bytes_per_step": int(g_np.nbytes), "calls": n_e2e, "checksum": checksum},
            "gpu_launches": int(launches), "roofline": roofline}

    if world == 1 and not args.no_recon:
        line["recon"] = time_recon(tn, torch, args)
        line["recon_low_mas"] = time_recon(tn, torch, args, which=3)
    if world == 1 and not args.no_cpu:
        v, sweeps, dt, cores = time_oracle(cfg, g_np.astype(np.float64), args.cpu_budget)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{sweeps} whole Gauss-Jacobi sweep(s) of the same cfg2 slice "
                                          f"(of {cfg.m2}) in {dt:.1f} s"}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def time_recon(tn, torch, args, which=4):
    """Second half of BASELINE.json's metric: seconds per 10-phase slice reconstruction
    (tnlm_reconstruct), on configs[3] (512x512x10, 60 views, 888 bins, W=15, d=7, 30 outer) or, which=3,
    configs[2] (360 views, W=11, d=5, 20 outer, 5 CGLS steps)."""
    cfg = workloads.config(which)
    inp = workloads.make_inputs(cfg)
    h = tn.create(tn.Geometry(**workloads.geometry_kwargs(cfg)), cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch,
                  cfg.h, cfg.mu)
    y = torch.from_numpy(inp["y"].astype(np.float32)).cuda()
    w = torch.from_numpy(inp["w"].astype(np.float32)).cuda()
    out = torch.empty(1, cfg.N, cfg.L, cfg.L, device="cuda")
    st = torch.cuda.current_stream()
    tn.reconstruct(h, y, w, None, 2, cfg.m1, cfg.m2, out, st)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, n0 = (3 if which == 4 else 1), h.launch_count
    a.record(st)
    for _ in range(reps):
        tn.reconstruct(h, y, w, None, cfg.K, cfg.m1, cfg.m2, out, st)
    b.record(st)
    torch.cuda.synchronize()
    s = a.elapsed_time(b) * 1e-3 / reps
    ph = torch.from_numpy(inp["phantom"].astype(np.float32)).cuda()
    err = float(((out - ph).norm() / ph.norm()).item())
    # quality figures of the paper's section 3 on the synthetic phantom (Eq. 10, Eq. 11): TNLM result vs the
    # all-phase FBP image (step 1 of the algorithm, tnlm_fbp_init), mean over the phases
    from workloads import quality
    fbp = torch.empty_like(out)
    tn.fbp_init(h, y, fbp, st)
    torch.cuda.synchronize()
    rec, fb, truth = out[0].cpu().numpy(), fbp[0].cpu().numpy(), inp["phantom"][0]
    q = {"snr_db_tnlm": 0.0, "snr_db_fbp_all_phases": 0.0, "cnr_tumour_tnlm": 0.0, "cnr_tumour_fbp_all_phases": 0.0}
    for i in range(cfg.N):
        sig, bg = quality.tumour_rois(truth[i])
        q["snr_db_tnlm"] += quality.snr_db(rec[i], truth[i]) / cfg.N
        q["snr_db_fbp_all_phases"] += quality.snr_db(fb[i], truth[i]) / cfg.N
        q["cnr_tumour_tnlm"] += quality.cnr(rec[i], sig, bg) / cfg.N
        q["cnr_tumour_fbp_all_phases"] += quality.cnr(fb[i], sig, bg) / cfg.N
    return {"metric": "s per 10-phase slice recon", "value": s, "unit": "s", "higher_is_better": False,
            "workload": f"BASELINE.json configs[{which - 1}]: {cfg.L}x{cfg.L}x{cfg.N}, {cfg.V} views x {cfg.B} bins, "
                        f"W={cfg.window} d={cfg.patch}, K={cfg.K} m1={cfg.m1} m2={cfg.m2}, f0=0",
            "gpu_launches": int((h.launch_count - n0) // reps), "rel_l2_to_phantom": err, "quality": q,
            "paper_context": "40-90 s per 10-phase slice on a Tesla C1060 (PAPER.md:L15), other workload"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-recon", action="store_true", help="skip the reconstruction timing")
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 5 if args.impl == "reference" else 200
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
