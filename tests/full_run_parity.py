#!/usr/bin/env python
"""Parity after the FULL run of a BASELINE.json configuration: tnlm_reconstruct with the config's K outer
iterations against oracle.reconstruct, every pixel ("relative L2 GPU-vs-oracle per
single step and after the full run").  Too slow for the pytest suite (the oracle needs minutes on the host
cores): run by hand on a B200 box,

    python tests/full_run_parity.py --config 4            # configs[3]: 512^2 x 10, 60 views, K = 30
    python tests/full_run_parity.py --config 3            # configs[2]: 360 views, K = 20, M1 = 5
    python tests/full_run_parity.py --config 5 --slices 0 63     # two slices of the 64-slice batch, K = 20

and the printed JSON lines are recorded in BASELINE.md.  For config 5 the library runs ALL 64 slices in one
call (the batch kernels: 8 / 4 slices per thread); the oracle runs only the named slices.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle       # noqa: E402
import workloads    # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=[1, 3, 4, 5])
    ap.add_argument("--slices", type=int, nargs="*", default=None, help="config 5: the slices the oracle runs")
    args = ap.parse_args()
    import torch
    import paper_1009_1351_b200 as tn
    cfg = workloads.config(args.config)
    inp = workloads.make_inputs(cfg, phantom=False)
    kw = workloads.geometry_kwargs(cfg)
    h = tn.create(tn.Geometry(**kw), cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch, cfg.h, cfg.mu)
    y, w = inp["y"].astype(np.float32), inp["w"].astype(np.float32)
    if y.ndim == 3:
        y, w = y[None], w[None]
    S = y.shape[0]
    out = torch.empty(S, cfg.N, cfg.L, cfg.L, device="cuda")
    t0 = time.perf_counter()
    tn.reconstruct(h, torch.from_numpy(y).cuda(), torch.from_numpy(w).cuda(), None, cfg.K, cfg.m1, cfg.m2, out)
    torch.cuda.synchronize()
    t_gpu = time.perf_counter() - t0
    pick = list(range(S)) if (args.slices is None or S == 1) else args.slices
    t0 = time.perf_counter()
    want = oracle.reconstruct(oracle.Geometry(**kw), y[pick], w[pick], None, cfg.L, cfg.L, cfg.window, cfg.patch,
                              cfg.h, cfg.mu, cfg.K, cfg.m1, cfg.m2)
    t_cpu = time.perf_counter() - t0
    got = out[pick].cpu().numpy().astype(np.float64)
    rel = [float(np.linalg.norm(got[i] - want[i]) / np.linalg.norm(want[i])) for i in range(len(pick))]
    mx = [float(np.abs(got[i] - want[i]).max() / np.abs(want[i]).max()) for i in range(len(pick))]
    print(json.dumps({"config": args.config, "workload": cfg.name, "outer_iterations": cfg.K, "m1": cfg.m1, "m2": cfg.m2,
                      "slices_in_the_call": S, "slices_compared": pick, "rel_l2_vs_oracle": rel,
                      "max_abs_over_max": mx, "bar": 1e-3, "gpu_seconds_incl_first_use": t_gpu,
                      "oracle_seconds": t_cpu, "oracle_threads": oracle.num_threads()}))


if __name__ == "__main__":
    main()
