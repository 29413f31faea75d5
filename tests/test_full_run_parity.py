"""Parity after the FULL run of a BASELINE.json configuration: tnlm_reconstruct with the config's K outer
iterations against oracle.reconstruct, every pixel ("relative L2 GPU-vs-oracle per
single step and after the full run"; north_star: <= 1e-3 after 20 outer iterations).

configs[0] runs in every `pytest -m gpu`.  The 512 x 512 configurations need 3 to 11 minutes of oracle time each on
16 host cores, so they run only on request:

    TNLM_FULL_RUN=1 python -m pytest tests/test_full_run_parity.py -m gpu -s

(-s shows the JSON line of each case; profiles/ keeps the lines of the last such run).  For config 5 the library runs
ALL 64 slices in one call (the batch kernels); the oracle runs slices 0 and 63 only.
"""
import json
import os
import time

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

RECON_TOL = 1e-3         # BASELINE.json north_star, after 20 outer iterations
REGRESSION_TOL = 3e-5    # a few times what these runs measure (3e-6 .. 8e-6)
FULL = os.environ.get("TNLM_FULL_RUN") == "1"
slow = pytest.mark.skipif(not FULL, reason="minutes of oracle time per case: set TNLM_FULL_RUN=1")


@pytest.mark.parametrize("config,slices", [(1, None),
                                           pytest.param(4, None, marks=[slow, pytest.mark.slow]),
                                           pytest.param(3, None, marks=[slow, pytest.mark.slow]),
                                           pytest.param(5, (0, 63), marks=[slow, pytest.mark.slow])],
                         ids=["configs0", "configs3", "configs2", "configs4_slices_0_63"])
def test_full_run_matches_oracle(config, slices):
    import torch
    from paper_1009_1351_b200 import build
    build.build()
    import paper_1009_1351_b200 as tn
    cfg = workloads.config(config)
    inp = workloads.make_inputs(cfg, phantom=False)
    kw = workloads.geometry_kwargs(cfg)
    h = tn.create(tn.Geometry(**kw), cfg.L, cfg.L, cfg.N, cfg.window, cfg.patch, cfg.h, cfg.mu)
    y, w = inp["y"].astype(np.float32), inp["w"].astype(np.float32)
    S = y.shape[0]
    out = torch.empty(S, cfg.N, cfg.L, cfg.L, device="cuda")
    t0 = time.perf_counter()
    tn.reconstruct(h, torch.from_numpy(y).cuda(), torch.from_numpy(w).cuda(), None, cfg.K, cfg.m1, cfg.m2, out)
    torch.cuda.synchronize()
    t_gpu = time.perf_counter() - t0
    pick = list(range(S)) if (slices is None or S == 1) else list(slices)
    t0 = time.perf_counter()
    want = oracle.reconstruct(oracle.Geometry(**kw), y[pick], w[pick], None, cfg.L, cfg.L, cfg.window, cfg.patch,
                              cfg.h, cfg.mu, cfg.K, cfg.m1, cfg.m2)
    t_cpu = time.perf_counter() - t0
    got = out[pick].cpu().numpy().astype(np.float64)
    rel = [float(np.linalg.norm(got[i] - want[i]) / np.linalg.norm(want[i])) for i in range(len(pick))]
    mx = [float(np.abs(got[i] - want[i]).max() / np.abs(want[i]).max()) for i in range(len(pick))]
    print("\n" + json.dumps({"config": config, "workload": cfg.name, "outer_iterations": cfg.K, "m1": cfg.m1, "m2": cfg.m2,
                             "slices_in_the_call": S, "slices_compared": pick, "rel_l2_vs_oracle": rel,
                             "max_abs_over_max": mx, "bar": RECON_TOL, "gpu_seconds_incl_first_use": t_gpu,
                             "oracle_seconds": t_cpu, "oracle_threads": oracle.num_threads(), "library": tn.version()}))
    assert max(rel) < RECON_TOL
    assert max(rel) < REGRESSION_TOL
    h.close()
