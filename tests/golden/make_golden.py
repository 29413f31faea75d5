"""Writes tests/golden/cfg1_oracle_digest.txt.  Calls ONLY oracle/ (and the input generator).

The paper prints no worked numerical example for the hot path (no intermediate image,
weight or iterate values; section 3 gives only NCAT quality tables), so there is no
paper-cited golden value.  This fixture is a regression digest of the oracle itself on
BASELINE config 1 so that an accidental change of the oracle's arithmetic is noticed.

Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle      # noqa: E402
import workloads   # noqa: E402


def digest():
    cfg = workloads.config(1)
    inp = workloads.make_inputs(cfg)
    geom = oracle.Geometry(**workloads.geometry_kwargs(cfg))
    y, w = inp["y"][0], inp["w"][0]
    g = oracle.cgls_step(geom, np.zeros((cfg.N, cfg.L, cfg.L)), y, w, cfg.m1)
    f1 = oracle.regularize_step(g, cfg.window, cfg.patch, cfg.h, cfg.mu, cfg.m2)
    rec = oracle.reconstruct(geom, y, w, None, cfg.L, cfg.L, cfg.window, cfg.patch, cfg.h, cfg.mu,
                             cfg.K, cfg.m1, cfg.m2)
    return {
        "sum_y": float(y.sum()),
        "l2_cgls_step": float(np.linalg.norm(g)),
        "l2_first_outer": float(np.linalg.norm(f1)),
        "l2_recon_K5": float(np.linalg.norm(rec)),
        "recon_pixel_3_32_40": float(rec[3, 32, 40]),
    }


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle_digest.txt")
    with open(out, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py (oracle only); BASELINE config 1, seed 0\n")
        for k, v in digest().items():
            fh.write(f"{k} = {v!r}\n")
    print(open(out).read())
