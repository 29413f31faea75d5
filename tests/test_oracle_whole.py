"""Pins for the oracle's outer loop, "TNLM Algorithm" -- CPU only."""
import numpy as np

import oracle
import workloads


def small_case(L=32, V=48, B=56, N=4, seed=0):
    cfg = workloads.Config("small", L=L, N=N, V=V, B=B, pitch=1.0, sid=60.0, sdd=100.0,
                           window=5, patch=3, h=0.01, mu=0.2, seed=seed)
    geom = oracle.Geometry(**workloads.geometry_kwargs(cfg))
    ph = workloads.make_inputs(cfg)["phantom"][0]
    return cfg, geom, ph


def test_mu_zero_is_restarted_cgls_with_clip():
    # With mu = 0 the regularisation step is the identity, so K outer iterations are K restarts
    # of M1-step CGLS least squares, each followed by the positivity clip (north_star pin).
    cfg, geom, ph = small_case()
    rng = np.random.default_rng(1)
    y = oracle.project(geom, ph) + 0.05 * rng.standard_normal((cfg.N, cfg.V, cfg.B))
    w = rng.uniform(0.5, 2.0, y.shape)
    got = oracle.reconstruct(geom, y, w, None, cfg.L, cfg.L, 5, 3, 0.01, 0.0, 3, 2, 1)
    f = np.zeros_like(ph)
    for _ in range(3):
        f = np.maximum(oracle.cgls_step(geom, f, y, w, 2), 0.0)
    assert np.array_equal(got, f)
    # K = 0 returns f0 untouched, and one outer iteration is cgls_step -> regularize_step
    f0 = rng.random(ph.shape)
    assert np.array_equal(oracle.reconstruct(geom, y, w, f0, cfg.L, cfg.L, 5, 3, 0.01, 0.3, 0, 2, 1), f0)
    one = oracle.reconstruct(geom, y, w, f0, cfg.L, cfg.L, 5, 3, 0.01, 0.3, 1, 2, 2)
    want = oracle.regularize_step(oracle.cgls_step(geom, f0, y, w, 2), 5, 3, 0.01, 0.3, 2)
    assert np.array_equal(one, want)


def test_noise_free_fully_sampled_converges_to_the_phantom():
    # Consistent data y = P f*, w = 1, plenty of views: the iteration must recover f*.
    cfg, geom, ph = small_case(N=3)
    y = oracle.project(geom, ph)
    errs = []
    for K in (2, 10, 40):
        rec = oracle.reconstruct(geom, y, None, None, cfg.L, cfg.L, 5, 3, 0.004, 0.05, K, 5, 1)
        errs.append(np.linalg.norm(rec - ph) / np.linalg.norm(ph))
    assert errs[0] > errs[1] > errs[2], errs
    assert errs[2] < 0.02, errs


def test_tnlm_reduces_noise_relative_to_plain_cgls():
    # The point of the method: features repeated across phases survive, noise
    # does not.  Same data, mu>0 vs mu=0, error to the phantom must drop.
    cfg = workloads.config(1)
    inp = workloads.make_inputs(cfg)
    geom = oracle.Geometry(**workloads.geometry_kwargs(cfg))
    ph, y, w = inp["phantom"][0], inp["y"][0], inp["w"][0]
    with_reg = oracle.reconstruct(geom, y, w, None, cfg.L, cfg.L, cfg.window, cfg.patch, cfg.h, cfg.mu, cfg.K, cfg.m1, cfg.m2)
    no_reg = oracle.reconstruct(geom, y, w, None, cfg.L, cfg.L, cfg.window, cfg.patch, cfg.h, 0.0, cfg.K, cfg.m1, cfg.m2)
    e1 = np.linalg.norm(with_reg - ph); e0 = np.linalg.norm(no_reg - ph)
    assert e1 < e0
    assert (with_reg >= 0).all()


def test_slices_are_independent():
    cfg, geom, ph = small_case(L=16, V=12, B=28, N=3)
    rng = np.random.default_rng(3)
    y = rng.random((2, cfg.N, cfg.V, cfg.B)); w = rng.uniform(1, 2, y.shape)
    both = oracle.reconstruct(geom, y, w, None, cfg.L, cfg.L, 3, 3, 0.05, 0.2, 2, 2, 1)
    for s in range(2):
        one = oracle.reconstruct(geom, y[s], w[s], None, cfg.L, cfg.L, 3, 3, 0.05, 0.2, 2, 2, 1)
        assert np.array_equal(both[s], one)


def test_golden_digest_of_config_1():
    # Regression fixture written by tests/golden/make_golden.py (which calls only oracle/).
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg1_oracle_digest.txt")
    vals = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split("=")
        vals[k.strip()] = float(v)
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(os.path.dirname(path), "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.digest()
    for k, v in vals.items():
        assert abs(now[k] - v) <= 1e-9 * abs(v), (k, now[k], v)
