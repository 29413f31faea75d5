"""tnlm_regularize_step_noalloc against the existing tnlm_regularize_step (`pytest -m gpu`).

Why the entry point exists: some users of this library cannot call cudaMalloc at the moment they need a TNLM
step -- all of HBM already belongs to another allocator (a framework's memory pool holding a multi-slice batch),
or other streams are in flight and must not be stalled by the device-wide synchronisation an allocation implies.
tnlm_regularize_step allocates its ping-pong images and stored weights on first use; the _noalloc variant keeps
the ping-pong images in a 20 MiB array compiled into the library and recomputes the weights in fp32 every sweep.

What is checked: its output equals the existing path's, on two calls in a row whose shapes, sweep counts and
parameters differ -- the second call finds the first call's images in the shared array and must not be affected by
them; then that a repeated call takes no device memory; then the size limit.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure of this add-on must not
hide the parity tests proper.  It needs nothing from the other test modules and passes alone in a fresh process.
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

STEP_TOL = 1e-4          # BASELINE.json north_star: relative L2 per single step, the bar of tests/test_gpu_parity.py


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def T():
    import torch
    from paper_1009_1351_b200 import build
    build.build()                    # no-op when libtnlm.so is newer than its sources
    import paper_1009_1351_b200 as tn
    assert torch.cuda.is_available()
    return torch, tn


def noisy_stack(N, ny, nx, seed, sigma=0.002):
    """Thorax-like phases (workloads' ellipse phantom) cropped to ny x nx, plus image-domain noise."""
    cfg = workloads.Config("p", L=max(ny, nx), N=N)
    ph = workloads.make_inputs(cfg)["phantom"][0][:, :ny, :nx]
    return (ph + sigma * np.random.default_rng(seed).standard_normal(ph.shape)).astype(np.float32)


def existing_path(torch, tn, h, gd, m2):
    """tnlm_regularize_step twice: with the opt-in stored bf16 weights (sweeps 2..m2 stream them) and as shipped
    (every sweep computes its weights in fp32)."""
    stored = torch.empty_like(gd)
    tn.set_option(h, "weight_cache_mb", 16384)
    tn.regularize_step(h, gd, m2, stored)
    tn.set_option(h, "weight_cache_mb", 0)
    fp32 = torch.empty_like(gd)
    tn.regularize_step(h, gd, m2, fp32)
    return stored, fp32


def test_two_calls_in_a_row_match_the_existing_path(T):
    torch, tn = T
    # call 1: three phases of 150 x 260 (three column tiles, ragged tails), 3 sweeps: both halves of the array used
    # call 2: a SMALLER stack with another window, patch and h, 2 sweeps, on another handle: it finds call 1's
    #         images in the array, beyond and inside its own extent
    cases = [(3, 150, 260, 9, 3, 0.006, 0.15, 3), (4, 41, 67, 5, 5, 0.01, 0.3, 2)]
    prepared = []
    for (N, ny, nx, W, d, h, mu, m2) in cases:
        g = noisy_stack(N, ny, nx, seed=N * 10 + W)
        g[0, 3, 4] = -0.003                                    # something for the clip to do
        hd = tn.create(None, nx, ny, N, W, d, h, mu)           # TNLM-only handle: owns no device memory
        gd = torch.from_numpy(g).cuda()
        stored, fp32 = existing_path(torch, tn, hd, gd, m2)
        prepared.append((g, gd, hd, m2, stored, fp32, (W, d, h, mu)))
    outs = []
    for (g, gd, hd, m2, stored, fp32, _) in prepared:          # the two calls, back to back on one stream
        out = torch.full_like(gd, float("nan"))
        tn.regularize_step_noalloc(hd, gd, m2, out)
        outs.append(out)
    torch.cuda.synchronize()
    for out, (g, gd, hd, m2, stored, fp32, (W, d, h, mu)) in zip(outs, prepared):
        assert torch.isfinite(out).all()
        assert rel(out.cpu().numpy(), stored.cpu().numpy()) < STEP_TOL      # vs the stored-weight path
        assert torch.equal(out, fp32)                                       # vs the path as shipped: same kernels, same bits
        assert rel(out.cpu().numpy(), oracle.regularize_step(g, W, d, h, mu, m2)) < STEP_TOL
    # in place (f_out aliases g), m2 = 1 and m2 = 0 behave like the existing call
    g, gd, hd, m2, stored, fp32, _ = prepared[1]
    b = gd.clone(); tn.regularize_step_noalloc(hd, b, m2, b)
    assert torch.equal(b, fp32)
    one = torch.empty_like(gd); ref1 = torch.empty_like(gd)
    tn.regularize_step_noalloc(hd, gd, 1, one); tn.regularize_step(hd, gd, 1, ref1)
    assert torch.equal(one, ref1)
    tn.regularize_step_noalloc(hd, gd, 0, one)
    assert torch.equal(one, gd.clamp_min(0))


def test_repeated_call_takes_no_device_memory(T):
    torch, tn = T
    N, ny, nx = 3, 64, 96
    gd = torch.from_numpy(noisy_stack(N, ny, nx, seed=5)).cuda()
    out = torch.empty_like(gd)
    hd = tn.create(None, nx, ny, N, 7, 3, 0.01, 0.2)
    tn.regularize_step_noalloc(hd, gd, 3, out)       # set-up call: address lookup, kernel loading
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    tn.regularize_step_noalloc(hd, gd, 3, out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, (free_before, free_after)


def test_sizes_beyond_the_built_in_scratch_are_refused(T):
    torch, tn = T
    N, ny, nx = 3, 1024, 1024                         # 3.1 M pixels > TNLM_NOALLOC_MAX_PIXELS
    assert N * ny * nx > tn.NOALLOC_MAX_PIXELS
    hd = tn.create(None, nx, ny, N, 5, 3, 0.01, 0.1)
    gd = torch.zeros(N, ny, nx, device="cuda")
    out = torch.full_like(gd, 7.0)
    n0 = hd.launch_count
    with pytest.raises(tn.TnlmError) as ei:
        tn.regularize_step_noalloc(hd, gd, 2, out)
    assert ei.value.code == 4                         # TNLM_UNSUPPORTED
    assert str(tn.NOALLOC_MAX_PIXELS) in str(ei.value) and str(N * ny * nx) in str(ei.value)
    assert hd.launch_count == n0 and bool((out == 7.0).all())     # nothing ran, nothing written
    # exactly at the limit is accepted: one 10-phase 512 x 512 slice (BASELINE.json configs[3] size)
    hb = tn.create(None, 512, 512, 10, 5, 3, 0.01, 0.1)
    gb = torch.rand(10, 512, 512, device="cuda") * 0.02
    assert gb.numel() == tn.NOALLOC_MAX_PIXELS
    a = torch.empty_like(gb); b = torch.empty_like(gb)
    tn.regularize_step_noalloc(hb, gb, 2, a)
    tn.set_option(hb, "weight_cache_mb", 0)
    tn.regularize_step(hb, gb, 2, b)
    assert torch.equal(a, b)
