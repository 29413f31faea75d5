"""Seeded synthetic inputs for the TNLM 4DCT hot path (numpy only).

This module holds NONE of the method's arithmetic: no projector matrix, no CGLS, no
weights, no Gauss-Jacobi.  It only draws inputs shaped like the paper's workload
(thorax slice, 10 phases, fan-beam arc detector, low-mAs noise) for
the five configurations of BASELINE.json, and serves both the oracle-side tests and the
CUDA-side tests/bench.  The NCAT phantom the paper uses is not available; the stand-in is
an ellipse thorax (body, two lungs, a moving tumour disc) -- see DESIGN.md "Input recipe".

Sinograms are the ANALYTIC line integrals of the continuous ellipse phantom along each
pencil ray (closed form per ellipse), so building inputs needs neither implementation of P.

Conventions (identical to include/tnlm.h and the oracle header, restated here):
  pixel (r,c) centre  X = (c-(nx-1)/2)*pix,  Y = (r-(ny-1)/2)*pix
  source of view th   S = SID*(cos th, sin th)
  bin k fan angle     gam_k = (k-(B-1)/2+off)*pitch/SDD,  ray direction -(cos(th+gam), sin(th+gam))
  view angles         th[i][v] = 2*pi*(v + i/N)/V   (phases interleaved)
"""
from dataclasses import dataclass, replace

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    L: int                 # image is L x L
    N: int = 10            # respiratory phases
    V: int = 0             # views per phase (0 = no projector in this config)
    B: int = 0             # detector bins
    pitch: float = 1.0     # mm along the arc
    sid: float = 541.0
    sdd: float = 949.0
    I0: float = 0.0        # photons per ray before the patient
    window: int = 11
    patch: int = 5
    h: float = 0.01
    mu: float = 0.1
    K: int = 1             # outer iterations
    m1: int = 3            # CGLS inner steps     ("such as M1 = 3")
    m2: int = 1            # Gauss-Jacobi sweeps  ("such as M2 = 1")
    S: int = 1             # independent slices
    seed: int = 0
    sigma: float = 0.0     # image-domain Gaussian noise (config 2 only)
    pix: float = 1.0       # mm


# BASELINE.json:configs[0..4]  (numbered 1..5 as in SURVEY.md section 8)
CONFIGS = {
    1: Config("cfg1_tiny", L=64, V=60, B=96, pitch=1.0, sid=1000.0, sdd=1500.0, I0=1e4,
              window=5, patch=3, h=0.01, mu=0.1, K=5, m1=3, m2=1, seed=0),
    2: Config("cfg2_tnlm_only", L=256, window=11, patch=5, h=0.008, mu=0.1, K=0, m1=0, m2=10,
              seed=1, sigma=0.002),
    3: Config("cfg3_lowmAs_full", L=512, V=360, B=888, I0=5e3, window=11, patch=5, h=0.006,
              mu=0.05, K=20, m1=5, m2=1, seed=2),
    4: Config("cfg4_undersampled_highmAs", L=512, V=60, B=888, I0=1e5, window=15, patch=7,
              h=0.005, mu=0.2, K=30, m1=3, m2=1, seed=3),
    5: Config("cfg5_multislice", L=512, V=60, B=888, I0=5e3, window=15, patch=7, h=0.006,
              mu=0.2, K=20, m1=3, m2=1, S=64, seed=4),
}


def config(i: int, **over) -> Config:
    return replace(CONFIGS[i], **over)


def view_angles(N: int, V: int) -> np.ndarray:
    """[N][V] source angles: equally spaced over 360 deg, phases interleaved by 1/N of a step."""
    v = np.arange(V, dtype=np.float64)[None, :]
    i = np.arange(N, dtype=np.float64)[:, None]
    return 2.0 * np.pi * (v + i / N) / V


def _ellipses(cfg: Config, phase: int, jitter_xy):
    """Additive ellipses (x0, y0, A, B, value) in mm of the continuous phantom at one phase."""
    Hw = 0.5 * cfg.L * cfg.pix
    body = (0.0, 0.0, 0.80 * Hw, 0.58 * Hw, 0.02)
    lung_r = (+0.38 * Hw, 0.0, 0.28 * Hw, 0.36 * Hw, 0.004 - 0.02)
    lung_l = (-0.38 * Hw, 0.0, 0.28 * Hw, 0.36 * Hw, 0.004 - 0.02)
    m = -np.cos(2.0 * np.pi * phase / cfg.N)
    tum = (0.38 * Hw + jitter_xy[0] + 1.0 * m, jitter_xy[1] + 3.0 * m, 4.0, 4.0, 0.02 - 0.004)
    return [body, lung_r, lung_l, tum]


def _raster(cfg: Config, ells, sub: int = 4) -> np.ndarray:
    """Area-sampled (sub x sub per pixel) image of additive ellipses."""
    L = cfg.L
    o = (np.arange(L * sub, dtype=np.float64) + 0.5) / sub - 0.5          # pixel-index units
    xs = (o - (L - 1) / 2.0) * cfg.pix
    X, Y = np.meshgrid(xs, xs)                                             # rows = Y
    img = np.zeros((L * sub, L * sub))
    for (x0, y0, A, B, val) in ells:
        img += val * ((((X - x0) / A) ** 2 + ((Y - y0) / B) ** 2) <= 1.0)
    return img.reshape(L, sub, L, sub).mean(axis=(1, 3))


def _line_integrals(cfg: Config, ells, theta: np.ndarray) -> np.ndarray:
    """Analytic line integrals [V][B] of additive ellipses along the pencil rays of one phase."""
    k = np.arange(cfg.B, dtype=np.float64)
    gam = (k - 0.5 * (cfg.B - 1)) * cfg.pitch / cfg.sdd
    th = theta[:, None]
    sx, sy = cfg.sid * np.cos(th), cfg.sid * np.sin(th)
    dx, dy = -np.cos(th + gam[None, :]), -np.sin(th + gam[None, :])
    p = np.zeros((theta.size, cfg.B))
    for (x0, y0, A, B, val) in ells:
        px, py = (sx - x0) / A, (sy - y0) / B
        qx, qy = dx / A, dy / B
        a = qx * qx + qy * qy
        b = px * qx + py * qy
        c = px * px + py * py - 1.0
        disc = b * b - a * c
        p += val * 2.0 * np.sqrt(np.maximum(disc, 0.0)) / a
    return p


def slice_jitter(cfg: Config, rng) -> np.ndarray:
    """[S][2] tumour offsets in mm: 0 for single-slice configs, U(-5,5) per slice otherwise."""
    if cfg.S == 1:
        return np.zeros((1, 2))
    return rng.uniform(-5.0, 5.0, size=(cfg.S, 2))


def make_inputs(cfg: Config, slices=None, phantom: bool = True) -> dict:
    """Seeded inputs of one configuration.

    Returns float64 arrays (callers cast):  phantom [S][N][L][L];  and, when cfg.V > 0,
    y, w [S][N][V][B] (noisy line integrals and the Sigma^-1 diagonal I0*exp(-pbar),
    Eq. 9), angles [N][V];  when cfg.sigma > 0, g = phantom + N(0, sigma^2).
    `slices` (iterable of slice indices) restricts what is built; the random stream is
    always advanced as for the full config so a sampled slice equals the full run's.
    phantom=False skips the rasterised phantom images (they consume no random numbers and the
    sinograms do not need them): the 64-slice batch of config 5 is built in seconds that way.
    """
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    jit = slice_jitter(cfg, rng)
    want = list(range(cfg.S)) if slices is None else list(slices)
    out = {"cfg": cfg, "slices": want}
    if phantom or cfg.sigma > 0:
        ph = np.zeros((len(want), cfg.N, cfg.L, cfg.L))
        for a, s in enumerate(want):
            for i in range(cfg.N):
                ph[a, i] = _raster(cfg, _ellipses(cfg, i, jit[s]))
        out["phantom"] = ph
    if cfg.V > 0:
        out["angles"] = view_angles(cfg.N, cfg.V)
    if cfg.V > 0 and cfg.I0 > 0:
        ang = out["angles"]
        y = np.zeros((len(want), cfg.N, cfg.V, cfg.B))
        w = np.zeros_like(y)
        pos = {s: a for a, s in enumerate(want)}
        for s in range(cfg.S):                       # noise drawn in array order, all slices
            if s not in pos and cfg.S > 1 and s > max(want):
                break
            for i in range(cfg.N):
                pbar = _line_integrals(cfg, _ellipses(cfg, i, jit[s]), ang[i])
                counts = rng.poisson(cfg.I0 * np.exp(-pbar)).astype(np.float64)
                if s in pos:
                    y[pos[s], i] = -np.log(np.maximum(counts, 1.0) / cfg.I0)
                    w[pos[s], i] = cfg.I0 * np.exp(-pbar)
        out["y"], out["w"] = y, w
    if cfg.sigma > 0:
        out["g"] = ph + rng.normal(0.0, cfg.sigma, size=ph.shape)
    return out


def geometry_kwargs(cfg: Config) -> dict:
    """Plain-number geometry of a config, to build either side's geometry object."""
    return dict(n_views=cfg.V, n_bins=cfg.B, sid_mm=cfg.sid, sdd_mm=cfg.sdd,
                bin_pitch_mm=cfg.pitch, bin_offset=0.0, pixel_mm=cfg.pix,
                angles_rad=view_angles(cfg.N, cfg.V))
