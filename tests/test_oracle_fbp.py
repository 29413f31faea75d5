"""Pins of the FBP-initialisation oracle (oracle/fbp.py) against what the mathematics fixes:
the analytic sinogram of a disc must come back as the disc at its true value (pins D, dgamma, the 1/2 of
the full scan and the ramp-filter constants), the view weights must be the trapezoid rule (repeated and
unequally spaced angles), linearity, the static ellipse phantom's closed-form sinogram must reconstruct to
the phantom, and the ramp filter must annihilate constants in the continuum sense (DC gain 0)."""
import numpy as np

import oracle
from oracle import fbp
import workloads


def disc_sino(geom, N, R, mu, cx=0.0, cy=0.0):
    """Closed-form line integrals of a disc (radius R, value mu, centre (cx, cy)) along every pencil ray."""
    ang = geom.angles_rad
    B = geom.n_bins
    gam = (np.arange(B) - 0.5 * (B - 1) + geom.bin_offset) * geom.bin_pitch_mm / geom.sdd_mm
    y = np.zeros(ang.shape + (B,))
    for i in range(ang.shape[0]):
        for v in range(ang.shape[1]):
            b = ang[i, v]
            sx, sy = geom.sid_mm * np.cos(b), geom.sid_mm * np.sin(b)
            dx, dy = -np.cos(b + gam), -np.sin(b + gam)
            t = (cx - sx) * dy - (cy - sy) * dx          # signed distance of the centre from each ray
            y[i, v] = 2.0 * mu * np.sqrt(np.maximum(R * R - t * t, 0.0))
    return y


def geometry(N=2, V=180, B=257, L=64):
    ang = workloads.view_angles(N, V)
    return oracle.Geometry(n_views=V, n_bins=B, sid_mm=300.0, sdd_mm=500.0, bin_pitch_mm=0.5, angles_rad=ang), L


def test_view_weights_are_the_trapezoid_rule():
    ang = workloads.view_angles(3, 8)                    # 24 equally spaced angles over 2 pi, interleaved phases
    w = fbp.view_weights(ang)
    assert np.allclose(w, 2 * np.pi / 24) and np.isclose(w.sum(), 2 * np.pi)
    rng = np.random.default_rng(0)
    a2 = np.sort(rng.uniform(0, 2 * np.pi, 10)).reshape(2, 5)
    w2 = fbp.view_weights(a2)
    flat = a2.ravel()
    assert np.isclose(w2.sum(), 2 * np.pi)
    assert np.isclose(w2.ravel()[3], 0.5 * (flat[4] - flat[2]))
    assert np.isclose(w2.ravel()[0], 0.5 * (flat[1] - (flat[-1] - 2 * np.pi)))
    # a repeated angle shares its interval: the two copies together weigh what the single one did
    a3 = np.array([[0.0, 1.0, 1.0, 2.5]])
    w3 = fbp.view_weights(a3)
    w1 = fbp.view_weights(np.array([[0.0, 1.0, 2.5]]))
    assert np.isclose(w3[0, 1] + w3[0, 2], w1[0, 1]) and np.isclose(w3.sum(), 2 * np.pi)


def test_ramp_kernel_values_and_zero_dc_gain():
    dg = 0.002
    g = fbp.ramp_kernel(5, dg)                           # k = -4..4
    assert np.isclose(g[4], 1 / (8 * dg * dg))
    assert g[3] == g[5] and np.isclose(g[5], -1 / (2 * np.pi ** 2 * np.sin(dg) ** 2))
    assert g[2] == 0.0 and g[6] == 0.0
    big = fbp.ramp_kernel(4001, 1e-4)
    assert abs(big.sum()) < 2e-3 * big[4000]             # sum_k g(k) -> 0: the ramp filter removes DC


def test_disc_comes_back_at_its_value():
    geom, L = geometry()
    mu, R = 0.02, 18.0
    y = disc_sino(geom, 2, R, mu)
    f = fbp.fbp_init(geom, y, L, L)
    assert np.array_equal(f[0], f[1])                    # every phase gets the same image
    X = (np.arange(L) - 0.5 * (L - 1))
    rr = np.hypot(*np.meshgrid(X, X))
    inside, outside = rr < R - 2.5, (rr > R + 2.5) & (rr < 30)
    assert abs(f[0][inside].mean() / mu - 1.0) < 5e-3
    assert np.abs(f[0][inside] / mu - 1.0).max() < 3e-2
    assert np.abs(f[0][outside]).max() < 3e-2 * mu
    # an off-centre disc pins the sign of gamma and the orientation of the axes
    y2 = disc_sino(geom, 2, 6.0, mu, cx=12.0, cy=-7.0)
    f2 = fbp.fbp_init(geom, y2, L, L)[0]
    m = f2 > 0.5 * mu                                    # centroid of the reconstructed disc
    XX, YY = np.meshgrid(X, X)
    assert abs(XX[m].mean() - 12.0) < 0.3 and abs(YY[m].mean() + 7.0) < 0.3
    d2 = np.hypot(*np.meshgrid(X - 12.0, X + 7.0))
    assert abs(f2[d2 < 3.5].mean() / mu - 1.0) < 1e-2 and np.abs(f2[(d2 > 9) & (rr < 30)]).max() < 6e-2 * mu


def test_linear_and_independent_of_view_duplication_and_phase_order():
    geom, L = geometry(N=2, V=60, B=129, L=32)
    rng = np.random.default_rng(3)
    y1, y2 = rng.random((2, 60, 129)), rng.random((2, 60, 129))
    f1, f2 = fbp.fbp_init(geom, y1, L, L), fbp.fbp_init(geom, y2, L, L)
    f12 = fbp.fbp_init(geom, 2.0 * y1 - 0.5 * y2, L, L)
    assert np.allclose(f12, 2.0 * f1 - 0.5 * f2, rtol=1e-10, atol=1e-12)
    # swapping the phases (and their angles) changes nothing
    g2 = oracle.Geometry(60, 129, 300.0, 500.0, 0.5, geom.angles_rad[::-1].copy())
    assert np.allclose(fbp.fbp_init(g2, y1[::-1].copy(), L, L), f1, rtol=1e-10, atol=1e-12)
    # measuring every view twice (same angle, same data) changes nothing either
    g3 = oracle.Geometry(120, 129, 300.0, 500.0, 0.5, np.repeat(geom.angles_rad, 2, axis=1))
    assert np.allclose(fbp.fbp_init(g3, np.repeat(y1, 2, axis=1), L, L), f1, rtol=1e-9, atol=1e-11)


def test_static_phantom_from_its_closed_form_sinogram():
    cfg = workloads.Config("fbp", L=64, N=2, V=180, B=192, pitch=1.0, sid=400.0, sdd=800.0, I0=0.0)
    ells = workloads._ellipses(cfg, 0, np.zeros(2))
    ang = workloads.view_angles(cfg.N, cfg.V)
    y = np.stack([workloads._line_integrals(cfg, ells, ang[i]) for i in range(cfg.N)])
    geom = oracle.Geometry(**workloads.geometry_kwargs(cfg))
    f = fbp.fbp_init(geom, y, cfg.L, cfg.L)[0]
    ph = workloads._raster(cfg, ells)
    assert np.linalg.norm(f - ph) / np.linalg.norm(ph) < 0.12     # edges ring, plateaus agree
    body = ph == ph.max()
    assert abs(f[body].mean() / ph.max() - 1.0) < 1e-2
