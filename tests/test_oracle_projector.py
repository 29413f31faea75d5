"""Pins for the oracle's P and P^T -- CPU only.

Each test checks the oracle against something the paper or the mathematics fixes, computed
WITHOUT the oracle: chords from edge crossings, a brute-force dense matrix, the analytic
Radon transform of a disc/ellipse, and the symmetries of the scan geometry.
"""
import numpy as np
import pytest

import oracle
import workloads
from brute_force import chord_by_edges, dense_system_matrix, pixel_box, ray


def geom(V, B, sid=200.0, sdd=350.0, pitch=1.5, N=1, interleave=True, off=0.0):
    ang = workloads.view_angles(N, V) if interleave else np.tile(2 * np.pi * np.arange(V) / V, (N, 1))
    return oracle.Geometry(n_views=V, n_bins=B, sid_mm=sid, sdd_mm=sdd, bin_pitch_mm=pitch,
                           angles_rad=ang, bin_offset=off, pixel_mm=1.0)


def test_all_ones_image_gives_chord_through_image_rectangle():
    # (P 1)[v,k] = length of the ray inside the whole L x L rectangle: pins "no gaps, no
    # double counting" of the per-pixel lengths.
    ny, nx = 12, 20
    g = geom(V=17, B=34, pitch=1.1)
    p = oracle.project(g, np.ones((1, ny, nx)))[0]
    for v in range(g.n_views):
        for k in range(g.n_bins):
            s, d = ray(g.sid_mm, g.sdd_mm, g.bin_pitch_mm, g.n_bins, g.angles_rad[0, v], k)
            want = chord_by_edges(s, d, -nx / 2, nx / 2, -ny / 2, ny / 2)
            assert abs(p[v, k] - want) < 1e-10, (v, k, p[v, k], want)


def test_non_square_pixel_size_and_bin_offset():
    ny, nx, pix = 9, 7, 0.8
    g = geom(V=11, B=21, pitch=0.9, off=0.3)
    g.pixel_mm = pix
    p = oracle.project(g, np.ones((1, ny, nx)))[0]
    for v in range(g.n_views):
        for k in range(g.n_bins):
            gam = (k - 0.5 * (g.n_bins - 1) + 0.3) * g.bin_pitch_mm / g.sdd_mm
            th = g.angles_rad[0, v]
            s = np.array([g.sid_mm * np.cos(th), g.sid_mm * np.sin(th)])
            d = -np.array([np.cos(th + gam), np.sin(th + gam)])
            want = chord_by_edges(s, d, -nx * pix / 2, nx * pix / 2, -ny * pix / 2, ny * pix / 2)
            assert abs(p[v, k] - want) < 1e-10


def test_dense_matrix_rows_and_columns_match_brute_force():
    # Column p of P (project the unit image e_p) and row q of P^T... both must equal the
    # brute-force matrix of per-(ray,pixel) chords; pins pixel indexing (r<->Y, c<->X),
    # bin/view ordering, and P^T = transpose of P entry by entry.
    ny, nx, V, B = 6, 5, 7, 12
    g = geom(V=V, B=B, sid=40.0, sdd=70.0, pitch=1.3)
    A = dense_system_matrix(g.sid_mm, g.sdd_mm, g.bin_pitch_mm, B, g.angles_rad[0], ny, nx, 1.0)
    cols = np.zeros_like(A)
    for p in range(ny * nx):
        e = np.zeros(ny * nx); e[p] = 1.0
        cols[:, p] = oracle.project(g, e.reshape(1, ny, nx)).ravel()
    rows = np.zeros_like(A)
    for q in range(V * B):
        e = np.zeros(V * B); e[q] = 1.0
        rows[q, :] = oracle.backproject(g, e.reshape(1, V, B), nx, ny).ravel()
    assert np.abs(cols - A).max() < 1e-10
    assert np.abs(rows - A).max() < 1e-10
    assert (A > 0).sum() > 100


def test_adjoint_identity_random():
    # <P f, g> = <f, P^T g>  (BASELINE north_star)
    rng = np.random.default_rng(5)
    N, L, V, B = 3, 24, 20, 40
    g = geom(V=V, B=B, N=N, sid=120.0, sdd=200.0)
    f = rng.standard_normal((N, L, L))
    s = rng.standard_normal((N, V, B))
    lhs = float((oracle.project(g, f) * s).sum())
    rhs = float((f * oracle.backproject(g, s, L, L)).sum())
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), 1.0)


def test_centred_disc_matches_analytic_radon():
    # Disc radius R value c at the isocentre: line integral 2c sqrt(R^2 - t^2), t = SID sin(gam).
    # Pins SID, the arc-detector fan angle gam_k = (k-(B-1)/2) pitch/SDD, and the mm scale.
    L, R, c0 = 256, 40.0, 0.02
    cfg = workloads.Config("disc", L=L, N=1, V=8, B=120, pitch=2.0, sid=300.0, sdd=500.0, pix=0.5)
    img = workloads._raster(cfg, [(0.0, 0.0, R, R, c0)], sub=8)
    g = oracle.Geometry(**workloads.geometry_kwargs(cfg))
    p = oracle.project(g, img[None])[0]
    k = np.arange(cfg.B)
    t = cfg.sid * np.sin((k - 0.5 * (cfg.B - 1)) * cfg.pitch / cfg.sdd)
    want = 2 * c0 * np.sqrt(np.maximum(R * R - t * t, 0.0))
    for v in range(cfg.V):
        assert np.linalg.norm(p[v] - want) / np.linalg.norm(want) < 8e-3
    assert want.max() > 1.5  # the disc is actually seen


def test_offcentre_ellipse_matches_analytic_and_converges_with_resolution():
    # Off-centre ellipse: pins the source position S = SID (cos th, sin th), the sign of the
    # ray direction and the view ordering against the closed-form ellipse chord.
    errs = []
    for L, pix in ((128, 1.0), (256, 0.5)):
        cfg = workloads.Config("ell", L=L, N=2, V=12, B=90, pitch=2.5, sid=300.0, sdd=500.0, pix=pix)
        ell = [(17.0, -23.0, 30.0, 18.0, 0.02), (-20.0, 25.0, 10.0, 14.0, 0.01)]
        img = np.stack([workloads._raster(cfg, ell, sub=8)] * 2)
        g = oracle.Geometry(**workloads.geometry_kwargs(cfg))
        p = oracle.project(g, img)
        want = np.stack([workloads._line_integrals(cfg, ell, g.angles_rad[i]) for i in range(2)])
        errs.append(np.linalg.norm(p - want) / np.linalg.norm(want))
    assert errs[1] < 0.01 and errs[1] < 0.75 * errs[0], errs


def test_rotation_by_90_degrees_shifts_views_and_mirror_reverses_bins():
    rng = np.random.default_rng(11)
    L, V, B = 16, 8, 32
    g = geom(V=V, B=B, sid=60.0, sdd=100.0, pitch=1.2, interleave=False)
    f = rng.random((L, L))
    p = oracle.project(g, f[None])[0]
    # object rotated by +90 deg: f'(X,Y) = f(Y,-X)  <=>  f'[r,c] = f[L-1-c, r]
    frot = np.zeros_like(f)
    for r in range(L):
        for c in range(L):
            frot[r, c] = f[L - 1 - c, r]
    prot = oracle.project(g, frot[None])[0]
    assert np.abs(prot - np.roll(p, V // 4, axis=0)).max() < 1e-10
    # mirror Y -> -Y: theta -> -theta, gam -> -gam
    pm = oracle.project(g, f[::-1, :][None].copy())[0]
    want = p[(-np.arange(V)) % V][:, ::-1]
    assert np.abs(pm - want).max() < 1e-10


def test_hand_derived_rays():
    # theta = pi, centre bin (gam = 0): the ray runs along Y = 0 in +X through the middle
    # row of an odd image -> sum of that row times the pixel size.
    L = 5
    f = np.arange(L * L, dtype=float).reshape(L, L)
    g = oracle.Geometry(n_views=2, n_bins=3, sid_mm=50.0, sdd_mm=80.0, bin_pitch_mm=1.0,
                        angles_rad=np.array([[np.pi, 1.25 * np.pi]]), pixel_mm=2.0)
    p = oracle.project(g, f[None])[0]
    assert abs(p[0, 1] - 2.0 * f[2].sum()) < 1e-9
    # theta = 5pi/4: ray along the main diagonal X = Y -> sqrt(2)*pix*trace.
    assert abs(p[1, 1] - np.sqrt(2.0) * 2.0 * np.trace(f)) < 1e-9


def test_sampled_entry_points_agree_with_full_operators():
    rng = np.random.default_rng(2)
    N, L, V, B = 2, 20, 9, 30
    g = geom(V=V, B=B, N=N, sid=90.0, sdd=150.0)
    f = rng.random((N, L, L)); s = rng.random((N, V, B))
    rays = rng.integers(0, N * V * B, 40)
    pix = rng.integers(0, N * L * L, 40)
    assert np.abs(oracle.project_rays(g, f, rays) - oracle.project(g, f).ravel()[rays]).max() < 1e-12
    full = oracle.backproject(g, s, L, L).ravel()[pix]
    assert np.abs(oracle.backproject_pixels(g, s, L, L, pix) - full).max() < 1e-11


@pytest.mark.parametrize("cfg_id", [1, 3])
def test_config_geometry_field_of_view(cfg_id):
    # BASELINE configs: the fan covers the inscribed circle (cfg 1: 64 mm, cfg 3: ~488 mm).
    cfg = workloads.config(cfg_id)
    half_fan = 0.5 * cfg.B * cfg.pitch / cfg.sdd
    fov = 2 * cfg.sid * np.sin(half_fan)
    assert fov > (63.9 if cfg_id == 1 else 480.0)
