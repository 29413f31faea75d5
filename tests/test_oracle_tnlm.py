"""Pins for the oracle's TNLM half: weights Eq.(3)/(8), Gauss-Jacobi Eq.(7), clip
 -- CPU only, no CUDA."""
import numpy as np
import pytest

import oracle
from brute_force import J_unrestricted, gauss_jacobi_unrestricted, weights_unrestricted


def rand_g(N, ny, nx, seed, scale=0.02):
    return scale * np.random.default_rng(seed).random((N, ny, nx))


def test_matches_window_free_brute_force_on_8x8():
    # PAPER.md:L204 first half: every pixel y of the neighbour phase is a candidate.  A window
    # of side >= 2L-1 must reproduce that definition exactly (BASELINE north_star pin).
    for N, patch, m2 in ((3, 3, 1), (4, 5, 2), (2, 3, 2), (1, 3, 1)):
        g = rand_g(N, 8, 8, 10 + N)
        g[0, 2, 3] = -0.004                                     # something for the clip to do
        want = gauss_jacobi_unrestricted(g, patch, 0.01, 0.3, m2)
        got = oracle.regularize_step(g, 15, patch, 0.01, 0.3, m2)
        assert np.abs(got - want).max() < 1e-13, (N, patch, m2)
        assert (want == 0).any()


def test_window_restricts_candidates_and_matches_renormalised_brute_force():
    # With a W x W window the weights are the unrestricted ones restricted to the window and
    # re-normalised (Z sums over the window, PAPER.md:L94 + L204).
    g = rand_g(3, 8, 8, 3)
    W, d, h = 5, 3, 0.012
    full = weights_unrestricted(g[1], g[2], d, h)
    for x in ((0, 0), (4, 3), (7, 6), (2, 7)):
        om = oracle.weights_pixel(g[1], g[2], W, d, h, x)
        want = np.zeros((W, W))
        for dr in range(-2, 3):
            for dc in range(-2, 3):
                yr, yc = x[0] + dr, x[1] + dc
                if 0 <= yr < 8 and 0 <= yc < 8:
                    want[dr + 2, dc + 2] = full[x[0], x[1], yr, yc]
        want /= want.sum()
        assert np.abs(om - want).max() < 1e-13
        assert abs(om.sum() - 1.0) < 1e-14                      # sum_y omega = 1 (L94)


def test_raw_weight_symmetry():
    # omega_{i,j}(x,y) and omega_{j,i}(y,x) are the same before normalisation.
    g = rand_g(2, 9, 11, 4)
    rng = np.random.default_rng(0)
    for _ in range(50):
        x = (int(rng.integers(0, 9)), int(rng.integers(0, 11)))
        y = (int(rng.integers(0, 9)), int(rng.integers(0, 11)))
        a = oracle.raw_weight(g[0], g[1], 5, 0.02, x, y)
        b = oracle.raw_weight(g[1], g[0], 5, 0.02, y, x)
        assert a == b
        assert 0 < a <= 1


def test_raw_weight_value_hand_derived():
    # two 3x3 images, d=3 at the centre: D = sum of squared differences of all 9 pixels.
    gi = np.arange(9, dtype=float).reshape(3, 3) * 0.01
    gj = gi + 0.002
    want = np.exp(-9 * 0.002 ** 2 / 0.01 ** 2)
    assert abs(oracle.raw_weight(gi, gj, 3, 0.01, (1, 1), (1, 1)) - want) < 1e-15
    # at the corner only the 2x2 in-image part of the patch differs (zero extension)
    want_c = np.exp(-4 * 0.002 ** 2 / 0.01 ** 2)
    assert abs(oracle.raw_weight(gi, gj, 3, 0.01, (0, 0), (0, 0)) - want_c) < 1e-15


def test_scaling_g_and_h_together_leaves_weights_unchanged():
    g = rand_g(2, 8, 8, 5)
    a = oracle.weights_pixel(g[0], g[1], 5, 3, 0.01, (3, 4))
    b = oracle.weights_pixel(3.0 * g[0], 3.0 * g[1], 5, 3, 0.03, (3, 4))
    assert np.abs(a - b).max() < 1e-14


def test_constant_image_is_a_fixed_point():
    g = np.full((4, 10, 12), 0.0173)
    out = oracle.regularize_step(g, 5, 3, 0.01, 0.7, 3)
    assert np.abs(out - g).max() < 1e-16


def test_window_one_is_pointwise_closed_form():
    g = rand_g(5, 6, 7, 6)
    mu = 0.4
    u = g.copy()
    for _ in range(3):
        u = g / (1 + mu) + mu / (2 * mu + 2) * (np.roll(u, 1, axis=0) + np.roll(u, -1, axis=0))
    got = oracle.regularize_step(g, 1, 3, 0.01, mu, 3)
    assert np.abs(got - np.maximum(u, 0)).max() < 1e-15


def test_huge_h_gives_box_mean_over_in_image_window():
    from scipy.ndimage import uniform_filter
    g = rand_g(3, 12, 9, 7)
    W, mu = 5, 0.25
    ones = np.ones((12, 9))
    cnt = uniform_filter(ones, W, mode="constant") * W * W
    def boxmean(im):
        return uniform_filter(im, W, mode="constant") * W * W / cnt
    want = np.stack([g[i] / (1 + mu) + mu / (2 * mu + 2) * (boxmean(g[(i - 1) % 3]) + boxmean(g[(i + 1) % 3]))
                     for i in range(3)])
    got = oracle.regularize_step(g, W, 3, 1e6, mu, 1)
    assert np.abs(got - want).max() < 1e-12


def test_tiny_h_with_translated_phases_reproduces_g_in_the_interior():
    # g_{i+1}(x) = g_i(x - s): the only matching candidate of x in phase i+1 is x + s, in phase
    # i-1 it is x - s, so Eq.(7) returns g_i(x)/(1+mu) + mu/(2mu+2)*2*g_i(x) = g_i(x).
    # Pins the sign of delta, where u_j is read, and which neighbour is which.
    rng = np.random.default_rng(8)
    base = 0.02 * rng.random((30, 30))
    s = (2, -1)
    g = np.stack([np.roll(base, (-s[0], -s[1]), (0, 1)), base, np.roll(base, s, (0, 1))])
    got = oracle.regularize_step(g, 7, 3, 1e-4, 0.5, 1)
    interior = (slice(8, 22), slice(8, 22))
    assert np.abs(got[1][interior] - g[1][interior]).max() < 1e-12
    # and a wrong neighbour assignment would not: phase 0's "previous" phase is phase 2 (cyclic)
    w = oracle.weights_pixel(g[1], g[2], 7, 3, 1e-4, (15, 15))
    assert w[3 + s[0], 3 + s[1]] > 0.999999


def test_mu_zero_returns_clipped_g_exactly():
    g = rand_g(3, 8, 8, 9) - 0.005
    assert np.array_equal(oracle.regularize_step(g, 5, 3, 0.01, 0.0, 2), np.maximum(g, 0))
    assert np.array_equal(oracle.regularize_step(g, 5, 3, 0.01, 0.3, 0), np.maximum(g, 0))


def test_output_is_a_convex_combination_and_sweeps_contract():
    g = rand_g(4, 10, 10, 12)
    mu, W = 0.6, 5
    u1 = oracle.regularize_step(g, W, 3, 0.01, mu, 1)
    assert u1.min() >= g.min() - 1e-15 and u1.max() <= g.max() + 1e-15
    # ||u^{m+1}-u^m||_inf <= mu/(1+mu) ||u^m-u^{m-1}||_inf (row sums of the Jacobi matrix; the
    # bound behind "converges for any mu_hat > 0").  g > 0 so the clip is idle.
    us = [g] + [oracle.regularize_step(g, W, 3, 0.01, mu, m) for m in (1, 2, 3, 4)]
    d = [np.abs(us[m + 1] - us[m]).max() for m in range(4)]
    for m in range(3):
        assert d[m + 1] <= mu / (1 + mu) * d[m] * (1 + 1e-12)


def test_softmax_does_not_underflow_for_tiny_h():
    g = rand_g(3, 8, 8, 13, scale=1.0)
    out = oracle.regularize_step(g, 5, 3, 1e-3, 0.5, 1)          # every D/h^2 >> 745
    assert np.isfinite(out).all()


def test_sampled_sweep_entry_point_agrees_with_full_sweep():
    g = rand_g(3, 9, 9, 14)
    u = oracle.regularize_step(g, 5, 3, 0.01, 0.3, 1)            # g > 0: no clip, u = sweep 1
    pix = np.random.default_rng(1).integers(0, g.size, 30)
    two = oracle.regularize_step(g, 5, 3, 0.01, 0.3, 2).ravel()[pix]
    assert np.abs(oracle.gj_sweep_pixels(g, u, 5, 3, 0.01, 0.3, pix) - two).max() < 1e-15


def test_cost_terms_against_brute_force():
    # Eq.(2) J with window-free weights, and the data term of Eq.(1) with a dense matrix.
    from brute_force import dense_system_matrix
    rng = np.random.default_rng(15)
    N, L, V, B = 3, 6, 5, 9
    f = 0.02 * rng.random((N, L, L)); gref = 0.02 * rng.random((N, L, L))
    th = 2 * np.pi * (np.arange(V)[None, :] + np.arange(N)[:, None] / N + 0.2) / V
    geom = oracle.Geometry(n_views=V, n_bins=B, sid_mm=25.0, sdd_mm=40.0, bin_pitch_mm=1.0, angles_rad=th)
    y = rng.random((N, V, B)); w = rng.uniform(1, 3, (N, V, B))
    data, reg = oracle.cost(geom, f, gref, y, w, 11, 3, 0.015)
    want_reg = sum(J_unrestricted(f[i], f[(i + s) % N], gref[i], gref[(i + s) % N], 3, 0.015)
                   for i in range(N) for s in (-1, 1))
    want_data = 0.0
    for i in range(N):
        A = dense_system_matrix(25.0, 40.0, 1.0, B, th[i], L, L, 1.0)
        e = A @ f[i].ravel() - y[i].ravel()
        want_data += float(e @ (w[i].ravel() * e))
    assert abs(reg - want_reg) < 1e-12 * want_reg
    assert abs(data - want_data) < 1e-11 * want_data
