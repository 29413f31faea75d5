"""Pins for the oracle's CGLS step (ref. 21 Hestenes-Stiefel) -- CPU only.

CGLS is characterised without its recurrences: after m steps from u0 the iterate minimises
||y_n - P_n u|| over u0 + K_m(P_n^T P_n, P_n^T r0).  The tests build that Krylov space and
the dense matrix by brute force and solve the small least-squares problems with numpy.
"""
import numpy as np

import oracle
from brute_force import dense_system_matrix

NY = NX = 8
V, B = 12, 18
SID, SDD, PITCH = 30.0, 50.0, 1.1


def setup(seed=0, weighted=True):
    rng = np.random.default_rng(seed)
    thetas = 2 * np.pi * (np.arange(V) + 0.3) / V
    g = oracle.Geometry(n_views=V, n_bins=B, sid_mm=SID, sdd_mm=SDD, bin_pitch_mm=PITCH,
                        angles_rad=thetas[None, :], pixel_mm=1.0)
    A = dense_system_matrix(SID, SDD, PITCH, B, thetas, NY, NX, 1.0)
    w = rng.uniform(0.5, 4.0, V * B) if weighted else None
    y = A @ rng.random(NY * NX) + 0.05 * rng.standard_normal(V * B)
    u0 = 0.1 * rng.random(NY * NX)
    return g, A, w, y, u0


def run(g, u0, y, w, m1):
    return oracle.cgls_step(g, u0.reshape(1, NY, NX), y.reshape(1, V, B),
                            None if w is None else w.reshape(1, V, B), m1).ravel()


def krylov_minimiser(An, yn, u0, m):
    r0 = yn - An @ u0
    M = An.T @ An
    basis = [An.T @ r0]
    for _ in range(m - 1):
        basis.append(M @ basis[-1])
    K, _ = np.linalg.qr(np.stack(basis, axis=1))        # orthonormalise (better conditioned)
    c, *_ = np.linalg.lstsq(An @ K, r0, rcond=None)
    return u0 + K @ c


def test_m_step_iterate_is_the_krylov_least_squares_minimiser():
    g, A, w, y, u0 = setup(1)
    sw = np.sqrt(w)
    An, yn = sw[:, None] * A, sw * y
    for m in (1, 2, 3, 5):
        got = run(g, u0, y, w, m)
        want = krylov_minimiser(An, yn, u0, m)
        assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want), m


def test_zero_steps_returns_input_and_no_clip():
    g, A, w, y, u0 = setup(2)
    assert np.array_equal(run(g, u0 - 0.2, y, w, 0), u0 - 0.2)     # negatives survive: no clip in CGLS
    assert (run(g, u0, -y, w, 2) < 0).any()


def test_many_steps_reach_the_weighted_least_squares_solution():
    g, A, w, y, u0 = setup(3)
    sw = np.sqrt(w)
    want, *_ = np.linalg.lstsq(sw[:, None] * A, sw * y, rcond=None)
    assert np.linalg.matrix_rank(A) == NY * NX
    got = run(g, u0, y, w, NY * NX)          # exact after n steps in exact arithmetic
    assert np.linalg.norm(got - want) <= 1e-9 * np.linalg.norm(want)


def test_residual_norm_is_non_increasing():
    g, A, w, y, u0 = setup(4)
    sw = np.sqrt(w)
    res = [np.linalg.norm(sw * (y - A @ run(g, u0, y, w, m))) for m in range(8)]
    assert all(res[m + 1] <= res[m] * (1 + 1e-12) for m in range(7))
    assert res[7] < 0.5 * res[0]


def test_iterates_invariant_to_scaling_of_the_weights_and_unweighted_is_w_equal_one():
    g, A, w, y, u0 = setup(5)
    a = run(g, u0, y, w, 3)
    b = run(g, u0, y, 7.5 * w, 3)
    assert np.linalg.norm(a - b) <= 1e-11 * np.linalg.norm(a)
    c = run(g, u0, y, None, 3)
    d = run(g, u0, y, np.ones(V * B), 3)
    assert np.array_equal(c, d)


def test_start_at_solution_or_zero_data_stays_put():
    g, A, w, y, u0 = setup(6)
    sw = np.sqrt(w)
    sol, *_ = np.linalg.lstsq(sw[:, None] * A, sw * y, rcond=None)
    got = run(g, sol, y, w, 3)
    assert np.linalg.norm(got - sol) <= 1e-9 * np.linalg.norm(sol)
    z = run(g, np.zeros(NY * NX), np.zeros(V * B), w, 3)               # breakdown guard: gamma = 0
    assert np.array_equal(z, np.zeros(NY * NX))


def test_phases_are_independent_problems_with_their_own_angles():
    rng = np.random.default_rng(7)
    th = np.stack([2 * np.pi * (np.arange(V) + 0.3) / V, 2 * np.pi * (np.arange(V) + 0.8) / V])
    g2 = oracle.Geometry(n_views=V, n_bins=B, sid_mm=SID, sdd_mm=SDD, bin_pitch_mm=PITCH,
                         angles_rad=th, pixel_mm=1.0)
    f = rng.random((2, NY, NX)); y = rng.random((2, V, B)); w = rng.uniform(1, 2, (2, V, B))
    both = oracle.cgls_step(g2, f, y, w, 3)
    for i in range(2):
        gi = oracle.Geometry(n_views=V, n_bins=B, sid_mm=SID, sdd_mm=SDD, bin_pitch_mm=PITCH,
                             angles_rad=th[i:i + 1], pixel_mm=1.0)
        one = oracle.cgls_step(gi, f[i:i + 1], y[i:i + 1], w[i:i + 1], 3)
        assert np.array_equal(both[i], one[0])
