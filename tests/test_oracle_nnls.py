"""Pins for the weight-solve oracle (oracle/nnls.py) against things other than itself:
scipy's Lawson-Hanson NNLS (a different algorithm), exhaustive enumeration of active sets, the KKT conditions,
the closed form for orthonormal columns, Eq. 3 summed term by term, and the ridge closed form."""
import itertools

import numpy as np
import pytest
import scipy.optimize

from oracle import nnls as onnls


def random_system(seed, n_con, n_orb, n_rhs=1, sparse=0.6):
    """A library-like system: non-negative entries, many zeros, targets from non-negative weights plus noise."""
    rng = np.random.default_rng(seed)
    U = rng.random((n_con, n_orb)) * (rng.random((n_con, n_orb)) > sparse)
    w_true = rng.random(n_orb) * (rng.random(n_orb) > 0.5)
    Y = (U @ w_true)[None, :] + 0.3 * rng.standard_normal((n_rhs, n_con))
    return U, Y


def augmented(U, lam, wtilde=None):
    """Q = 1/2 ||[U; diag(sqrt d)] w - [y; 0]||^2, the form a plain NNLS routine takes."""
    d = 2.0 * lam / (U.shape[1] * (np.ones(U.shape[1]) if wtilde is None else wtilde) ** 2)
    return np.vstack([U, np.diag(np.sqrt(d))])


@pytest.mark.parametrize("seed,n_con,n_orb,lam", [(1, 40, 25, 0.0), (2, 30, 45, 0.5), (3, 60, 60, 5.0)])
def test_converged_admm_equals_lawson_hanson(seed, n_con, n_orb, lam):
    U, Y = random_system(seed, n_con, n_orb, n_rhs=3)
    lam_eff = max(lam, 1e-3) if n_orb > n_con else lam   # keep the problem strictly convex
    w, resid = onnls.admm_nnls(U, Y, lam_eff, rho=2.0, n_iter=20000)
    A = augmented(U, lam_eff)
    for b in range(Y.shape[0]):
        ref, _ = scipy.optimize.nnls(A, np.concatenate([Y[b], np.zeros(n_orb)]), maxiter=10000)
        assert np.max(np.abs(w[b] - ref)) < 1e-7 * max(1.0, np.max(ref))
    assert np.all(resid < 1e-8)


def test_against_exhaustive_active_sets():
    """Tiny problems: the constrained minimum is the best feasible unconstrained solve over all supports."""
    for seed in range(6):
        U, Y = random_system(100 + seed, 7, 5, sparse=0.3)
        lam = 0.2
        d = onnls.reg_diagonal(5, lam)
        best, best_q = None, np.inf
        for r in range(6):
            for S in itertools.combinations(range(5), r):
                w = np.zeros(5)
                if S:
                    Us = U[:, S]
                    w[list(S)] = np.linalg.solve(Us.T @ Us + np.diag(d[list(S)]), Us.T @ Y[0])
                if np.all(w >= 0):
                    q = 0.5 * np.sum((U @ w - Y[0]) ** 2) + 0.5 * np.sum(d * w * w)   # Eq. 4 written out
                    if q < best_q:
                        best, best_q = w, q
        w, _ = onnls.admm_nnls(U, Y, lam, rho=1.0, n_iter=5000)
        assert np.max(np.abs(w[0] - best)) < 1e-9
        assert abs(onnls.objective(U, Y[0], w[0], lam) - best_q) < 1e-12


def test_kkt_conditions_and_feasibility_at_every_iteration_count():
    U, Y = random_system(7, 50, 35)
    wt = 0.5 + np.random.default_rng(8).random(35)
    lam = 0.7
    for n_iter in (1, 2, 10):
        w, _ = onnls.admm_nnls(U, Y, lam, 1.5, n_iter, wtilde=wt)
        assert np.all(w >= 0)                              # the clipped iterate is feasible from the first iteration
    w, _ = onnls.admm_nnls(U, Y, lam, 1.5, 20000, wtilde=wt)
    g = U.T @ (U @ w[0] - Y[0]) + 2 * lam / 35 * w[0] / wt ** 2   # grad Q from Eq. 3
    assert np.all(g > -1e-8)
    assert np.max(np.abs(g[w[0] > 1e-9])) < 1e-8
    assert np.all(w[0][g > 1e-6] == 0.0)


def test_orthonormal_columns_closed_form():
    """U^T U = I: the problem separates, w_i = max(0, (U^T y)_i) / (1 + d_i); and ADMM reaches it."""
    rng = np.random.default_rng(11)
    Q, _ = np.linalg.qr(rng.standard_normal((30, 12)))
    y = rng.standard_normal((2, 30))
    lam = 3.0
    w, _ = onnls.admm_nnls(Q, y, lam, rho=1.0, n_iter=400)
    expect = np.maximum(0.0, y @ Q) / (1.0 + 2 * lam / 12)
    assert np.max(np.abs(w - expect)) < 1e-12


def test_first_iterate_is_clipped_ridge_solution_and_positive_problem_is_ridge():
    """z^1 = max(0, (G + rho)^-1 U^T y) from z^0 = u^0 = 0; if the ridge solution is positive it is the answer."""
    rng = np.random.default_rng(5)
    U = rng.random((40, 6)) + np.vstack([np.eye(6) * 3] + [np.zeros((34, 6))])
    w_true = 1.0 + rng.random(6)
    y = (U @ w_true)[None, :]
    rho, lam = 0.8, 0.3
    w1, _ = onnls.admm_nnls(U, y, lam, rho, 1)
    x1 = np.linalg.lstsq(np.vstack([U, np.sqrt(2 * lam / 6 + rho) * np.eye(6)]), np.concatenate([y[0], np.zeros(6)]), rcond=None)[0]
    assert np.max(np.abs(w1[0] - np.maximum(0, x1))) < 1e-12
    w, _ = onnls.admm_nnls(U, y, lam, rho, 3000)
    ridge = np.linalg.lstsq(np.vstack([U, np.sqrt(2 * lam / 6) * np.eye(6)]), np.concatenate([y[0], np.zeros(6)]), rcond=None)[0]
    assert np.all(ridge > 0) and np.max(np.abs(w[0] - ridge)) < 1e-10


def test_stack_system_is_eq3_term_by_term():
    rng = np.random.default_rng(21)
    n_orb, n_dens, n_obs, n_gh = 9, 7, 5, 4
    m = rng.random((n_orb, n_dens)); S = rng.random((n_orb, n_obs)); h = rng.standard_normal((n_orb, n_gh, n_obs))
    m_t = rng.random(n_dens) + 0.5; S_t = rng.random(n_obs) + 0.5
    h_t = rng.standard_normal((n_gh, n_obs)); dh = 0.02 + 0.05 * rng.random((n_gh, n_obs))
    w = rng.random(n_orb); wt = np.full(n_orb, 1.0 / n_orb); lam = 0.4
    keep = np.ones(n_orb, bool); keep[3] = False
    U, y, s = onnls.stack_system([m, S, h.reshape(n_orb, -1)], [m_t, S_t, h_t], [0.01 * m_t, 0.01 * S_t, dh], keep=keep)
    # Eq. 3, the three chi^2 sums and the regularisation, with loops
    wk = np.where(keep, w, 0.0)
    Q = 0.0
    for n in range(n_dens):
        Q += 0.5 * ((sum(wk[i] * m[i, n] for i in range(n_orb)) - m_t[n]) / (0.01 * m_t[n])) ** 2
    for n in range(n_obs):
        Q += 0.5 * ((sum(wk[i] * S[i, n] for i in range(n_orb)) - S_t[n]) / (0.01 * S_t[n])) ** 2
    for mm in range(n_gh):
        for n in range(n_obs):
            Q += 0.5 * ((sum(wk[i] * h[i, mm, n] for i in range(n_orb)) - h_t[mm, n]) / dh[mm, n]) ** 2
    Q += lam / n_orb * sum((w[i] / wt[i]) ** 2 for i in range(n_orb))
    assert abs(onnls.objective(U, y, w, lam, wt) - Q) < 1e-9 * Q
    assert U.shape == (n_dens + n_obs + n_gh * n_obs, n_orb) and np.all(U[:, 3] == 0)


def test_bootstrap_and_shared_matrix():
    """only y changes between realisations; xi = 0 reproduces the unperturbed solve and every
    realisation equals its own single-rhs solve; a dropped orbit gets exactly zero weight."""
    U, Y = random_system(31, 35, 20)
    rng = np.random.default_rng(32)
    xi = rng.standard_normal((4, 35)); xi[0] = 0.0; xi[:, :10] = 0.0     # first 10 rows: 3-D density, not bootstrapped
    Yb = onnls.bootstrap(Y[0], xi)
    assert np.array_equal(Yb[0], Y[0]) and np.array_equal(Yb[:, :10], np.tile(Y[0, :10], (4, 1)))
    U[:, 4] = 0.0
    w, _ = onnls.admm_nnls(U, Yb, 0.1, 1.0, 300)
    for b in range(4):
        wb, _ = onnls.admm_nnls(U, Yb[b], 0.1, 1.0, 300)
        assert np.max(np.abs(wb[0] - w[b])) < 1e-12
    assert np.all(w[:, 4] == 0.0)


def test_regularisation_shrinks_weights_monotonically():
    U, Y = random_system(41, 30, 30)
    norms = [np.linalg.norm(onnls.admm_nnls(U, Y, lam, 1.0, 4000)[0]) for lam in (1e-3, 1e-1, 10.0, 1e3)]
    assert all(a > b for a, b in zip(norms, norms[1:]))


def test_chi2_blocks_and_marginalisation():
    """Eq. 5-6: block chi^2 add up to 2 (Q - regularisation) of Eq. 3/4; the marginalised chi^2 has the
    closed forms of a log-mean-exp: equal values -> that value, B = 1 -> the value, one dominant term -> chi2_min + 2 ln B,
    invariance under permutation, and it lies between chi2_min and chi2_min + 2 ln B."""
    U, Y = random_system(51, 30, 12, n_rhs=4)
    w = np.random.default_rng(52).random((4, 12))
    sizes = [7, 5, 18]
    c = onnls.chi2_blocks(U, Y[0], w, sizes)
    for b in range(4):
        q_noreg = onnls.objective(U, Y[0], w[b], 0.0)
        assert abs(c[b].sum() - 2 * q_noreg) < 1e-10 * q_noreg
        assert abs(c[b, 1] - sum((U[n] @ w[b] - Y[0, n]) ** 2 for n in range(7, 12))) < 1e-10
    assert abs(onnls.marginal_chi2([37.5] * 100) - 37.5) < 1e-12
    assert abs(onnls.marginal_chi2([12.0]) - 12.0) < 1e-12
    big = np.array([10.0] + [1e4] * 99)
    assert abs(onnls.marginal_chi2(big) - (10.0 + 2 * np.log(100))) < 1e-9
    vals = np.random.default_rng(53).random(100) * 30 + 400
    m = onnls.marginal_chi2(vals)
    assert vals.min() <= m <= vals.min() + 2 * np.log(100)
    assert abs(m - onnls.marginal_chi2(vals[::-1])) < 1e-12
    # two values a and a + d: chi2 = a - 2 ln((1 + exp(-d/2)) / 2)
    assert abs(onnls.marginal_chi2([50.0, 54.0]) - (50.0 - 2 * np.log(0.5 * (1 + np.exp(-2.0))))) < 1e-12
