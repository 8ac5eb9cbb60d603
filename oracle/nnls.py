"""CPU oracle for the orbital-weight solve (Sect. 2.3).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module; it shares no code with the CUDA path.  numpy, fp64, written in the paper's order and notation:

  stack_system   Eq. 3 -> Eq. 4: U is the stack of the library matrices, each row divided by its tolerance
                 (0.01 m*_n for the density and surface-density rows, Delta h*_{m,n} for the Gauss-Hermite rows),
                 y the stacked targets divided the same way.
  bootstrap      y_b = y + xi_b: the targets perturbed by their uncertainties; the normal draws
                 xi are an INPUT (zero on the 3-D density rows, which "are not bootstrapped").
  objective      Q(w) of Eq. 3/4.
  admm_nnls      the ADMM iteration of PAPER.md:132: "solving the unconstrained quadratic problem with a linear
                 solver and enforcing the non-negative constraints by clipping negative orbit weights to zero.  A
                 vector that tracks the differences between the solution before and after the constraint is
                 recorded and reused at the next iteration".  The paper prints neither the penalty parameter, the
                 start nor the stopping rule: DESIGN.md reading R19 takes the scaled form of Boyd et al. (2011,
                 Sect. 3.1.1) with z^0 = u^0 = 0, a caller-given rho and a fixed iteration count.

Pins (tests/test_oracle_nnls.py): the converged iterate against scipy.optimize.nnls (Lawson-Hanson active set,
a different algorithm) on the augmented system, against exhaustive enumeration of the active sets on tiny
problems, the KKT conditions, the closed form for orthonormal columns, Q of Eq. 3 summed term by term.
"""
import numpy as np
import scipy.linalg


def stack_system(blocks, targets, sigmas, keep=None):
    """Eq. 3 -> Eq. 4.

    blocks   list of library matrices, each [n_orb][n_k] (row i = orbit i's contribution to the n_k cells of
             block k: m_{i,n}, Sigma_{i,n}, h_{m,i,n})
    targets  list of [n_k] observed values (m*_n, Sigma*_n, h*_{m,n})
    sigmas   list of [n_k] tolerances (0.01 m*_n, 0.01 Sigma*_n, Delta h*_{m,n}), all > 0
    keep     optional [n_orb] bool: orbits failing the Jacobi-drift cut contribute nothing
    Returns U [n_con][n_orb], y [n_con], sigma [n_con] with n_con = sum n_k.
    """
    n_orb = blocks[0].shape[0]
    U = np.concatenate([np.asarray(b, dtype=np.float64).reshape(n_orb, -1) for b in blocks], axis=1).T.copy()
    t = np.concatenate([np.asarray(v, dtype=np.float64).ravel() for v in targets])
    s = np.concatenate([np.asarray(v, dtype=np.float64).ravel() for v in sigmas])
    assert U.shape[0] == t.size == s.size and np.all(s > 0)
    U /= s[:, None]
    if keep is not None:
        U[:, ~np.asarray(keep, dtype=bool)] = 0.0
    return U, t / s, s


def bootstrap(y, xi):
    """bootstrap realisations of the (normalised) targets, y_b = y + xi_b.

    In units of the tolerance a perturbation "according to the measurement uncertainties" is a unit normal;
    xi [n_rhs][n_con] is drawn by the caller and is zero on the rows that are not bootstrapped."""
    return np.asarray(y, dtype=np.float64)[None, :] + np.asarray(xi, dtype=np.float64)


def reg_diagonal(n_orb, lam, wtilde=None):
    """d_i with regularisation term of Eq. 3 = 1/2 sum_i d_i w_i^2, i.e. d_i = 2 lambda / (N_orb wtilde_i^2).

    wtilde=None is Eq. 4 as printed ((lambda/N_orb) ||w||^2, i.e. wtilde_i = 1)."""
    wt = np.ones(n_orb) if wtilde is None else np.asarray(wtilde, dtype=np.float64)
    return 2.0 * lam / (n_orb * wt * wt)


def objective(U, y, w, lam, wtilde=None):
    """Q(w) of Eq. 4 with the regularisation of Eq. 3."""
    r = U @ w - y
    d = reg_diagonal(U.shape[1], lam, wtilde)
    return 0.5 * float(r @ r) + 0.5 * float(np.sum(d * w * w))


def admm_nnls(U, Y, lam, rho, n_iter, wtilde=None):
    """ADMM for min Q(w) s.t. w >= 0, one column of the result per right-hand side.

    U [n_con][n_orb], Y [n_rhs][n_con] (all realisations share U: PAPER.md:136).
    Returns w [n_rhs][n_orb] (the clipped iterate z^{n_iter}, feasible by construction) and
    resid [n_rhs][2] = (||x - z||_2, rho ||z - z_prev||_2) of the last iteration.
    """
    U = np.asarray(U, dtype=np.float64)
    Y = np.atleast_2d(np.asarray(Y, dtype=np.float64))
    n_orb = U.shape[1]
    d = reg_diagonal(n_orb, lam, wtilde)
    # the unconstrained quadratic problem: (U^T U + diag(d) + rho I) x = U^T y + rho (z - u)
    G = U.T @ U + np.diag(d + rho)
    chol = scipy.linalg.cho_factor(G, lower=True)
    q = U.T @ Y.T                       # [n_orb][n_rhs]
    z = np.zeros_like(q)
    u = np.zeros_like(q)
    resid = np.zeros((Y.shape[0], 2))
    for _ in range(int(n_iter)):
        x = scipy.linalg.cho_solve(chol, q + rho * (z - u))   # linear solve
        z_prev = z
        z = np.maximum(0.0, x + u)                             # clip negative weights to zero
        u = u + x - z                                          # the recorded difference, reused next iteration
        resid[:, 0] = np.sqrt(np.sum((x - z) ** 2, axis=0))
        resid[:, 1] = rho * np.sqrt(np.sum((z - z_prev) ** 2, axis=0))
    return z.T.copy(), resid


def chi2_blocks(U, y, w, block_sizes):
    """Per realisation b and block k: chi^2_{b,k} = sum over the block's rows of ((U w_b)_n - y_n)^2 -- the terms of Eq. 3
     evaluated against the UNPERTURBED data y (reading R20); Eq. 5 is the sum over the surface-density
    and Gauss-Hermite blocks, "excludes chi^2_dens".  U [n_con][n_orb], y [n_con], w [n_rhs][n_orb]."""
    w = np.atleast_2d(np.asarray(w, dtype=np.float64))
    res = w @ np.asarray(U, dtype=np.float64).T - np.asarray(y, dtype=np.float64)[None, :]
    out = np.zeros((w.shape[0], len(block_sizes)))
    o = 0
    for k, nk in enumerate(block_sizes):
        out[:, k] = np.sum(res[:, o:o + nk] ** 2, axis=1)
        o += nk
    return out


def marginal_chi2(chi2_b):
    """Eq. 6, which prints "ln[sum_b exp((chi2_min - chi2_b)/2)] + const": reading R20 takes the
    -2 ln of the bootstrap-averaged likelihood, chi2_model = chi2_min - 2 ln[(1/B) sum_b exp((chi2_min - chi2_b)/2)]
    (the same quantity up to the factor -2 and constants, with the sign that makes it a chi^2: equal chi2_b give chi2_b)."""
    c = np.asarray(chi2_b, dtype=np.float64)
    cmin = c.min()
    return float(cmin - 2.0 * np.log(np.mean(np.exp(0.5 * (cmin - c)))))
