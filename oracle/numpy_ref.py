"""Independent numpy statement of the oracle's definitions -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A second, vectorised write-up of what oracle/birkhoff4_oracle.c computes, using library routines
(scipy logsumexp, numpy pinv) where the C file writes loops.  The tests cross-check the two and pin
both against what the paper and the mathematics fix.  Never imported by paper_2606_07574_b200.
"""
import numpy as np
from scipy.special import logsumexp


def marginal_err(T):
    """Err(T)."""
    T = np.asarray(T, np.float64).reshape(-1, 4, 4)
    return np.abs(T.sum(2) - 1).sum(1) + np.abs(T.sum(1) - 1).sum(1)


def forward_sinkhorn(H, tol=1e-14, max_sweeps=20000):
    """Log-domain Sinkhorn-Knopp (eq. (2) PAPER.md:76 via (5),(6),(7) PAPER.md:103-113, eta=1, a=b=1).
    Returns P, Err(P), sweeps.  Runs every matrix until the whole batch is below tol (small B only)."""
    H = np.asarray(H, np.float64).reshape(-1, 4, 4)
    b = np.zeros((H.shape[0], 1, 4))
    k = 0
    while True:
        a = -logsumexp(H + b, axis=2, keepdims=True)      # alpha*(beta), eq. (5)
        P = np.exp(a + H + b)                             # primal recovery PAPER.md:99
        e = marginal_err(P)
        if not (e.max() > tol) or k >= max_sweeps:
            return P, e, k
        b = -logsumexp(H + a, axis=1, keepdims=True)      # beta*(alpha), eq. (6)
        k += 1


def kkt_matrix(P):
    """[diag(r) P; P^T diag(c)] for each matrix: the Hessian of -L of the dual (4)."""
    P = np.asarray(P, np.float64).reshape(-1, 4, 4)
    B = P.shape[0]
    K = np.zeros((B, 8, 8))
    idx = np.arange(4)
    K[:, idx, idx] = P.sum(2)
    K[:, 4 + idx, 4 + idx] = P.sum(1)
    K[:, :4, 4:] = P
    K[:, 4:, :4] = P.transpose(0, 2, 1)
    return K


def backward_pinv(P, G, rcond=1e-13):
    """dH_ij = P_ij (G_ij - v_i - w_j), [v;w] = K^+ [(GoP)1; (GoP)^T 1]   (PAPER.md:527-563 ungauged).
    Valid for well-scaled logits only (|H| of a few units): LAPACK's eigen-solver loses the small eigenvalues of K
    that the C oracle's Jacobi sweep keeps, and at N(0,10^2) and above this write-up is off by up to 1e-3.  The
    tests use it at s <= 3; at s >= 10 the value pin is an 80-digit solve (tests/test_oracle_backward.py)."""
    P = np.asarray(P, np.float64).reshape(-1, 4, 4)
    G = np.asarray(G, np.float64).reshape(-1, 4, 4)
    Gam = G * P
    rhs = np.concatenate([Gam.sum(2), Gam.sum(1)], axis=1)[..., None]
    y = (np.linalg.pinv(kkt_matrix(P), rcond=rcond, hermitian=True) @ rhs)[..., 0]
    return P * (G - y[:, :4, None] - y[:, None, 4:])


def backward_finite_difference(forward_fn, H, G, eps=1e-6):
    """dH_kl = sum_ij G_ij dP_ij/dH_kl by central differences of `forward_fn` (definition of derivative)."""
    H = np.asarray(H, np.float64).reshape(-1, 4, 4)
    G = np.asarray(G, np.float64).reshape(-1, 4, 4)
    dH = np.zeros_like(H)
    for k in range(4):
        for l in range(4):
            E = np.zeros((1, 4, 4))
            E[0, k, l] = eps
            dP = (forward_fn(H + E) - forward_fn(H - E)) / (2 * eps)
            dH[:, k, l] = (G * dP).sum((1, 2))
    return dH
