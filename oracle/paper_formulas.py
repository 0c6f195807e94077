"""The paper's own closed forms, step by step in its notation, in float64 numpy -- TEST INFRASTRUCTURE.

These follow /root/reference/PAPER.md literally (section 3.2 and 4.2), one matrix at a time, so a reader
can check them against the paper by eye.  They are NOT how the oracle gets its answer (that is the
plain definition, oracle/birkhoff4_oracle.c); the tests use them to pin (i) the readings of the
garbled passages (G1, G2) and (ii) that the paper's formulas and the oracle's definitions
agree.  Never imported by paper_2606_07574_b200.
"""
import numpy as np


def T_of_beta(R, beta3):
    """eq. (10): U = 1 beta^T + R (beta_4 = 0), mu_i = max_j U_ij,
    T_ij = e^{U_ij - mu_i} / sum_k e^{U_ik - mu_i}.  (Softmax read as e^{v_k}/sum e^{v_l}: DESIGN.md G1.)"""
    beta = np.array([beta3[0], beta3[1], beta3[2], 0.0])
    U = R + beta[None, :]
    mu = U.max(axis=1, keepdims=True)
    E = np.exp(U - mu)
    return E / E.sum(axis=1, keepdims=True)


def f_value(R, beta3):
    """f(beta_{-m}) = -L(alpha*(beta), beta) = eta 1^T a - alpha*^T a - beta^T b, eta=1, a=b=1."""
    beta = np.array([beta3[0], beta3[1], beta3[2], 0.0])
    U = R + beta[None, :]
    mu = U.max(axis=1)
    alpha = -(mu + np.log(np.exp(U - mu[:, None]).sum(axis=1)))   # eq. (5)
    return 4.0 - alpha.sum() - beta.sum()


def grad_hess(T):
    """eq. (11) PAPER.md:193 and H = diag(c) - T_{-m}^T T_{-m}."""
    L = T[:, :3]                                           # T_{-m} = [l1, l2, l3]
    c = L.sum(axis=0)
    g = c - 1.0
    Hm = np.diag(c) - L.T @ L
    return g, Hm


def solve3_closed_form(Hm, g, as_printed=False):
    """d = -H^{-1} g by eq. (12) PAPER.md:225-233.
    The first cofactor is printed as (h12 h33 - h23^2); the adjugate of a symmetric 3x3 has
    (h22 h33 - h23^2) there (G2).  `as_printed=True` evaluates the formula exactly as printed."""
    h11, h12, h13 = Hm[0, 0], Hm[0, 1], Hm[0, 2]
    h22, h23, h33 = Hm[1, 1], Hm[1, 2], Hm[2, 2]
    g1, g2, g3 = g
    det = h11 * (h22 * h33 - h23 ** 2) - h12 * (h12 * h33 - h23 * h13) + h13 * (h12 * h23 - h22 * h13)
    first = (h12 * h33 - h23 ** 2) if as_printed else (h22 * h33 - h23 ** 2)
    d1 = -(first * g1 + (h13 * h23 - h12 * h33) * g2 + (h12 * h23 - h22 * h13) * g3) / det
    d2 = -((h13 * h23 - h12 * h33) * g1 + (h11 * h33 - h13 ** 2) * g2 + (h12 * h13 - h11 * h23) * g3) / det
    d3 = -((h12 * h23 - h22 * h13) * g1 + (h12 * h13 - h11 * h23) * g2 + (h11 * h22 - h12 ** 2) * g3) / det
    return np.array([d1, d2, d3])


def newton_forward(R, tol=1e-12, max_iter=200):
    """Newton's method on (8) from x0 = 0 with Armijo backtracking for gamma_k
    (the paper names 'line search' and gives no rule: DESIGN.md S2).  Returns T*, beta*, iterations."""
    x = np.zeros(3)
    for k in range(max_iter):
        T = T_of_beta(R, x)
        g, Hm = grad_hess(T)
        if np.abs(g).sum() + abs(g.sum()) <= tol:
            return T, x, k
        d = solve3_closed_form(Hm, g)
        f0, gam = f_value(R, x), 1.0
        while f_value(R, x + gam * d) > f0 + 1e-4 * gam * (g @ d) + 1e-14 * (1 + abs(f0)) and gam > 1e-12:
            gam *= 0.5
        x = x + gam * d
    return T_of_beta(R, x), x, max_iter


def backward_closed_form(T, G):
    """Section 4.2: Gamma = G o T*, mu_r, mu_c, Delta = I - T_{-m}^T T_{-m},
    w_{-m} = Delta^{-1}[mu_c - T_{-m}^T mu_r], w_4 = 0, v = mu_r - T* w, D_ij = (v_i + w_j - g_ij) t_ij.
    Returns dL/dR = -D."""
    Gam = G * T
    mu_r = Gam.sum(axis=1)
    mu_c = Gam[:, :3].sum(axis=0)
    L = T[:, :3]
    Delta = np.eye(3) - L.T @ L                            # eq. (13) with b_{-m} = 1, a = 1
    rhs = mu_c - L.T @ mu_r
    w3 = -solve3_closed_form(Delta, rhs)                   # eq. (12) gives -Delta^{-1} rhs
    w = np.array([w3[0], w3[1], w3[2], 0.0])
    v = mu_r - T @ w
    D = (v[:, None] + w[None, :] - G) * T
    return -D
