"""Pins for the general small entropic-OT oracle (oracle/ot_oracle.c through oracle/ot.py) and its n = 8 Birkhoff
special case (CPU only).  Each pin is something the paper or the mathematics fixes independently of the oracle's own
arithmetic: closed forms, invariants, scaling laws, limits, an independent implementation, finite differences,
an 80-digit solve."""
import itertools

import numpy as np
import pytest
from scipy.optimize import linear_sum_assignment

import oracle as oracle4
from oracle import ot
from paper_2606_07574_b200 import inputs

SHAPES = [(4, 4), (8, 8), (4, 8), (8, 4), (3, 5)]


def _prob(B, n, m, s, sub=0):
    M, a, b, G = inputs.ot_problem(B, n, m, s, config=91, sub=sub)
    return M.astype(np.float64), a.astype(np.float64), b.astype(np.float64), G.astype(np.float64)


def _certified(T, info):
    assert info["uncertified"] == 0, info["err"].max()
    return T


# ---- O1: separable cost M_ij = p_i + q_j => T = a b^T / sum(a) (the entropy term alone decides) ----
@pytest.mark.parametrize("n,m", SHAPES)
def test_separable_cost_gives_product_coupling(n, m):
    rng = np.random.default_rng(1)
    _, a, b, _ = _prob(32, n, m, 1.0)
    b = b * (a.sum(1, keepdims=True) / b.sum(1, keepdims=True))
    M = rng.normal(size=(32, n, 1)) * 7 + rng.normal(size=(32, 1, m)) * 7
    for eta in (0.3, 1.0, 5.0):
        T = ot.forward(M, a, b, eta)
        want = a[:, :, None] * b[:, None, :] / a.sum(1)[:, None, None]
        assert np.abs(T - want).max() < 1e-13


# ---- O2: scaling form and marginals (=> uniqueness: the strictly convex problem (3) has one solution) ------------
@pytest.mark.parametrize("n,m", SHAPES)
@pytest.mark.parametrize("s", [1.0, 10.0, 50.0])
def test_scaling_form_and_marginals(n, m, s):
    M, a, b, _ = _prob(256, n, m, s)
    b = b * (a.sum(1, keepdims=True) / b.sum(1, keepdims=True))
    eta = 0.7
    T = _certified(*ot.forward(M, a, b, eta, return_info=True))
    assert np.abs(T.sum(2) - a).max() < 1e-12 and np.abs(T.sum(1) - b).max() < 1e-12
    with np.errstate(divide="ignore"):
        L = eta * np.log(T) + M                                       # = alpha_i + beta_j
    ok = np.isfinite(L).all(axis=(1, 2)) & (T.min(axis=(1, 2)) > 1e-250)
    L = L[ok]
    R = L - L[:, :1, :] - L[:, :, :1] + L[:, :1, :1]                   # rank-2 additive <=> all 2x2 "cross differences" vanish
    assert ok.sum() > 10 and np.abs(R).max() < 1e-7 * max(1.0, s)


# ---- O3: permutation equivariance ---------------------------------------------------------------------------------
def test_permutation_equivariance():
    M, a, b, _ = _prob(8, 4, 5, 3.0)
    b = b * (a.sum(1, keepdims=True) / b.sum(1, keepdims=True))
    T = ot.forward(M, a, b, 0.9)
    rng = np.random.default_rng(3)
    for _ in range(10):
        pr, pc = rng.permutation(4), rng.permutation(5)
        Tp = ot.forward(M[:, pr][:, :, pc], a[:, pr], b[:, pc], 0.9)
        assert np.abs(Tp - T[:, pr][:, :, pc]).max() < 1e-13


# ---- O4: the 2x2 problem in closed form with general marginals ---------------------------------------------------
def test_two_by_two_closed_form():
    rng = np.random.default_rng(4)
    B = 200
    M = rng.normal(size=(B, 2, 2)) * 3
    a = rng.uniform(0.2, 2.0, size=(B, 2))
    b1 = rng.uniform(0.05, 0.95, size=B) * a.sum(1)
    b = np.stack([b1, a.sum(1) - b1], 1)
    eta = 0.8
    T = ot.forward(M, a, b, eta)
    # T = [[t, a1-t],[b1-t, a2-b1+t]] with  t (a2-b1+t) = K (a1-t)(b1-t),  K = exp(-(M11+M22-M12-M21)/eta)
    K = np.exp(-(M[:, 0, 0] + M[:, 1, 1] - M[:, 0, 1] - M[:, 1, 0]) / eta)
    a1, a2, bb = a[:, 0], a[:, 1], b[:, 0]
    A, Bq, C = 1 - K, (a2 - bb) + K * (a1 + bb), -K * a1 * bb
    disc = np.sqrt(Bq * Bq - 4 * A * C)
    t = np.where(np.abs(A) < 1e-12, -C / Bq, (-Bq + disc) / (2 * A))
    lo, hi = np.maximum(0, bb - a2), np.minimum(a1, bb)
    t2 = np.where(np.abs(A) < 1e-12, t, (-Bq - disc) / (2 * A))
    t = np.where((t >= lo - 1e-12) & (t <= hi + 1e-12), t, t2)
    assert np.abs(T[:, 0, 0] - t).max() < 1e-12


# ---- O5: scaling laws: OT(M, eta) = OT(M / eta, 1);  OT(M, c a, c b) = c OT(M, a, b);  row/column offsets --------
def test_scaling_laws():
    M, a, b, _ = _prob(64, 4, 8, 2.0)
    b = b * (a.sum(1, keepdims=True) / b.sum(1, keepdims=True))
    T = ot.forward(M, a, b, 2.5)
    assert np.abs(T - ot.forward(M / 2.5, a, b, 1.0)).max() < 1e-13
    assert np.abs(3.0 * T - ot.forward(M, 3.0 * a, 3.0 * b, 2.5)).max() < 1e-12
    rng = np.random.default_rng(5)
    M2 = M + rng.normal(size=(64, 4, 1)) * 9 + rng.normal(size=(64, 1, 8)) * 9
    assert np.abs(T - ot.forward(M2, a, b, 2.5)).max() < 1e-12


# ---- O6: eta -> 0: the support of T is the optimal assignment (LP limit of (3)) ---------------------
def test_assignment_limit_n8():
    H = inputs.normal_n(64, 8, 400.0, config=92)[0].astype(np.float64)
    P = ot.birkhoff_forward(H)
    checked = 0
    for k in range(64):
        r, c = linear_sum_assignment(-H[k])
        tot = H[k][r, c].sum()
        # second-best value: drop one assigned edge at a time (a lower bound on the gap suffices to skip near-ties)
        gap = min(tot - (lambda Hx: Hx[linear_sum_assignment(-Hx)].sum())(np.where(
            (np.arange(8)[:, None] == r[q]) & (np.arange(8)[None, :] == c[q]), -1e9, H[k])) for q in range(8))
        if gap > 60.0:     # an off-assignment entry is exp(-slack) and the slacks of a cycle add up to the gap (8 edges at most)
            want = np.zeros((8, 8))
            want[r, c] = 1.0
            assert np.abs(P[k] - want).max() < 1e-3
            assert (P[k][r, c] > 0.999).all()
            checked += 1
    assert checked >= 5


# ---- O7: the two independent oracles agree where they overlap ---------------------------------------------------
@pytest.mark.parametrize("s", [1.0, 10.0, 100.0])
def test_agrees_with_the_4x4_oracle(s):
    H, G = inputs.normal(512, s, config=93)
    P4, i4 = oracle4.forward(H, return_info=True)
    P, i = ot.forward(-H.astype(np.float64), None, None, 1.0, return_info=True)
    assert i4["uncertified"] == 0 and i["uncertified"] == 0
    assert np.abs(P - P4).max() < 1e-12
    assert np.abs(ot.birkhoff_backward(P, G) - oracle4.backward(P4, G)).max() < 1e-11
    assert np.abs(ot.marginal_err(P) - oracle4.marginal_err(P)).max() < 1e-15


# ---- O8: n = 8 Birkhoff: separable => 1/8, doubly stochastic, permutation equivariance ---------------------------
def test_birkhoff8_properties():
    rng = np.random.default_rng(8)
    H = rng.normal(size=(16, 8, 1)) * 4 + rng.normal(size=(16, 1, 8)) * 4
    assert np.abs(ot.birkhoff_forward(H) - 0.125).max() < 1e-14
    for s in (1.0, 10.0):
        H = inputs.normal_n(128, 8, s, config=94)[0].astype(np.float64)
        P, info = ot.forward(-H, return_info=True)
        assert info["uncertified"] == 0
        assert np.abs(P.sum(1) - 1).max() < 1e-13 and np.abs(P.sum(2) - 1).max() < 1e-13 and P.min() >= 0
        pr, pc = rng.permutation(8), rng.permutation(8)
        assert np.abs(ot.birkhoff_forward(H[:, pr][:, :, pc]) - P[:, pr][:, :, pc]).max() < 1e-12


# ---- O9: backward == central finite differences of the forward (definition of the derivative) -------------------
@pytest.mark.parametrize("n,m", [(4, 4), (8, 8), (4, 8), (3, 5)])
def test_backward_matches_finite_differences(n, m):
    M, a, b, G = _prob(4, n, m, 1.5, sub=9)
    b = b * (a.sum(1, keepdims=True) / b.sum(1, keepdims=True))
    eta = 0.8
    T = ot.forward(M, a, b, eta)
    D = ot.backward(T, G, eta)
    fd = np.zeros_like(M)
    eps = 1e-6
    for i in range(n):
        for j in range(m):
            E = np.zeros((1, n, m))
            E[0, i, j] = eps
            dT = (ot.forward(M + E, a, b, eta) - ot.forward(M - E, a, b, eta)) / (2 * eps)
            fd[:, i, j] = (G * dT).sum((1, 2))
    assert np.abs(D - fd).max() < 2e-8
    # T does not change under row/column offsets of M: every row and column of D sums to zero
    assert np.abs(D.sum(1)).max() < 1e-12 and np.abs(D.sum(2)).max() < 1e-12


# ---- O10: the paper's closed form (13) (gauge beta_m = 0) equals the ungauged solve ------------
@pytest.mark.parametrize("n,m", [(4, 4), (8, 8), (4, 8), (8, 4)])
def test_paper_closed_form_13(n, m):
    M, a, b, G = _prob(32, n, m, 2.0, sub=10)
    b = b * (a.sum(1, keepdims=True) / b.sum(1, keepdims=True))
    eta = 1.3
    T = ot.forward(M, a, b, eta)
    D = ot.backward(T, G, eta)
    for k in range(32):
        Tk, Gk, ak, bk_ = T[k], G[k], a[k], b[k]
        Gam = Gk * Tk
        mur, muc = Gam.sum(1), Gam.sum(0)[:-1]
        Tm = Tk[:, :-1]
        Delta = np.diag(bk_[:-1]) - Tm.T @ np.diag(1 / ak) @ Tm
        w = np.append(np.linalg.solve(Delta, muc - Tm.T @ (mur / ak)), 0.0)
        want = (np.diag((mur - Tm @ w[:-1]) / ak) @ Tk + Tk @ np.diag(w) - Gam) / eta
        assert np.abs(D[k] - want).max() < 1e-10


# ---- O11: value pin of the backward at large scale: gauge-fixed system in 80-digit arithmetic -------------------
@pytest.mark.parametrize("s", [10.0, 30.0])
def test_backward_n8_against_80_digit_solve(s):
    import mpmath as mp
    H, G = inputs.normal_n(12, 8, s, config=95)
    H, G = H.astype(np.float64), G.astype(np.float64)
    P = ot.birkhoff_forward(H)
    dH = ot.birkhoff_backward(P, G)
    checked = 0
    for k in range(12):
        if P[k].min() <= 0.0:
            continue
        with mp.workdps(80):
            n = 8
            Pm = [[mp.mpf(float(P[k, i, j])) for j in range(n)] for i in range(n)]
            Gm = [[mp.mpf(float(G[k, i, j])) for j in range(n)] for i in range(n)]
            K, rhs = mp.zeros(2 * n - 1, 2 * n - 1), mp.zeros(2 * n - 1, 1)
            for i in range(n):
                K[i, i] = sum(Pm[i])
                rhs[i] = sum(Gm[i][j] * Pm[i][j] for j in range(n))
                for j in range(n - 1):
                    K[i, n + j] = K[n + j, i] = Pm[i][j]
            for j in range(n - 1):
                K[n + j, n + j] = sum(Pm[i][j] for i in range(n))
                rhs[n + j] = sum(Gm[i][j] * Pm[i][j] for i in range(n))
            try:
                y = mp.lu_solve(K, rhs)
            except ZeroDivisionError:
                continue
            w = [y[n + j] for j in range(n - 1)] + [mp.mpf(0)]
            ex = np.array([[float(Pm[i][j] * (Gm[i][j] - y[i] - w[j])) for j in range(n)] for i in range(n)])
        assert np.abs(ex - dH[k]).max() < 1e-11
        checked += 1
    assert checked >= 10


def test_marginal_err_with_given_marginals_on_a_hand_built_plan():
    """pin of ot.marginal_err (PAPER.md:323 with marginals a, b): the plan T = a b^T / sum(a) has row sums a and column
    sums b; moving mass d from entry (0,0) to (0,1) leaves the rows alone and puts columns 0 and 1 off by d each; adding e
    to entry (2,3) puts row 2 and column 3 off by e each."""
    a = np.array([[0.5, 1.5, 0.75]])
    b = np.array([[0.25, 1.0, 0.5, 0.5, 0.5]])                      # both sum to 2.75
    T = a[:, :, None] * b[:, None, :] / a.sum()
    assert ot.marginal_err(T, a, b)[0] < 1e-15
    d, e = 1e-3, 2e-4
    T[0, 0, 0] -= d
    T[0, 0, 1] += d
    assert abs(ot.marginal_err(T, a, b)[0] - 2 * d) < 1e-15
    T[0, 2, 3] += e
    assert abs(ot.marginal_err(T, a, b)[0] - (2 * d + 2 * e)) < 1e-15
    assert abs(ot.marginal_err(T, b=b, a=a)[0] - (2 * d + 2 * e)) < 1e-15
    # against unit marginals the same plan is off by |a_i - 1| and |b_j - 1| (up to the moved mass): a and b are not ignored
    T0 = a[:, :, None] * b[:, None, :] / a.sum()
    n1 = np.ones((1, 3))
    m1 = np.ones((1, 5))
    assert abs(ot.marginal_err(T0, n1, m1)[0] - (np.abs(a - 1).sum() + np.abs(b - 1).sum())) < 1e-14
