"""Pins for the fp64 oracle's BACKWARD and the Sinkhorn-20 convention (CPU only)."""
import os

import numpy as np
import pytest

from oracle import numpy_ref, paper_formulas as pf
from paper_2606_07574_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _HG(B, s, sub=0):
    H, G = inputs.normal(B, s, config=51, sub=sub)
    return H.astype(np.float64), G.astype(np.float64)


# ---- P10: backward == central finite differences of the oracle forward (definition of derivative) --
@pytest.mark.parametrize("s", [1.0, 3.0])
def test_backward_matches_finite_differences(oracle, s):
    H, G = _HG(16, s)
    P = oracle.forward(H)
    dH = oracle.backward(P, G)
    fd = numpy_ref.backward_finite_difference(lambda X: oracle.forward(X), H, G, eps=1e-6)
    assert np.abs(dH - fd).max() < 5e-9
    # the numpy write-up (library pinv) gives the same numbers as the C Jacobi solve
    assert np.abs(dH - numpy_ref.backward_pinv(P, G)).max() < 1e-13


# ---- P10b: value pin at LARGE scale: the gauge-fixed 7x7 system (PAPER.md:543-563 with w_4 = 0) solved in 80-digit
# arithmetic.  The library pinv of numpy_ref.backward_pinv loses the small eigenvalues there (off by up to 1e-3 at
# s >= 10) and is NOT the cross-check at these scales; this is.
def _backward_exact_mp(P, G):
    import mpmath as mp
    with mp.workdps(80):
        Pm = [[mp.mpf(float(P[i, j])) for j in range(4)] for i in range(4)]
        Gm = [[mp.mpf(float(G[i, j])) for j in range(4)] for i in range(4)]
        K, rhs = mp.zeros(7, 7), mp.zeros(7, 1)
        for i in range(4):
            K[i, i] = sum(Pm[i])                                           # diag(r)
            rhs[i] = sum(Gm[i][j] * Pm[i][j] for j in range(4))            # mu_r
            for j in range(3):
                K[i, 4 + j] = K[4 + j, i] = Pm[i][j]
        for j in range(3):
            K[4 + j, 4 + j] = sum(Pm[i][j] for i in range(4))              # diag(c), last column dropped (gauge)
            rhs[4 + j] = sum(Gm[i][j] * Pm[i][j] for i in range(4))        # mu_c
        y = mp.lu_solve(K, rhs)
        v, w = [y[i] for i in range(4)], [y[4], y[5], y[6], mp.mpf(0)]
        return np.array([[float(Pm[i][j] * (Gm[i][j] - v[i] - w[j])) for j in range(4)] for i in range(4)])


@pytest.mark.parametrize("s", [10.0, 30.0, 100.0])
def test_backward_large_scale_against_80_digit_solve(oracle, s):
    H, G = inputs.normal(64, s, config=51, sub=7)
    P = oracle.forward(H)
    dH = oracle.backward(P, G)
    checked, worst = 0, 0.0
    for b in range(64):
        if P[b].min() <= 0.0:                                             # exactly decomposed: the 7x7 system is singular
            continue
        try:
            ex = _backward_exact_mp(P[b], G[b].astype(np.float64))
        except ZeroDivisionError:
            continue
        worst = max(worst, float(np.abs(ex - dH[b]).max()))
        checked += 1
    assert checked >= 60
    assert worst < 1e-12


# ---- P11: every row and column sum of dH vanishes (P(H + a 1^T + 1 b^T) = P(H)) --------------------
@pytest.mark.parametrize("s", [1.0, 10.0, 100.0])
def test_backward_row_col_sums_zero(oracle, s):
    H, G = _HG(1024, s)
    dH = oracle.backward(oracle.forward(H), G)
    assert np.isfinite(dH).all()
    assert np.abs(dH.sum(1)).max() < 1e-12 and np.abs(dH.sum(2)).max() < 1e-12


# ---- P12: additive G gives zero gradient; dH is linear in G ----------------------------------------
def test_backward_additive_G_and_linearity(oracle):
    H, G = _HG(256, 2.0)
    P = oracle.forward(H)
    rng = np.random.default_rng(12)
    a, b = rng.normal(size=(256, 4, 1)), rng.normal(size=(256, 1, 4))
    assert np.abs(oracle.backward(P, a + b + np.zeros_like(P))).max() < 1e-13
    G2 = rng.normal(size=G.shape)
    lhs = oracle.backward(P, 2.0 * G - 3.0 * G2)
    rhs = 2.0 * oracle.backward(P, G) - 3.0 * oracle.backward(P, G2)
    assert np.abs(lhs - rhs).max() < 1e-13


# ---- P13: the paper's closed form (13) / section 4.2 equals the gauge-free KKT solve ---------------
@pytest.mark.parametrize("s", [1.0, 3.0])
def test_paper_closed_form_equals_kkt(oracle, s):
    H, G = _HG(128, s)
    P = oracle.forward(H)
    dH = oracle.backward(P, G)
    for b in range(P.shape[0]):
        assert np.abs(pf.backward_closed_form(P[b], G[b]) - dH[b]).max() < 1e-11


# ---- near-permutation P: the ungauged solve stays finite and consistent with finite differences ----
def test_backward_near_permutation(oracle):
    H, G = _HG(8, 1.0, sub=3)
    for i in range(4):
        H[:, i, (i + 1) % 4] += 12.0
    P = oracle.forward(H)
    assert P.max() > 0.9999
    dH = oracle.backward(P, G)
    fd = numpy_ref.backward_finite_difference(lambda X: oracle.forward(X), H, G, eps=1e-6)
    assert np.abs(dH - fd).max() < 5e-9
    # exactly decomposed P (leak below fp64): each block is its own problem, min-norm solve is finite
    Hb = np.full((1, 4, 4), -800.0)
    Hb[0, :2, :2] = H[0, :2, :2]
    Hb[0, 2:, 2:] = H[0, 2:, 2:]
    Pb = oracle.forward(Hb)
    dHb = oracle.backward(Pb, G[:1])
    assert np.isfinite(dHb).all()
    for blk in (slice(0, 2), slice(2, 4)):
        # 2x2 block: p = sigmoid(z/2), z = h11+h22-h12-h21; dL/dz by the chain rule
        p = Pb[0, blk, blk][0, 0]
        g = G[0, blk, blk]
        dz = (g[0, 0] + g[1, 1] - g[0, 1] - g[1, 0]) * p * (1 - p) / 2
        want = dz * np.array([[1.0, -1.0], [-1.0, 1.0]])
        assert np.abs(dHb[0, blk, blk] - want).max() < 1e-13


# ---- P9: Sinkhorn-20 convention and the Err metric against PAPER.md Table 2 ------------------------
def _table2():
    rows = {}
    for line in open(os.path.join(GOLDEN, "paper_table2_sinkhorn20.txt")):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        rows[f[0]] = dict(mean=float(f[1]) * 1e-3, std=float(f[2]) * 1e-3, median=float(f[3]) * 1e-3)
    return rows


def test_sinkhorn20_statistics_match_paper_table2(oracle):
    t2 = _table2()
    N = 10000
    for name, H in (("N(0,10^2)", inputs.normal(N, 10.0, config=52)[0]),
                    ("Unif(-10,10)", inputs.uniform(N, 10.0, config=52)[0])):
        err = oracle.marginal_err(oracle.sinkhorn(H, 20))
        se = t2[name]["std"] / np.sqrt(N)
        assert abs(err.mean() - t2[name]["mean"]) < 5 * se + 0.01 * t2[name]["mean"]
        assert abs(np.median(err) - t2[name]["median"]) < 5 * 1.2533 * se + 0.01 * t2[name]["median"]


def test_sinkhorn_converges_to_projection(oracle):
    H, _ = _HG(64, 1.0)
    assert np.abs(oracle.sinkhorn(H, 2000) - oracle.forward(H)).max() < 1e-13
    # one iteration, by hand
    K = np.exp(H)
    K = K / K.sum(2, keepdims=True)
    K = K / K.sum(1, keepdims=True)
    assert np.abs(oracle.sinkhorn(H, 1) - K).max() < 1e-15
