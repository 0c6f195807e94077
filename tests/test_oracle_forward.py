"""Pins for the fp64 oracle's FORWARD against what the paper and the mathematics fix (CPU only).

Each test names the pin of SURVEY.md 8(c) / DESIGN.md it implements.  Nothing here calls the CUDA path.
"""
import itertools

import numpy as np
import pytest

from oracle import numpy_ref, paper_formulas as pf
from paper_2606_07574_b200 import inputs

PERMS = list(itertools.permutations(range(4)))


def _H(B, s, sub=0):
    return inputs.normal(B, s, config=50, sub=sub)[0].astype(np.float64)


# ---- P1: additively separable logits (incl. all-equal) project to the uniform matrix ---------------
def test_separable_gives_uniform(oracle):
    rng = np.random.default_rng(1)
    a = rng.normal(size=(64, 4, 1)) * 5
    b = rng.normal(size=(64, 1, 4)) * 5
    H = np.concatenate([a + b, np.full((1, 4, 4), 3.25), np.zeros((1, 4, 4))])
    P = oracle.forward(H)
    assert np.abs(P - 0.25).max() < 1e-14


# ---- P2: equivariance under all 24 x 24 row/column permutations ------------------------------------
@pytest.mark.parametrize("s", [1.0, 10.0])
def test_permutation_equivariance(oracle, s):
    H = _H(3, s)
    P = oracle.forward(H)
    Hp, Pp = [], []
    for b in range(H.shape[0]):
        for pr in PERMS:
            for pc in PERMS:
                Hp.append(H[b][np.ix_(pr, pc)])
                Pp.append(P[b][np.ix_(pr, pc)])
    got = oracle.forward(np.array(Hp))
    assert np.abs(got - np.array(Pp)).max() < 5e-13


# ---- P3 + P4 (=> P5: P is THE projection, by uniqueness PAPER.md:62) -------------------------------
@pytest.mark.parametrize("s", [1.0, 2.0, 10.0, 30.0, 100.0])
def test_scaling_form_and_marginals(oracle, s):
    H = _H(2048, s)
    P, info = oracle.forward(H, return_info=True)
    assert info["uncertified"] == 0
    assert oracle.marginal_err(P).max() < 1e-12                     # P4
    assert numpy_ref.marginal_err(P).max() < 1e-12                  # same metric, independent write-up
    # P3: L = log P - H is rank-2 additive: L_ij - L_il - L_kj + L_kl = 0.
    # Entries below 1e-280 are excluded (log of a denormal/zero).
    with np.errstate(divide="ignore"):
        L = np.log(P) - H
    worst = 0.0
    for i, k in itertools.combinations(range(4), 2):
        for j, l in itertools.combinations(range(4), 2):
            q = L[:, i, j] - L[:, i, l] - L[:, k, j] + L[:, k, l]
            ok = (P[:, [i, i, k, k], [j, l, j, l]] > 1e-280).all(axis=1)
            worst = max(worst, np.abs(q[ok]).max())
    assert worst < 1e-10 * max(1.0, s)


# ---- P6: 2x2 closed form, embedded as two blocks in a 4x4 ------------------------------------------
def test_two_by_two_closed_form(oracle):
    rng = np.random.default_rng(6)
    B = 200
    H = np.full((B, 4, 4), -200.0)                                  # leakage between blocks ~ e^-200
    H[:, :2, :2] = rng.normal(size=(B, 2, 2)) * 3
    H[:, 2:, 2:] = rng.normal(size=(B, 2, 2)) * 3
    P = oracle.forward(H)
    for blk in (slice(0, 2), slice(2, 4)):
        K = np.exp(H[:, blk, blk])
        p = 1.0 / (1.0 + np.sqrt(K[:, 0, 1] * K[:, 1, 0] / (K[:, 0, 0] * K[:, 1, 1])))
        want = np.stack([np.stack([p, 1 - p], -1), np.stack([1 - p, p], -1)], -2)
        assert np.abs(P[:, blk, blk] - want).max() < 1e-13
    assert P[:, :2, 2:].max() < 1e-80 and P[:, 2:, :2].max() < 1e-80


# ---- P7: symmetry, circulant structure, shift invariance -------------------------------------------
def test_symmetry_circulant_shift(oracle):
    H = _H(256, 2.0)
    Hs = H + H.transpose(0, 2, 1)
    Ps = oracle.forward(Hs)
    assert np.abs(Ps - Ps.transpose(0, 2, 1)).max() < 1e-13
    c = _H(256, 2.0, sub=1)[:, 0, :]
    idx = (np.arange(4)[None, :] - np.arange(4)[:, None]) % 4
    Pc = oracle.forward(c[:, idx])
    assert np.abs(Pc - Pc[:, 0, :][:, idx]).max() < 1e-13
    assert np.abs(oracle.forward(H + 7.5) - oracle.forward(H)).max() < 1e-13
    # row / column shifts: P(H + a 1^T + 1 b^T) = P(H)
    rng = np.random.default_rng(7)
    a, b = rng.normal(size=(256, 4, 1)), rng.normal(size=(256, 1, 4))
    assert np.abs(oracle.forward(H + a + b) - oracle.forward(H)).max() < 1e-13


# ---- P8: large-magnitude limit = max-weight assignment (LP limit of (3)) --------------
def test_assignment_limit(oracle):
    H = _H(4096, 100.0)
    tot = np.stack([sum(H[:, i, p[i]] for i in range(4)) for p in PERMS], axis=1)
    order = np.sort(tot, axis=1)
    margin = order[:, -1] - order[:, -2]
    # around a cycle of k <= 4 swapped entries the off-assignment product is e^{-margin' } with
    # margin' >= margin, so every off-assignment entry is at most ~e^{-margin/4}
    keep = margin > 160.0
    assert keep.sum() > 200
    best = np.array(PERMS)[np.argmax(tot, axis=1)]
    P = oracle.forward(H)
    want = np.zeros_like(P)
    for i in range(4):
        want[np.arange(P.shape[0]), i, best[:, i]] = 1.0
    # 1e-12: the oracle's own certified accuracy at |H| ~ 300 (fp64 rounding of a_i + H_ij + b_j)
    assert np.abs(P[keep] - want[keep]).max() < 1e-12


# ---- the two tiers and the numpy write-up agree ----------------------------------------------------
@pytest.mark.parametrize("s", [1.0, 2.0])
def test_tiers_and_numpy_agree(oracle, s):
    H = _H(512, s)
    P1, i1 = oracle.forward(H, max_sweeps=20000, return_info=True)
    P2, i2 = oracle.forward(H, max_sweeps=0, return_info=True)      # forces tier 2 (Newton on full dual)
    assert (i1["tier"] == 1).all() and (i2["tier"] == 2).all()
    assert np.abs(P1 - P2).max() < 2e-14
    Pn, en, _ = numpy_ref.forward_sinkhorn(H)
    assert en.max() <= 1e-14
    assert np.abs(P1 - Pn).max() < 2e-14


# ---- the paper's own Newton iteration (eqs. (8)-(12), fp64) lands on the oracle's P ----------------
def test_paper_newton_reaches_oracle(oracle):
    H = _H(64, 1.0)
    P = oracle.forward(H)
    for b in range(H.shape[0]):
        T, _, it = pf.newton_forward(H[b])
        assert it < 50
        assert np.abs(T - P[b]).max() < 1e-12


# ---- eq. (9): gradient and Hessian of f by finite differences of f ---------
def test_paper_gradient_hessian_match_f(oracle):
    rng = np.random.default_rng(9)
    R = rng.normal(size=(4, 4))
    x = rng.normal(size=3) * 0.3
    g, Hm = pf.grad_hess(pf.T_of_beta(R, x))
    eps = 1e-5
    for j in range(3):
        e = np.zeros(3)
        e[j] = eps
        gj = (pf.f_value(R, x + e) - pf.f_value(R, x - e)) / (2 * eps)
        assert abs(gj - g[j]) < 1e-9
        gp, _ = pf.grad_hess(pf.T_of_beta(R, x + e))
        gm, _ = pf.grad_hess(pf.T_of_beta(R, x - e))
        assert np.abs((gp - gm) / (2 * eps) - Hm[:, j]).max() < 1e-9


# ---- DESIGN.md G2: eq. (12) as printed has a typo in the first cofactor ----------------------------
def test_eq12_first_cofactor_reading():
    rng = np.random.default_rng(12)
    worst_fixed, worst_printed = 0.0, 0.0
    for _ in range(50):
        A = rng.normal(size=(3, 3))
        Hm = A @ A.T + 0.5 * np.eye(3)
        g = rng.normal(size=3)
        want = -np.linalg.solve(Hm, g)
        worst_fixed = max(worst_fixed, np.abs(pf.solve3_closed_form(Hm, g) - want).max())
        worst_printed = max(worst_printed, np.abs(pf.solve3_closed_form(Hm, g, as_printed=True) - want).max())
    assert worst_fixed < 1e-12
    assert worst_printed > 1e-2


# ---- degenerate inputs -----------------------------------------------------------------------------
def test_empty_and_nonfinite(oracle):
    assert oracle.forward(np.zeros((0, 4, 4))).shape == (0, 4, 4)
    H = _H(4, 1.0)
    H[1, 2, 3] = np.nan
    H[2, 0, 0] = np.inf
    P = oracle.forward(H)
    assert np.isnan(P[1]).all() and np.isnan(P[2]).all()
    assert np.isfinite(P[0]).all() and np.isfinite(P[3]).all()
    assert oracle.marginal_err(P[[0, 3]]).max() < 1e-13


def test_marginal_error_helpers_on_hand_built_matrices(oracle):
    """pins of oracle.marginal_err_inf and oracle.marginal_err on matrices whose row and column
    deviations are known by construction, not computed by the helpers: T = 1/4 + D with D built from chosen row
    deviations r and column deviations c (sum r = sum c) as D_ij = r_i/4 + c_j/4 - sum(r)/16, whose row sums are r_i and
    column sums c_j exactly in exact arithmetic."""
    r = np.array([3e-7, -1e-7, 0.0, 0.0])
    c = np.array([2e-7, 0.0, 5e-8, -5e-8])                          # sum r = sum c = 2e-7
    D = r[:, None] / 4 + c[None, :] / 4 - r.sum() / 16
    T = (0.25 + D)[None]
    assert abs(oracle.marginal_err_inf(T)[0] - 3e-7) < 1e-15        # the largest single deviation: row 0
    assert abs(oracle.marginal_err(T)[0] - (4e-7 + 3e-7)) < 1e-15   # sum |r| + sum |c|
    # the largest deviation in a column, and a transposed operand would be caught: rows exact, one column pair off
    T2 = np.full((1, 4, 4), 0.25)
    T2[0, :, 1] += 2.5e-7
    T2[0, :, 2] -= 2.5e-7
    assert abs(oracle.marginal_err_inf(T2)[0] - 1e-6) < 1e-15 and abs(oracle.marginal_err(T2)[0] - 2e-6) < 1e-15
    T3 = np.transpose(T2, (0, 2, 1)).copy()
    T3[0, 0, :] += 1e-7                                             # now rows 1, 2 are off by 1e-6 and row 0 by 4e-7, columns by 1e-7
    assert abs(oracle.marginal_err_inf(T3)[0] - 1e-6) < 1e-15 and abs(oracle.marginal_err(T3)[0] - 2.8e-6) < 1e-15
    # Err_inf <= Err <= 8 Err_inf (8 marginals) on arbitrary matrices
    rng = np.random.default_rng(5)
    X = rng.random((500, 4, 4))
    e, einf = oracle.marginal_err(X), oracle.marginal_err_inf(X)
    assert (einf <= e + 1e-15).all() and (e <= 8 * einf + 1e-15).all()
