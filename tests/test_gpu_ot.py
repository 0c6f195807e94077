"""GPU parity of the widenings (include/birkhoff_ot.h): the n = 8 Birkhoff projection and small general entropic OT,
through the C ABI, against the fp64 oracle oracle/ot_oracle.c on the same seeded inputs.

Gates: max |T - T_oracle| <= 1e-5 (relative to the largest marginal), Err_ab <= 2e-6 * sum(a) / 4 ... stated per test,
D relative error <= 1e-4 (both readings of S10)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
from oracle import ot
from paper_2606_07574_b200 import binding as bk, inputs

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy()


def d_errors(D, D_o, G):
    e1 = np.abs(D - D_o).max() / max(np.abs(D_o).max(), 1e-300)
    e2 = (np.abs(D - D_o).reshape(len(G), -1).max(1) / np.abs(G).reshape(len(G), -1).max(1)).max()
    return e1, e2


# ---------------------------------------------------------------------------------------------------
# NEXT-1: n = 8 Birkhoff projection
@pytest.mark.parametrize("s", [0.1, 1.0, 3.0, 10.0, 30.0, 100.0])
def test_birkhoff8_parity(s):
    H, G = inputs.normal_n(4096 + 3 if s <= 10 else 2048 + 3, 8, s, config=8)
    P_o, info = ot.forward(-H.astype(np.float64), return_info=True)
    assert info["uncertified"] == 0
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    it = torch.zeros(len(H), dtype=torch.int32, device="cuda")
    Pd = bk.birkhoff8_forward(dev(H), tol=2e-6, max_iter=60, iters=it, n_unconverged=unc)
    P = host(Pd).astype(np.float64)
    assert np.isfinite(P).all() and P.min() >= 0
    eP = np.abs(P - P_o).max()
    err = ot.marginal_err(P)
    print("birkhoff8 s=%g: eP %.2e Err max %.2e mean %.2e  iters mean %.2f max %d  unconverged %d" % (
        s, eP, err.max(), err.mean(), float(it.float().mean()), int(it.max()), int(unc.item())))
    assert eP <= 1e-5
    assert err.max() <= 2e-6                                          # 16 marginals: twice the 4x4 gate
    assert int(unc.item()) == 0
    dH = host(bk.birkhoff8_backward(Pd, dev(G))).astype(np.float64)
    dH_o = ot.birkhoff_backward(P_o, G.astype(np.float64))
    e1, e2 = d_errors(dH, dH_o, G)
    assert e1 <= 1e-4 and e2 <= 1e-4, (e1, e2)


def test_birkhoff8_properties_and_edges():
    rng = np.random.default_rng(1)
    H = (rng.normal(size=(64, 8, 1)) * 4 + rng.normal(size=(64, 1, 8)) * 4).astype(np.float32)
    P = host(bk.birkhoff8_forward(dev(H)))
    assert np.abs(P - 0.125).max() < 5e-6                              # separable => uniform (fp32 H is separable up to rounding)
    H = inputs.normal_n(1000, 8, 1.0, config=8, sub=1)[0]
    pr, pc = rng.permutation(8), rng.permutation(8)
    P = host(bk.birkhoff8_forward(dev(H)))
    Pp = host(bk.birkhoff8_forward(dev(H[:, pr][:, :, pc])))
    assert np.abs(Pp - P[:, pr][:, :, pc]).max() < 2e-6
    # ragged sizes, guard cells, NaN isolation, in-place
    for B in (1, 127, 129, 1000):
        Hb = H[:B].copy()
        buf = torch.full((B + 2, 8, 8), 7.0, device="cuda")
        bk.birkhoff8_forward(dev(Hb), buf[1:B + 1])
        assert (host(buf[0]) == 7.0).all() and (host(buf[B + 1]) == 7.0).all()
        assert np.array_equal(host(buf[1:B + 1]), P[:B])
    Hn = H.copy()
    Hn[5, 2, 3] = np.nan
    Hn[6, 0, 0] = np.inf
    Pn = host(bk.birkhoff8_forward(dev(Hn)))
    assert np.isnan(Pn[5]).all() and np.isnan(Pn[6]).all()
    good = np.ones(1000, bool)
    good[[5, 6]] = False
    assert np.array_equal(Pn[good], P[good])
    X = dev(H).clone()
    bk.birkhoff8_forward(X, X)
    assert np.array_equal(host(X), P)
    e = torch.empty((0, 8, 8), device="cuda")
    assert bk.birkhoff8_forward(e).shape == (0, 8, 8) and bk.birkhoff8_backward(e, e).shape == (0, 8, 8)
    L = bk.lib()
    import ctypes
    p = ctypes.c_void_p(X.data_ptr())
    assert L.birkhoff8_forward(p, p, -1, 1e-6, 20, None, None, None) == 1
    assert L.birkhoff8_forward(None, p, 4, 1e-6, 20, None, None, None) == 1
    assert L.birkhoff8_forward(ctypes.c_void_p(X.data_ptr() + 4), p, 1, 1e-6, 20, None, None, None) == 1
    assert L.entropic_ot_forward(p, None, None, p, 4, 9, 9, 1.0, 1e-6, 20, None, None, None) == 1     # unsupported size (> 8)
    assert L.entropic_ot_forward(p, p, p, p, 4, 1, 4, 1.0, 1e-6, 20, None, None, None) == 1           # unsupported size (< 2)
    assert L.entropic_ot_backward(p, p, p, 4, 4, 9, 1.0, None) == 1
    assert L.entropic_ot_forward(p, None, None, p, 4, 4, 8, 1.0, 1e-6, 20, None, None, None) == 1     # unit marginals, n != m
    assert L.entropic_ot_forward(p, p, None, p, 4, 4, 4, 1.0, 1e-6, 20, None, None, None) == 1        # one marginal missing
    assert L.entropic_ot_forward(p, None, None, p, 4, 4, 4, 0.0, 1e-6, 20, None, None, None) == 1     # eta = 0


# ---------------------------------------------------------------------------------------------------
# NEXT-3: general small entropic OT (PAPER.md:83-168 forward, eq. (13) backward)
@pytest.mark.parametrize("n,m", [(4, 4), (8, 8), (4, 8), (8, 4)])
@pytest.mark.parametrize("s,eta,skew", [(1.0, 1.0, None), (3.0, 0.5, None), (2.0, 2.0, None), (10.0, 1.0, None),
                                        (1.0, 0.1, None), (3.0, 0.1, None), (30.0, 1.0, None),      # eta << range
                                        (1.0, 1.0, 1e-6), (3.0, 0.5, 1e-6)])                       # one column with next to no mass
def test_entropic_ot_parity(n, m, s, eta, skew):
    Cm, a, b, G = inputs.ot_problem(2048 + 5, n, m, s, config=9, sub=n * 10 + m)
    if skew:
        b = b.astype(np.float64)
        b[:, 0] = skew
        b[:, 1:] *= ((a.astype(np.float64).sum(1) - skew) / b[:, 1:].sum(1))[:, None]
        b = b.astype(np.float32)
    # the fp32 marginals' sums agree only to fp32 rounding; problem (3) needs them equal, so the
    # oracle gets b rescaled in fp64 by 1 + O(1e-7): a perturbation far inside the tolerances below
    a64, b64 = a.astype(np.float64), b.astype(np.float64)
    b64 = b64 * (a64.sum(1, keepdims=True) / b64.sum(1, keepdims=True))
    T_o, info = ot.forward(Cm, a64, b64, eta, return_info=True)
    assert info["uncertified"] == 0
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    tol = 2e-6 * max(n, m) / 4
    Td = bk.entropic_ot_forward(dev(Cm), dev(a), dev(b), eta=eta, tol=tol, max_iter=80, n_unconverged=unc)
    T = host(Td).astype(np.float64)
    assert np.isfinite(T).all() and T.min() >= 0
    eT = np.abs(T - T_o).max() / a.max()
    err = ot.marginal_err(T, a, b)
    print("ot %dx%d s=%g eta=%g: eT %.2e Err max %.2e  unconverged %d" % (n, m, s, eta, eT, err.max(), int(unc.item())))
    assert eT <= 1e-5
    # the marginals given in fp32 do not have exactly equal sums: that mismatch is part of Err_ab and not the solver's
    mism = np.abs(a.astype(np.float64).sum(1) - b.astype(np.float64).sum(1)).max()
    assert err.max() <= tol + mism
    assert int(unc.item()) == 0
    D = host(bk.entropic_ot_backward(Td, dev(G), eta=eta)).astype(np.float64)
    D_o = ot.backward(T_o, G.astype(np.float64), eta)
    e1, e2 = d_errors(D * eta, D_o * eta, G)
    assert e1 <= 1e-4 and e2 <= 1e-4 * a.max(), (e1, e2)


def test_entropic_ot_reduces_to_birkhoff4():
    """C = -H, eta = 1, unit marginals: the 4x4 Birkhoff projection of the main path"""
    H, G = inputs.normal(8192, 2.0, config=96)
    P = host(bk.birkhoff4_forward(dev(H)))
    T = host(bk.entropic_ot_forward(dev(-H), tol=1e-6, max_iter=40))
    assert np.abs(T - P).max() < 2e-6
    dH = host(bk.birkhoff4_backward(dev(P), dev(G)))
    D = host(bk.entropic_ot_backward(dev(P), dev(G)))
    assert np.abs(D + dH).max() < 5e-6
    T8 = host(bk.entropic_ot_forward(dev(-inputs.normal_n(512, 8, 1.0, config=97)[0])))
    P8 = host(bk.birkhoff8_forward(dev(inputs.normal_n(512, 8, 1.0, config=97)[0])))
    assert np.array_equal(T8, P8)


def test_ot_runs_out_of_updates_mid_continuation():
    """max_iter spent before the last continuation stage: the result is finite, its rows still carry the row marginals,
    every such problem is counted, and no problem reports more updates than it was given"""
    H = inputs.normal_n(2048 + 3, 8, 100.0, config=8)[0]
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    it = torch.zeros(len(H), dtype=torch.int32, device="cuda")
    P = host(bk.birkhoff8_forward(dev(H), tol=2e-6, max_iter=8, iters=it, n_unconverged=unc)).astype(np.float64)
    iters = host(it)
    assert np.isfinite(P).all() and P.min() >= 0 and iters.max() <= 8
    assert np.abs(P.sum(2) - 1).max() <= 1e-6
    bad = ot.marginal_err(P) > 2e-6
    assert bad.any() and int(unc.item()) >= bad.sum() and (iters[bad] == 8).all()
    Cm, a, b, _ = inputs.ot_problem(1024 + 1, 4, 8, 30.0, config=9, sub=48)
    unc.zero_()
    T = host(bk.entropic_ot_forward(dev(Cm), dev(a), dev(b), eta=1.0, tol=4e-6, max_iter=5, n_unconverged=unc)).astype(np.float64)
    assert np.isfinite(T).all() and np.abs(T.sum(2) - a).max() <= 1e-5 and int(unc.item()) > 0


def test_ot_inf_cost_gives_nan_for_that_problem_only():
    Cm, a, b, _ = inputs.ot_problem(300, 8, 8, 2.0, config=9, sub=5)
    T = host(bk.entropic_ot_forward(dev(Cm), dev(a), dev(b), eta=0.5))
    Cn = Cm.copy()
    Cn[7, 1, 2] = np.inf
    Cn[9, 0, 0] = -np.inf
    Cn[11, 3, 3] = np.nan
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    Tn = host(bk.entropic_ot_forward(dev(Cn), dev(a), dev(b), eta=0.5, n_unconverged=unc))
    good = np.ones(300, bool)
    good[[7, 9, 11]] = False
    assert np.isnan(Tn[~good]).all() and np.array_equal(Tn[good], T[good]) and int(unc.item()) == 3


# ---------------------------------------------------------------------------------------------------
# NEXT-3 at every size 2 <= n, m <= 8 (PAPER.md:83-168 is written for any n x m; eq. (13)): sizes other
# than {4, 8} x {4, 8} run padded inside the next tile, the padding carrying no mass
RAGGED = [(3, 5), (5, 8), (6, 6), (2, 2), (7, 3), (5, 4), (2, 8), (8, 2), (3, 3), (4, 7), (8, 7)]


@pytest.mark.parametrize("n,m", RAGGED)
@pytest.mark.parametrize("s,eta", [(1.0, 1.0), (3.0, 0.5), (10.0, 1.0)])
def test_entropic_ot_parity_any_size(n, m, s, eta):
    B = 1024 + 5
    Cm, a, b, G = inputs.ot_problem(B, n, m, s, config=9, sub=100 + n * 10 + m)
    a64, b64 = a.astype(np.float64), b.astype(np.float64)
    b64 = b64 * (a64.sum(1, keepdims=True) / b64.sum(1, keepdims=True))
    T_o, info = ot.forward(Cm, a64, b64, eta, return_info=True)
    assert info["uncertified"] == 0
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    tol = 2e-6 * max(n, m) / 4
    # guard cells on both sides of the output: a padded tile must not write outside its n x m problem
    buf = torch.full((B + 2, n, m), 7.0, device="cuda")
    Td = bk.entropic_ot_forward(dev(Cm), dev(a), dev(b), buf[1:B + 1], eta=eta, tol=tol, max_iter=80, n_unconverged=unc)
    assert (host(buf[0]) == 7.0).all() and (host(buf[B + 1]) == 7.0).all()
    T = host(Td).astype(np.float64)
    assert np.isfinite(T).all() and T.min() >= 0
    eT = np.abs(T - T_o).max() / a.max()
    err = ot.marginal_err(T, a, b)
    mism = np.abs(a64.sum(1) - b.astype(np.float64).sum(1)).max()
    print("ot %dx%d s=%g eta=%g: eT %.2e Err max %.2e  unconverged %d" % (n, m, s, eta, eT, err.max(), int(unc.item())))
    assert eT <= 1e-5
    assert err.max() <= max(tol, 2e-6) + mism and int(unc.item()) == 0
    dbuf = torch.full((B + 2, n, m), 7.0, device="cuda")
    Dd = bk.entropic_ot_backward(Td.contiguous(), dev(G), dbuf[1:B + 1], eta=eta)
    assert (host(dbuf[0]) == 7.0).all() and (host(dbuf[B + 1]) == 7.0).all()
    D = host(Dd).astype(np.float64)
    D_o = ot.backward(T_o, G.astype(np.float64), eta)
    e1, e2 = d_errors(D * eta, D_o * eta, G)
    assert np.isfinite(D).all() and e1 <= 1e-4 and e2 <= 1e-4 * a.max(), (e1, e2)


@pytest.mark.parametrize("n", [2, 3, 5, 6, 7])
def test_birkhoff_projection_any_n(n):
    """unit marginals (a = b = NULL) at sizes other than 4 and 8: the n x n Birkhoff projection of exp(H), C = -H"""
    H, G = inputs.normal_n(2048 + 1, n, 3.0, config=8, sub=n)
    P_o = ot.birkhoff_forward(H.astype(np.float64))
    P = host(bk.entropic_ot_forward(dev(-H), tol=1e-6 * max(n, 4) / 4, max_iter=60)).astype(np.float64)
    assert np.abs(P - P_o).max() <= 1e-5
    assert ot.marginal_err(P).max() <= 1e-6 * max(n, 4) / 4 + 1e-7 * n
    dH = -host(bk.entropic_ot_backward(dev(P.astype(np.float32)), dev(G))).astype(np.float64)
    dH_o = ot.birkhoff_backward(P_o, G.astype(np.float64))
    e1, e2 = d_errors(dH, dH_o, G)
    assert e1 <= 1e-4 and e2 <= 1e-4, (e1, e2)


def test_two_by_two_closed_form_gpu():
    """2 x 2 with general marginals: T = [[t, a1-t], [b1-t, a2-b1+t]] with t (a2-b1+t) = K (a1-t)(b1-t),
    K = exp(-(C11+C22-C12-C21)/eta): the quadratic solved in fp64 here, not by the oracle"""
    rng = np.random.default_rng(4)
    B, eta = 999, 0.8
    C = (rng.normal(size=(B, 2, 2)) * 3).astype(np.float32)
    a = rng.uniform(0.2, 2.0, size=(B, 2)).astype(np.float32)
    b1 = (rng.uniform(0.05, 0.95, size=B) * a.astype(np.float64).sum(1))
    b = np.stack([b1, a.astype(np.float64).sum(1) - b1], 1).astype(np.float32)
    T = host(bk.entropic_ot_forward(dev(C), dev(a), dev(b), eta=eta, tol=1e-6, max_iter=60)).astype(np.float64)
    C64, a64, b64 = C.astype(np.float64), a.astype(np.float64), b.astype(np.float64)
    K = np.exp(-(C64[:, 0, 0] + C64[:, 1, 1] - C64[:, 0, 1] - C64[:, 1, 0]) / eta)
    a1, a2, bb = a64[:, 0], a64[:, 1], b64[:, 0]
    A, Bq, Cq = 1 - K, (a2 - bb) + K * (a1 + bb), -K * a1 * bb
    disc = np.sqrt(Bq * Bq - 4 * A * Cq)
    t = np.where(np.abs(A) < 1e-12, -Cq / Bq, (-Bq + disc) / (2 * A))
    t2 = np.where(np.abs(A) < 1e-12, t, (-Bq - disc) / (2 * A))
    lo, hi = np.maximum(0, bb - a2), np.minimum(a1, bb)
    t = np.where((t >= lo - 1e-12) & (t <= hi + 1e-12), t, t2)
    assert np.abs(T[:, 0, 0] - t).max() <= 1e-5 and np.abs(T.sum(2) - a64).max() <= 2e-6
