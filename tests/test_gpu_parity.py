"""GPU parity: libbirkhoff4.so (through the ctypes binding, i.e. through the C ABI) against the fp64 oracle.

Same seeded inputs on both sides (paper_2606_07574_b200.inputs); the oracle never sees a CUDA result.
Gates (BASELINE.json north_star; readings S9/S10 in DESIGN.md):
    max |P - P_oracle|                        <= 1e-5
    max Err(P)  (fp64 on the stored fp32 P)   <= 1e-6   at every scale
    dH: (i)  max|dH - dH_o| / max|dH_o|       <= 1e-4
        (ii) max_b ||dH_b - dH_o,b||_inf / ||G_b||_inf      <= 1e-4
"""
import itertools

import numpy as np
import pytest

torch = pytest.importorskip("torch")
from paper_2606_07574_b200 import binding as bk, inputs

pytestmark = pytest.mark.gpu

TOL_P = 1e-5
TOL_ERR = 1e-6
TOL_DH = 1e-4


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    torch.cuda.synchronize()
    return t.cpu().numpy()


MODES = ("default", "guarded")        # birkhoff4_forward, and the guarded solver for every matrix


def forward_fn(mode):
    return bk.birkhoff4_forward if mode == "default" else bk.birkhoff4_forward_guarded


def gpu_forward(H, mode="default", **kw):
    return host(forward_fn(mode)(dev(H), **kw)).astype(np.float64)


def dh_errors(dH, dH_o, G):
    e1 = np.abs(dH - dH_o).max() / max(np.abs(dH_o).max(), 1e-300)
    e2 = (np.abs(dH - dH_o).reshape(len(G), -1).max(1) / np.abs(G).reshape(len(G), -1).max(1)).max()
    return e1, e2


def check_forward_backward(oracle, H32, G32, H_for_oracle=None, P_gpu=None, err_gate=TOL_ERR, max_iter=20, mode="default"):
    """full element-by-element parity of forward and backward on one batch; returns the measured errors"""
    Ho = (H32 if H_for_oracle is None else H_for_oracle).astype(np.float64)
    P_o, info = oracle.forward(Ho, return_info=True)
    ok = info["err"] <= oracle.CERTIFY
    assert ok.all(), "oracle uncertified on %d of %d matrices" % ((~ok).sum(), len(ok))
    if P_gpu is None:
        P_gpu = forward_fn(mode)(dev(H32), max_iter=max_iter)
    P = host(P_gpu).astype(np.float64)
    assert np.isfinite(P).all()
    eP = np.abs(P - P_o)[ok].max()
    err = oracle.marginal_err(P)
    assert eP <= TOL_P, "max|P-P_o| = %.3e" % eP
    assert err.max() <= err_gate, "max Err = %.3e" % err.max()
    dH = host(bk.birkhoff4_backward(P_gpu, dev(G32))).astype(np.float64)
    dH_o = oracle.backward(P_o, G32.astype(np.float64))
    assert np.isfinite(dH).all()
    e1, e2 = dh_errors(dH[ok], dH_o[ok], G32[ok])
    if len(G32) < 256:
        e1 = 0.0        # reading (i) of S10 normalises by the batch maximum of |dH_o|: meaningless for a handful of matrices
    assert e1 <= TOL_DH and e2 <= TOL_DH, "dH errors %.3e %.3e" % (e1, e2)
    err_inf = oracle.marginal_err_inf(P).max()
    assert err_inf <= TOL_ERR, "largest single marginal deviation %.3e" % err_inf
    return dict(eP=eP, err=err.max(), err_inf=err_inf, e1=e1, e2=e2)


# ---------------------------------------------------------------------------------------------------
# config 1 (BASELINE.json configs[0]): B = 1024, N(0,1), every element against the oracle
@pytest.mark.parametrize("mode", MODES)
def test_config1_full_parity(oracle, mode):
    c = inputs.make(1)
    r = check_forward_backward(oracle, c["H"], c["G"], mode=mode)
    print("config1", mode, r)


# several tiles and a ragged tail; well-scaled and wide logits (the wide start goes through shared memory)
@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("s", [1.0, 20.0])
@pytest.mark.parametrize("B", [1, 2, 3, 31, 33, 255, 257, 1000, 4097, 70001])
def test_ragged_sizes(oracle, mode, s, B):
    H, G = inputs.normal(B, s, config=60, sub=B)
    # guard cells around the output: nothing may be written past B matrices
    buf = torch.full((B + 2, 4, 4), 7.0, device="cuda")
    forward_fn(mode)(dev(H), buf[1:B + 1], max_iter=32)
    assert (host(buf[0]) == 7.0).all() and (host(buf[B + 1]) == 7.0).all()
    check_forward_backward(oracle, H, G, P_gpu=buf[1:B + 1].contiguous())
    dbuf = torch.full((B + 2, 4, 4), 7.0, device="cuda")
    bk.birkhoff4_backward(buf[1:B + 1], dev(G), dbuf[1:B + 1])
    assert (host(dbuf[0]) == 7.0).all() and (host(dbuf[B + 1]) == 7.0).all()


def test_empty_batch():
    e = torch.empty((0, 4, 4), device="cuda")
    assert bk.birkhoff4_forward(e).shape == (0, 4, 4)
    assert bk.birkhoff4_backward(e, e).shape == (0, 4, 4)
    assert bk.birkhoff4_sinkhorn(e).shape == (0, 4, 4)
    L = bk.lib()
    assert L.birkhoff4_forward(None, None, 0, 1e-6, 20, None) == 0       # B == 0: no-op even with null pointers


# the paper's distributions (Tables 1-2) and the larger scales of config 3
@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("s", [0.1, 1.0, 2.0, 3.0, 5.0, 10.0, 30.0, 100.0])
def test_scales_parity(oracle, s, mode):
    H, G = inputs.normal(8192, s, config=61)
    r = check_forward_backward(oracle, H, G, max_iter=32, mode=mode)
    print("scale", s, mode, r)


@pytest.mark.parametrize("w", [1.0, 10.0])
def test_uniform_parity(oracle, w):
    H, G = inputs.uniform(8192, w, config=62)
    r = check_forward_backward(oracle, H, G, max_iter=32)
    print("uniform", w, r)


# config 4: bf16 logits, fp32 P; the oracle gets the exactly widened values
def test_config4_bf16_small(oracle):
    c = inputs.make(4, B=8192 + 5)
    Hb = torch.from_numpy(c["H"].view(np.int16)).cuda().view(torch.bfloat16)
    P = bk.birkhoff4_forward_bf16(Hb)
    r = check_forward_backward(oracle, c["H_f32"], c["G"], P_gpu=P)
    # the bf16 entry point equals the fp32 entry point on the widened values, bit for bit
    P32 = bk.birkhoff4_forward(dev(c["H_f32"]))
    assert torch.equal(P, P32)
    print("config4", r)


# config 5: heterogeneous structure (near-permutations, duplicate rows, ties, scales 0.1..100)
@pytest.mark.parametrize("mode", MODES)
def test_config5_small(oracle, mode):
    c = inputs.make(5, B=16384 + 7)
    r = check_forward_backward(oracle, c["H"], c["G"], max_iter=32, mode=mode)
    print("config5", mode, r)


# ---------------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times: properties over the whole
# output, the oracle on a sample of matrices
def _iteration_counts(H_dev, P_gpu, max_iter, bf16=False):
    """updates taken by every matrix and the unconverged count, from the diagnostic variant of the same kernel, whose
    projection must equal the timed variant's bit for bit"""
    iters = torch.zeros(P_gpu.shape[0], dtype=torch.int32, device="cuda")
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    P2 = (bk.birkhoff4_forward_bf16_ex if bf16 else bk.birkhoff4_forward_ex)(H_dev, max_iter=max_iter, iters=iters,
                                                                              n_unconverged=unc)
    assert torch.equal(P2, P_gpu)
    del P2
    return host(iters), int(host(unc)[0])


def _full_size(oracle, H32, G32, P_gpu, n_sample, err_gate, seed, iters=None):
    """properties over all B matrices; the oracle on a STRATIFIED sample: n_sample matrices drawn at random plus, when
    the per-matrix update counts are given, the n_sample / 2 matrices that took the most updates (which include every
    matrix that ran out of updates or stalled: where a fault that hits one matrix in 10^4 would live)"""
    B = H32.shape[0]
    P = host(P_gpu)
    assert np.isfinite(P).all()
    P64 = P.astype(np.float64)
    rows = np.abs(P64.sum(2) - 1).sum(1)
    cols = np.abs(P64.sum(1) - 1).sum(1)
    err = rows + cols                                                  # PAPER.md:323, all B matrices
    assert err.max() <= err_gate, "max Err over %d matrices = %.3e" % (B, err.max())
    assert P.min() >= 0.0
    dH_gpu = bk.birkhoff4_backward(P_gpu, dev(G32))
    dH = host(dH_gpu).astype(np.float64)
    assert np.isfinite(dH).all()
    scale = np.abs(G32).reshape(B, -1).max(1).astype(np.float64)
    # P11: row and column sums of dH vanish (every matrix)
    assert (np.abs(dH.sum(1)).max(1) / scale).max() < 2e-5
    assert (np.abs(dH.sum(2)).max(1) / scale).max() < 2e-5
    idx = np.random.default_rng(seed).choice(B, n_sample, replace=False)
    idx[0], idx[-1] = 0, B - 1
    if iters is not None:
        assert iters.shape == (B,)
        hardest = np.argsort(-iters.astype(np.int64), kind="stable")[:n_sample // 2]
        idx = np.concatenate([idx, hardest])
    idx = np.unique(idx)
    P_o, info = oracle.forward(H32[idx].astype(np.float64), return_info=True)
    ok = info["err"] <= oracle.CERTIFY
    assert ok.all(), "oracle uncertified on %d of %d sampled matrices" % ((~ok).sum(), len(ok))
    eP = np.abs(P64[idx] - P_o)[ok].max()
    assert eP <= TOL_P, "max|P-P_o| = %.3e" % eP
    dH_o = oracle.backward(P_o, G32[idx].astype(np.float64))
    e1, e2 = dh_errors(dH[idx][ok], dH_o[ok], G32[idx][ok])
    assert e1 <= TOL_DH and e2 <= TOL_DH
    err_inf = max(np.abs(P64.sum(2) - 1).max(), np.abs(P64.sum(1) - 1).max())
    assert err_inf <= TOL_ERR
    return dict(eP=eP, err=err.max(), err_mean=err.mean(), err_inf=err_inf, e1=e1, e2=e2, compared=len(idx),
                most_updates=None if iters is None else int(iters.max()))


def test_config2_full_size(oracle):
    c = inputs.make(2)
    Hd = dev(c["H"])
    P = bk.birkhoff4_forward(Hd)
    iters, unc = _iteration_counts(Hd, P, 20)
    print("config2", _full_size(oracle, c["H"], c["G"], P, 8192, TOL_ERR, 2, iters), "unconverged", unc)


@pytest.mark.parametrize("s", [10.0, 30.0, 100.0])
def test_config3_full_size(oracle, s):
    c = inputs.make(3, s=s)
    hist = torch.zeros(64, dtype=torch.int64, device="cuda")
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    iters = torch.zeros(c["B"], dtype=torch.int32, device="cuda")
    P = bk.birkhoff4_forward_ex(dev(c["H"]), max_iter=32, iters=iters, hist=hist, n_unconverged=unc)
    r = _full_size(oracle, c["H"], c["G"], P, 2048, TOL_ERR, 3, host(iters))
    h = host(hist)
    assert h.sum() == c["B"]
    print("config3 s=%g" % s, r, "mean iters %.2f" % ((h * np.arange(64)).sum() / h.sum()), "max", np.nonzero(h)[0].max(),
          "unconverged", int(host(unc)[0]))


def test_config4_full_size(oracle):
    c = inputs.make(4)
    Hb = torch.from_numpy(c["H"].view(np.int16)).cuda().view(torch.bfloat16)
    P = bk.birkhoff4_forward_bf16(Hb)
    iters, unc = _iteration_counts(Hb, P, 20, bf16=True)
    del Hb
    print("config4", _full_size(oracle, c["H_f32"], c["G"], P, 4096, TOL_ERR, 4, iters), "unconverged", unc)


def test_bf16_diagnostics_match_fp32_path():
    """bf16 logits widen exactly, so the bf16 entry points must equal the fp32 ones on the widened values"""
    c = inputs.make(4, B=50001)
    Hb = torch.from_numpy(c["H"].view(np.int16)).cuda().view(torch.bfloat16)
    Hf = dev(c["H_f32"])
    ib, i32 = (torch.zeros(50001, dtype=torch.int32, device="cuda") for _ in range(2))
    hb, h32 = (torch.zeros(64, dtype=torch.int64, device="cuda") for _ in range(2))
    Pb = bk.birkhoff4_forward_bf16_ex(Hb, iters=ib, hist=hb)
    P32 = bk.birkhoff4_forward_ex(Hf, iters=i32, hist=h32)
    assert torch.equal(Pb, P32) and torch.equal(ib, i32) and torch.equal(hb, h32)
    assert torch.equal(bk.birkhoff4_forward_bf16(Hb), Pb)
    assert int(hb.sum()) == 50001


def test_config5_full_size(oracle):
    c = inputs.make(5)
    Hd = dev(c["H"])
    P = bk.birkhoff4_forward(Hd, max_iter=32)
    iters, unc = _iteration_counts(Hd, P, 32)
    print("config5", _full_size(oracle, c["H"], c["G"], P, 8192, TOL_ERR, 5, iters), "unconverged", unc)


# ---------------------------------------------------------------------------------------------------
# properties of the CUDA forward that hold at any size
def test_separable_gives_uniform_gpu():
    rng = np.random.default_rng(1)
    a = rng.normal(size=(64, 4, 1)) * 5
    b = rng.normal(size=(64, 1, 4)) * 5
    H = np.concatenate([a + b, np.full((1, 4, 4), 3.25), np.zeros((1, 4, 4)), np.full((1, 4, 4), -1e4)]).astype(np.float32)
    P = gpu_forward(H)
    # fp32 H = a+b is separable only up to its own rounding (ulp(20) ~ 2e-6)
    assert np.abs(P[:64] - 0.25).max() < 5e-6
    assert np.abs(P[64:] - 0.25).max() < 1e-7


def test_permutation_equivariance_gpu():
    perms = list(itertools.permutations(range(4)))
    for s in (1.0, 10.0):
        H = inputs.normal(4, s, config=63)[0]
        Hp = np.array([H[b][np.ix_(pr, pc)] for b in range(4) for pr in perms for pc in perms])
        P = gpu_forward(H, max_iter=32)
        want = np.array([P[b][np.ix_(pr, pc)] for b in range(4) for pr in perms for pc in perms])
        assert np.abs(gpu_forward(Hp, max_iter=32) - want).max() < 2e-6


def test_assignment_limit_gpu():
    H = inputs.normal(1 << 16, 100.0, config=64)[0]
    perms = np.array(list(itertools.permutations(range(4))))
    tot = np.stack([sum(H[:, i, p[i]].astype(np.float64) for i in range(4)) for p in perms], axis=1)
    order = np.sort(tot, axis=1)
    keep = order[:, -1] - order[:, -2] > 160.0
    best = perms[np.argmax(tot, axis=1)]
    want = np.zeros((len(H), 4, 4))
    for i in range(4):
        want[np.arange(len(H)), i, best[:, i]] = 1.0
    P = gpu_forward(H, max_iter=32)
    assert keep.sum() > 1000
    assert np.abs(P[keep] - want[keep]).max() < 1e-6


def test_guarded_solver_agrees_and_deterministic():
    """regression test of the nvcc mask miscompile (bk4_guarded.cuh): the guarded solver is deterministic and lands
    where the lean iteration lands"""
    H = dev(inputs.normal(1 << 16, 3.0, config=65)[0])
    a1, a2 = bk.birkhoff4_forward_guarded(H), bk.birkhoff4_forward_guarded(H)
    b1 = bk.birkhoff4_forward(H)
    assert torch.equal(a1, a2)
    assert (a1 - b1).abs().max().item() < 2e-6


def _mixed_batch(n=4096, seed=71):
    """well-scaled, large-range, row-offset, near-permutation and NaN matrices interleaved inside every warp"""
    rng = np.random.default_rng(seed)
    H = rng.normal(size=(n, 4, 4)).astype(np.float32)
    k = np.arange(n) % 8
    H[k == 1] *= 30.0                                                            # guarded solver, LP start
    H[k == 2] += (rng.normal(size=(n, 4, 1)) * 50).astype(np.float32)[k == 2]    # huge row offsets, small in-row range
    H[k == 3] *= 6.0                                                             # in-row range around the lean limit
    idx = np.nonzero(k == 4)[0]
    for i in range(4):
        H[idx, i, (i + idx) % 4] += 9.0                                          # near-permutation
    H[k == 5] += (rng.normal(size=(n, 1, 4)) * 50).astype(np.float32)[k == 5]    # huge column offsets
    return H


def test_lean_and_guarded_matrices_share_warps(oracle):
    H = _mixed_batch()
    G = np.random.default_rng(72).normal(size=H.shape).astype(np.float32)
    r = check_forward_backward(oracle, H, G, max_iter=32)
    print("mixed warps", r)
    Hn = H.copy()
    Hn[7::64, 1, 2] = np.nan                                                     # one NaN matrix in every other warp
    P = gpu_forward(Hn, max_iter=32)
    bad = np.zeros(len(H), bool)
    bad[7::64] = True
    assert np.isnan(P[bad]).all() and np.isfinite(P[~bad]).all()
    assert np.abs(P[~bad] - gpu_forward(H, max_iter=32)[~bad]).max() == 0.0      # neighbours of a NaN are untouched


def test_result_depends_on_the_matrix_alone():
    """default kernel: permuting the batch permutes the output bit for bit (no dependence on warp neighbours)"""
    H = _mixed_batch(8192, seed=73)
    P = gpu_forward(H, max_iter=32)
    perm = np.random.default_rng(74).permutation(len(H))
    Pp = gpu_forward(H[perm], max_iter=32)
    assert np.array_equal(Pp, P[perm])
    assert np.array_equal(gpu_forward(H[:1000], max_iter=32), P[:1000])          # and so does truncating it
    assert np.array_equal(gpu_forward(H, max_iter=32), P)                        # deterministic


@pytest.mark.parametrize("max_iter", [32, 3, 2])
def test_schedule_of_free_updates_is_per_matrix(max_iter):
    """a wide matrix takes three plain untested updates and a narrow one two (S1/S2) whatever shares its warp:
    warps of wide matrices only, of narrow ones only, alternating ones, and one stranger per warp give the same bits"""
    n = 1 << 13
    W = inputs.normal(n, 30.0, config=3, sub=5)[0]
    N = inputs.normal(n, 1.0, config=2, sub=5)[0]
    PW, PN = gpu_forward(W, max_iter=max_iter), gpu_forward(N, max_iter=max_iter)
    mix = np.empty((2 * n, 4, 4), np.float32)
    mix[0::2], mix[1::2] = W, N
    PM = gpu_forward(mix, max_iter=max_iter)
    assert np.array_equal(PM[0::2], PW) and np.array_equal(PM[1::2], PN)
    for host, guest, Ph, Pg in ((W, N, PW, PN), (N, W, PN, PW)):
        sp, exp = host.copy(), Ph.copy()
        sp[5::32], exp[5::32] = guest[5::32], Pg[5::32]
        assert np.array_equal(gpu_forward(sp, max_iter=max_iter), exp)


def test_guarded_solver_agrees_on_mixed_batch():
    H = dev(_mixed_batch(1 << 15, seed=75))
    a = bk.birkhoff4_forward(H, max_iter=32)
    b = bk.birkhoff4_forward_guarded(H, max_iter=32)
    assert (a - b).abs().max().item() < 3e-6


def test_lean_iteration_counts_and_floor():
    """well-scaled logits: two untested updates, then tested ones; tol = 0 stops at the fp32 floor"""
    H = dev(inputs.normal(1 << 14, 1.0, config=76)[0])
    it = torch.zeros(1 << 14, dtype=torch.int32, device="cuda")
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    P = bk.birkhoff4_forward_ex(H, iters=it, n_unconverged=unc)
    assert int(it.min()) == 2 and int(it.max()) <= 5 and int(unc.item()) == 0    # (5: a polishing step that did not do, then Newton updates)
    assert float(it.float().mean()) < 2.1
    it1 = torch.zeros_like(it)
    P1 = bk.birkhoff4_forward_ex(H, max_iter=1, iters=it1)
    assert int(it1.max()) == 1 and int(it1.min()) == 1
    unc.zero_()
    Pz = bk.birkhoff4_forward_ex(H, tol=0.0, max_iter=50, iters=it, n_unconverged=unc)
    assert int(it.max()) < 12 and int(unc.item()) > 0.99 * (1 << 14)             # (almost) nobody computes Err = 0: they stop at the floor
    assert (Pz - P).abs().max().item() < 5e-7
    rows = host(P1).astype(np.float64).sum(2)
    assert np.abs(rows - 1).max() < 1e-6


# ---------------------------------------------------------------------------------------------------
# edge cases of the ABI
def test_nonfinite_inputs_are_isolated(oracle):
    H = inputs.normal(64, 1.0, config=66)[0]
    H[5, 2, 3] = np.nan
    H[17, 0, 0] = np.inf
    H[18, 1, 1] = -np.inf
    for mode in MODES:
        P = gpu_forward(H, mode=mode)
        for b in (5, 17, 18):
            assert np.isnan(P[b]).all()
        good = np.ones(64, bool)
        good[[5, 17, 18]] = False
        assert np.isfinite(P[good]).all()
        assert np.abs(P[good] - oracle.forward(H[good])).max() < TOL_P


def test_extreme_magnitudes(oracle):
    rng = np.random.default_rng(3)
    H = (rng.normal(size=(512, 4, 4)) * 1e4).astype(np.float32)
    H[:8] = rng.choice([-1e4, 1e4], size=(8, 4, 4)).astype(np.float32)          # massive ties
    H[8:16] = (rng.normal(size=(8, 4, 4)) * 1e-6).astype(np.float32)
    P = gpu_forward(H, max_iter=64)
    assert np.isfinite(P).all()
    assert np.abs(P.sum(2) - 1).max() < 1e-6
    P_o, info = oracle.forward(H.astype(np.float64), return_info=True)
    ok = info["err"] <= oracle.CERTIFY
    assert np.abs(P - P_o)[ok].max() < 1e-4                                      # |H| ~ 4e4: ulp(H) alone is 4e-3


def test_max_iter_and_tol_semantics():
    H = dev(inputs.normal(4096, 1.0, config=67)[0])
    it = torch.zeros(4096, dtype=torch.int32, device="cuda")
    P0 = bk.birkhoff4_forward_ex(H, max_iter=0, iters=it)
    assert int(it.max()) == 0
    rows = host(P0).astype(np.float64).sum(2)
    assert np.abs(rows - 1).max() < 1e-6                                         # rows normalised even at max_iter = 0
    for cap in (1, 2, 3):
        bk.birkhoff4_forward_ex(H, max_iter=cap, iters=it)
        assert int(it.max()) <= cap
    # looser tolerance never takes more updates; tol = 0 runs to the floor and still terminates
    it_loose, it_tight, it_zero = (torch.zeros(4096, dtype=torch.int32, device="cuda") for _ in range(3))
    bk.birkhoff4_forward_ex(H, tol=1e-3, iters=it_loose)
    bk.birkhoff4_forward_ex(H, tol=1e-6, iters=it_tight)
    Pz = bk.birkhoff4_forward_ex(H, tol=0.0, max_iter=50, iters=it_zero)
    assert bool((it_loose <= it_tight).all())
    assert int(it_zero.max()) < 50
    assert np.isfinite(host(Pz)).all()


def test_diagnostics_consistent():
    c = inputs.make(5, B=50001)
    H = dev(c["H"])
    it = torch.zeros(50001, dtype=torch.int32, device="cuda")
    hist = torch.zeros(64, dtype=torch.int64, device="cuda")
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    for mode in MODES:
        it.zero_(), hist.zero_(), unc.zero_()
        fn = bk.birkhoff4_forward_ex if mode == "default" else bk.birkhoff4_forward_guarded
        P = fn(H, max_iter=32, iters=it, hist=hist, n_unconverged=unc)
        P_plain = bk.birkhoff4_forward(H, max_iter=32) if mode == "default" else bk.birkhoff4_forward_guarded(H, max_iter=32)
        h = host(hist)
        assert h.sum() == 50001
        assert (np.bincount(np.minimum(host(it), 63), minlength=64) == h).all()
        assert torch.equal(P, P_plain)                                           # diagnostics do not change P
        assert 0 <= int(host(unc)[0]) <= 50001


def test_aliasing_in_place():
    H, G = inputs.normal(5000, 1.0, config=68)
    Hd, Gd = dev(H), dev(G)
    P = bk.birkhoff4_forward(Hd)
    dH = bk.birkhoff4_backward(P, Gd)
    X = Hd.clone()
    bk.birkhoff4_forward(X, X)                                                   # P == H
    assert torch.equal(X, P)
    Y = Gd.clone()
    bk.birkhoff4_backward(P, Y, Y)                                               # dH == dP
    assert torch.equal(Y, dH)


def test_invalid_arguments_return_einval():
    L = bk.lib()
    import ctypes
    t = torch.zeros((4, 4, 4), device="cuda")
    p = ctypes.c_void_p(t.data_ptr())
    mis = ctypes.c_void_p(t.data_ptr() + 4)
    nan = float("nan")
    assert L.birkhoff4_forward(p, p, -1, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward(None, p, 4, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward(p, None, 4, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward(mis, p, 1, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward(p, p, 4, -1.0, 20, None) == 1
    assert L.birkhoff4_forward(p, p, 4, nan, 20, None) == 1
    assert L.birkhoff4_forward(p, p, 4, 1e-6, -1, None) == 1
    assert L.birkhoff4_backward(p, None, p, 4, None) == 1
    assert L.birkhoff4_backward(p, mis, p, 1, None) == 1
    assert L.birkhoff4_sinkhorn(p, p, 4, -1, None) == 1
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_forward(torch.zeros(4, 4, 4))                               # CPU tensor: no CPU path
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_forward(torch.zeros(4, 4, 4, device="cuda", dtype=torch.float64))
    # an output (or second input) of the wrong size never reaches the library
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_forward(t, torch.zeros((3, 4, 4), device="cuda"))
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_backward(t, torch.zeros((5, 4, 4), device="cuda"))
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_backward(t, t, torch.zeros((3, 4, 4), device="cuda"))
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_sinkhorn(t, torch.zeros((3, 4, 4), device="cuda"))
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_forward_ex(t, iters=torch.zeros(3, dtype=torch.int32, device="cuda"))
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_forward_host(torch.zeros(4, 4, 4), torch.zeros(3, 4, 4))


def test_non_default_stream():
    H, G = inputs.normal(1 << 16, 1.0, config=69)
    Hd, Gd = dev(H), dev(G)
    ref = bk.birkhoff4_forward(Hd)
    ref_d = bk.birkhoff4_backward(ref, Gd)
    torch.cuda.synchronize()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        P = bk.birkhoff4_forward(Hd)
        dH = bk.birkhoff4_backward(P, Gd)
    st.synchronize()
    assert torch.equal(P, ref) and torch.equal(dH, ref_d)


def test_legacy_default_stream_and_stream_order():
    """stream 0 through the raw C ABI, and a dependent chain on one stream (forward -> backward -> forward in place):
    programmatic dependent launch must not let a kernel read what its predecessor has not written yet"""
    import ctypes
    H, G = inputs.normal((1 << 18) + 3, 2.0, config=70)
    Hd, Gd = dev(H), dev(G)
    ref = bk.birkhoff4_forward(Hd)
    ref_d = bk.birkhoff4_backward(ref, Gd)
    ref_2 = bk.birkhoff4_forward(ref_d)
    torch.cuda.synchronize()
    L, B = bk.lib(), Hd.shape[0]
    P, dH = torch.empty_like(Hd), torch.empty_like(Hd)
    torch.cuda.synchronize()
    null = ctypes.c_void_p(0)
    assert L.birkhoff4_forward(ctypes.c_void_p(Hd.data_ptr()), ctypes.c_void_p(P.data_ptr()), B, 1e-6, 20, null) == 0
    assert L.birkhoff4_backward(ctypes.c_void_p(P.data_ptr()), ctypes.c_void_p(Gd.data_ptr()),
                                ctypes.c_void_p(dH.data_ptr()), B, null) == 0
    torch.cuda.synchronize()
    assert torch.equal(P, ref) and torch.equal(dH, ref_d)
    for _ in range(20):                                                          # back-to-back dependent launches
        P.zero_(), dH.zero_()
        bk.birkhoff4_forward(Hd, P)
        bk.birkhoff4_backward(P, Gd, dH)
        bk.birkhoff4_forward(dH, dH)
        torch.cuda.synchronize()
        assert torch.equal(P, ref) and torch.equal(dH, ref_2)


# ---------------------------------------------------------------------------------------------------
# backward on its own: fed the oracle's P (rounded to fp32), including near-permutation P where the
# paper's Delta is singular (S7)
@pytest.mark.parametrize("s", [1.0, 10.0, 100.0])
def test_backward_alone(oracle, s):
    H, G = inputs.normal(8192, s, config=70)
    P_o = oracle.forward(H.astype(np.float64))
    dH = host(bk.birkhoff4_backward(dev(P_o.astype(np.float32)), dev(G))).astype(np.float64)
    dH_o = oracle.backward(P_o, G.astype(np.float64))
    assert np.isfinite(dH).all()
    e1, e2 = dh_errors(dH, dH_o, G)
    assert e1 <= TOL_DH and e2 <= TOL_DH
    print("backward alone s=%g" % s, e1, e2)


def test_backward_exact_permutation_and_additive_G():
    P = np.zeros((24, 4, 4), np.float32)
    for k, p in enumerate(itertools.permutations(range(4))):
        P[k, np.arange(4), list(p)] = 1.0
    G = inputs.normal(24, 1.0, config=71)[1]
    dH = host(bk.birkhoff4_backward(dev(P), dev(G)))
    assert np.isfinite(dH).all() and np.abs(dH).max() < 1e-5                     # a vertex: the Jacobian vanishes
    # P12: G_ij = a_i + b_j gives dH = 0
    Hn = inputs.normal(1024, 2.0, config=72)[0]
    Pn = bk.birkhoff4_forward(dev(Hn))
    rng = np.random.default_rng(5)
    Ga = (rng.normal(size=(1024, 4, 1)) + rng.normal(size=(1024, 1, 4))).astype(np.float32)
    assert np.abs(host(bk.birkhoff4_backward(Pn, dev(Ga)))).max() < 5e-6


# ---------------------------------------------------------------------------------------------------
# Sinkhorn-20 baseline kernel: same convention as the oracle's eq. (2) and as the paper's Table 2
def test_sinkhorn_kernel_matches_oracle(oracle):
    for s, n_iter in ((1.0, 20), (10.0, 20), (3.0, 1), (3.0, 0)):
        H = inputs.normal(4096, s, config=73)[0]
        T = host(bk.birkhoff4_sinkhorn(dev(H), n_iter=n_iter)).astype(np.float64)
        T_o = oracle.sinkhorn(H.astype(np.float64), n_iter=n_iter)
        if n_iter == 0:                                                           # K = exp(H) up to the row shift
            T_o = T_o / T_o.max(axis=2, keepdims=True)
            T = T / T.max(axis=2, keepdims=True)
        assert np.abs(T - T_o).max() < 2e-5


def test_sinkhorn20_table2_statistics(oracle):
    import os
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_table2_sinkhorn20.txt")) as f:
        for line in f:
            if not line.startswith("#") and line.strip():
                k = line.split()
                rows[k[0]] = (float(k[1]) * 1e-3, float(k[3]) * 1e-3)
    H = inputs.normal(100000, 10.0, config=74)[0]
    err = oracle.marginal_err(host(bk.birkhoff4_sinkhorn(dev(H), n_iter=20)))
    mean, med = rows["N(0,10^2)"]
    assert abs(err.mean() - mean) < 0.05 * mean and abs(np.median(err) - med) < 0.05 * med
    H = inputs.uniform(100000, 10.0, config=74)[0]
    err = oracle.marginal_err(host(bk.birkhoff4_sinkhorn(dev(H), n_iter=20)))
    mean, med = rows["Unif(-10,10)"]
    assert abs(err.mean() - mean) < 0.05 * mean and abs(np.median(err) - med) < 0.05 * med


def test_marginal_error_not_worse_than_the_papers_solver(oracle):
    """Tables 1-2 (tests/golden/paper_tables_newton_err.txt): same distributions, N = 10^4, tol 1e-6, max_iter 20"""
    import os
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_tables_newton_err.txt")) as f:
        for line in f:
            if not line.startswith("#") and line.strip():
                k = line.split()
                u = float(k[1])
                rows[k[0]] = dict(mean=float(k[2]) * u, median=float(k[4]) * u, max=float(k[5]) * u)
    draws = {"N(0,1)": inputs.normal(10000, 1.0, config=81)[0], "Unif(-1,1)": inputs.uniform(10000, 1.0, config=82)[0],
             "N(0,10^2)": inputs.normal(10000, 10.0, config=83)[0], "Unif(-10,10)": inputs.uniform(10000, 10.0, config=84)[0]}
    for name, H in draws.items():
        err = oracle.marginal_err(gpu_forward(H, tol=1e-6, max_iter=20))
        print(name, "Err mean %.3e median %.3e max %.3e   paper %s" % (err.mean(), np.median(err), err.max(), rows[name]))
        assert err.mean() <= rows[name]["mean"] and err.max() <= rows[name]["max"]
        assert err.max() <= TOL_ERR                                              # and converged everywhere, unlike Table 2


# ---------------------------------------------------------------------------------------------------
# host-buffer entry points (the end-to-end path bench.py times): same bits as the device-pointer calls
@pytest.mark.parametrize("B", [1, 1000, (1 << 18) + 17, (1 << 19) * 3 + 5])
def test_host_calls_match_device_calls(B):
    H, G = inputs.normal(B, 2.0, config=75)
    Hd, Gd = dev(H), dev(G)
    P = bk.birkhoff4_forward(Hd)
    dH = bk.birkhoff4_backward(P, Gd)
    Hh, Gh = torch.from_numpy(H).pin_memory(), torch.from_numpy(G).pin_memory()
    Ph = bk.birkhoff4_forward_host(Hh)
    assert torch.equal(Ph, P.cpu())
    assert torch.equal(bk.birkhoff4_backward_host(Ph, Gh), dH.cpu())
    P2, dH2 = bk.birkhoff4_forward_backward_host(Hh, Gh)
    assert torch.equal(P2, P.cpu()) and torch.equal(dH2, dH.cpu())
    _, dH3 = bk.birkhoff4_forward_backward_host(torch.from_numpy(H), torch.from_numpy(G), want_P=False)   # pageable
    assert torch.equal(dH3, dH.cpu())
    bk.birkhoff4_host_release()


# ---------------------------------------------------------------------------------------------------
# fused forward + backward: bit-identical to the two separate calls
@pytest.mark.parametrize("s", [1.0, 30.0])
@pytest.mark.parametrize("B", [1, 33, 1000, 70001])
def test_fused_forward_backward_equals_separate_calls(oracle, B, s):
    H, G = inputs.normal(B, s, config=90, sub=B)
    Hd, Gd = dev(H), dev(G)
    P = bk.birkhoff4_forward(Hd, max_iter=32)
    dH = bk.birkhoff4_backward(P, Gd)
    # guard cells: nothing is written past B matrices
    pbuf, dbuf = torch.full((B + 2, 4, 4), 7.0, device="cuda"), torch.full((B + 2, 4, 4), 7.0, device="cuda")
    bk.birkhoff4_forward_backward(Hd, Gd, pbuf[1:B + 1], dbuf[1:B + 1], max_iter=32)
    assert torch.equal(pbuf[1:B + 1], P) and torch.equal(dbuf[1:B + 1], dH)
    for buf in (pbuf, dbuf):
        assert (host(buf[0]) == 7.0).all() and (host(buf[B + 1]) == 7.0).all()
    none, dH2 = bk.birkhoff4_forward_backward(Hd, Gd, want_P=False, max_iter=32)    # P never written
    assert none is None and torch.equal(dH2, dH)
    X, Y = Hd.clone(), Gd.clone()
    bk.birkhoff4_forward_backward(X, Y, X, Y, max_iter=32)                          # P == H and dH == dP
    assert torch.equal(X, P) and torch.equal(Y, dH)
    if B >= 1000:                                                                   # and against the oracle
        P_o = oracle.forward(H.astype(np.float64))
        e1, e2 = dh_errors(host(dH2).astype(np.float64), oracle.backward(P_o, G.astype(np.float64)), G)
        assert e1 <= TOL_DH and e2 <= TOL_DH


def test_fused_forward_backward_mixed_and_nonfinite():
    H = _mixed_batch(8192, seed=91)
    H[5::64, 0, 1] = np.nan
    G = np.random.default_rng(92).normal(size=H.shape).astype(np.float32)
    Hd, Gd = dev(H), dev(G)
    P = bk.birkhoff4_forward(Hd, max_iter=32)
    dH = bk.birkhoff4_backward(P, Gd)
    P2, dH2 = bk.birkhoff4_forward_backward(Hd, Gd, max_iter=32)
    assert torch.equal(torch.nan_to_num(P2, nan=-1.0), torch.nan_to_num(P, nan=-1.0))
    assert torch.equal(torch.nan_to_num(dH2, nan=-1.0), torch.nan_to_num(dH, nan=-1.0))
    assert bool(torch.isnan(P2[5::64]).all()) and bool(torch.isfinite(P2[6::64]).all())
    L = bk.lib()
    import ctypes
    p = ctypes.c_void_p(Hd.data_ptr())
    assert L.birkhoff4_forward_backward(p, None, p, p, 4, 1e-6, 20, None) == 1       # dP missing
    assert L.birkhoff4_forward_backward(p, p, None, None, 4, 1e-6, 20, None) == 1    # dH missing
    assert L.birkhoff4_forward_backward(None, None, None, None, 0, 1e-6, 20, None) == 0


# ---------------------------------------------------------------------------------------------------
# fused consumer: Y_b = proj(exp(H_b)) X_b in one kernel.  The oracle is the
# definition: the fp64 oracle's P times X (a matrix product, numpy).
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("B,C", [(1, 8), (129, 64), (1000, 1024), (4097, 200)])
def test_fused_mix_matches_oracle(oracle, B, C, dtype):
    H = inputs.normal(B, 3.0, config=98, sub=B)[0]
    X = np.random.Generator(np.random.Philox(key=inputs.SEED + 99 + B)).standard_normal((B, 4, C), dtype=np.float32)
    Hd = dev(H)
    if dtype == "bf16":
        Xb = inputs.f32_to_bf16_bits(X)
        X = inputs.bf16_bits_to_f32(Xb)                                 # the oracle sees what the kernel sees
        Xd = torch.from_numpy(Xb.view(np.int16)).cuda().view(torch.bfloat16)
    else:
        Xd = dev(X)
    ybuf = torch.full((B + 2, 4, C), 7.0, device="cuda", dtype=Xd.dtype)
    Y, P = bk.birkhoff4_forward_mix(Hd, Xd, ybuf[1:B + 1], want_P=True, max_iter=32)
    assert (ybuf[0].float() == 7.0).all() and (ybuf[B + 1].float() == 7.0).all()   # guard cells
    assert torch.equal(P, bk.birkhoff4_forward(Hd, max_iter=32))        # the same projection, bit for bit
    P_o = oracle.forward(H.astype(np.float64))
    Y_o = np.einsum("bij,bjc->bic", P_o, X.astype(np.float64))
    Yh = host(Y.float()).astype(np.float64)
    tol = 2.0 ** -8 if dtype == "bf16" else 2e-6                        # bf16: half an ulp of the stored result
    assert (np.abs(Yh - Y_o) <= tol * np.maximum(np.abs(Y_o), 1.0) + 1e-6).all()
    Y2, none = bk.birkhoff4_forward_mix(Hd, Xd, max_iter=32)            # P not requested: never written
    assert none is None and torch.equal(Y2, Y)


# backward of the fused consumer (PAPER.md:46-50 differentiated, then section 4.2) in one kernel.  The
# oracle is the definition: dX = P_o^T dY and G = dY X^T as fp64 matrix products (numpy), dH = the oracle's backward at
# (P_o, G).
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("B,C", [(1, 8), (129, 64), (1000, 1024), (4097, 200), (300, 4096)])
def test_fused_mix_backward_matches_oracle(oracle, B, C, dtype):
    H = inputs.normal(B, 3.0, config=98, sub=B)[0]
    rng = np.random.Generator(np.random.Philox(key=inputs.SEED + 199 + B))
    X = rng.standard_normal((B, 4, C), dtype=np.float32)
    dY = rng.standard_normal((B, 4, C), dtype=np.float32)
    Hd = dev(H)
    if dtype == "bf16":
        Xb, dYb = inputs.f32_to_bf16_bits(X), inputs.f32_to_bf16_bits(dY)
        X, dY = inputs.bf16_bits_to_f32(Xb), inputs.bf16_bits_to_f32(dYb)          # the oracle sees what the kernel sees
        Xd = torch.from_numpy(Xb.view(np.int16)).cuda().view(torch.bfloat16)
        dYd = torch.from_numpy(dYb.view(np.int16)).cuda().view(torch.bfloat16)
    else:
        Xd, dYd = dev(X), dev(dY)
    xbuf = torch.full((B + 2, 4, C), 7.0, device="cuda", dtype=Xd.dtype)
    hbuf = torch.full((B + 2, 4, 4), 7.0, device="cuda")
    dX, dH, P = bk.birkhoff4_backward_mix(Hd, Xd, dYd, xbuf[1:B + 1], hbuf[1:B + 1], want_P=True, max_iter=32)
    for buf in (xbuf, hbuf):                                                       # guard cells
        assert (buf[0].float() == 7.0).all() and (buf[B + 1].float() == 7.0).all()
    assert torch.equal(P, bk.birkhoff4_forward(Hd, max_iter=32))                   # the same projection, bit for bit
    P_o = oracle.forward(H.astype(np.float64))
    dX_o = np.einsum("bij,bic->bjc", P_o, dY.astype(np.float64))
    G_o = np.einsum("bic,bjc->bij", dY.astype(np.float64), X.astype(np.float64))
    dH_o = oracle.backward(P_o, G_o)
    dXh = host(dX.float()).astype(np.float64)
    tol = 2.0 ** -8 if dtype == "bf16" else 2e-6
    assert (np.abs(dXh - dX_o) <= tol * np.maximum(np.abs(dX_o), 1.0) + 1e-6).all()
    dHh = host(dH).astype(np.float64)
    assert np.isfinite(dHh).all()
    e1, e2 = dh_errors(dHh, dH_o, G_o)
    if B < 256:
        e1 = 0.0
    assert e1 <= TOL_DH and e2 <= TOL_DH, (e1, e2)
    # against the library's own separate calls: G formed by torch in fp32, then birkhoff4_backward
    G32 = torch.einsum("bic,bjc->bij", dYd.float(), Xd.float()).contiguous()
    dH_sep = host(bk.birkhoff4_backward(P, G32)).astype(np.float64)
    assert np.abs(dHh - dH_sep).max() <= 1e-4 * max(np.abs(dH_o).max(), 1.0)
    dX2, dH2, none = bk.birkhoff4_backward_mix(Hd, Xd, dYd, max_iter=32)             # P not requested: never written
    assert none is None and torch.equal(dX2, dX) and torch.equal(dH2, dH)


def test_fused_mix_backward_edges():
    H = dev(inputs.normal(64, 1.0, config=98)[0])
    X = torch.ones((64, 4, 16), device="cuda")
    L = bk.lib()
    import ctypes
    ph, px, pd = ctypes.c_void_p(H.data_ptr()), ctypes.c_void_p(X.data_ptr()), ctypes.c_void_p(torch.empty_like(H).data_ptr())
    assert L.birkhoff4_backward_mix(ph, px, px, px, pd, None, 64, 6, 1e-6, 20, None) == 1       # C not a multiple of 4
    assert L.birkhoff4_backward_mix(ph, px, None, px, pd, None, 64, 16, 1e-6, 20, None) == 1    # null dY
    assert L.birkhoff4_backward_mix(ph, px, px, px, None, None, 64, 16, 1e-6, 20, None) == 1    # null dH
    assert L.birkhoff4_backward_mix(None, None, None, None, None, None, 0, 16, 1e-6, 20, None) == 0
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_backward_mix(H, X, torch.ones((63, 4, 16), device="cuda"))
    Hn = H.clone()
    Hn[3, 1, 1] = float("nan")
    dX, dH, _ = bk.birkhoff4_backward_mix(Hn, X, X)
    assert torch.isnan(dX[3]).all() and torch.isnan(dH[3]).all()
    ok = torch.ones(64, dtype=torch.bool, device="cuda")
    ok[3] = False
    dX0, dH0, _ = bk.birkhoff4_backward_mix(H, X, X)
    assert torch.equal(dX[ok], dX0[ok]) and torch.equal(dH[ok], dH0[ok])              # the other tokens are untouched
    e = torch.empty((0, 4, 4), device="cuda")
    assert bk.birkhoff4_backward_mix(e, torch.empty((0, 4, 16), device="cuda"), torch.empty((0, 4, 16), device="cuda"))[1].shape == (0, 4, 4)


def test_fused_mix_edges():
    H = dev(inputs.normal(64, 1.0, config=98)[0])
    X = torch.zeros((64, 4, 16), device="cuda")
    L = bk.lib()
    import ctypes
    ph, px = ctypes.c_void_p(H.data_ptr()), ctypes.c_void_p(X.data_ptr())
    assert L.birkhoff4_forward_mix(ph, px, px, None, 64, 6, 1e-6, 20, None) == 1      # C not a multiple of 4
    assert L.birkhoff4_forward_mix(ph, None, px, None, 64, 16, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward_mix(ph, ctypes.c_void_p(X.data_ptr() + 4), px, None, 64, 16, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward_mix(None, None, None, None, 0, 16, 1e-6, 20, None) == 0
    with pytest.raises(bk.Birkhoff4Error):
        bk.birkhoff4_forward_mix(H, torch.zeros((63, 4, 16), device="cuda"))
    Hn = H.clone()
    Hn[3, 0, 0] = float("nan")
    Y, _ = bk.birkhoff4_forward_mix(Hn, torch.ones((64, 4, 16), device="cuda"))
    assert bool(torch.isnan(Y[3]).all()) and bool(torch.isfinite(Y[4]).all())
    assert (Y[4].sum(0) - 4.0).abs().max().item() < 1e-5               # columns of P sum to 1: the mix conserves the stream sum
