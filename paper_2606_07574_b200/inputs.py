"""Seeded synthetic workloads for the batched 4x4 Birkhoff projection (BASELINE.json `configs`).

This module holds NONE of the method's arithmetic: it only draws the input tensors (logits H and
upstream gradients G = dL/dP) with the shapes, value distributions and structure of the paper's
workloads (N x 4 x 4 iid tensors) as extended by BASELINE.json.  It is the
one module both the CUDA path's tests/bench and the oracle's tests are fed from.  numpy only (CPU,
counter-based Philox), so the same bits reach the GPU path and the fp64 oracle.

Recipe (also in DESIGN.md):
  seed   Philox(key = SEED + config index [+ 1000*sub-batch]), SEED = 20260607
  1      B=1024        H, G ~ N(0,1) fp32
  2      B=2^20        H, G ~ N(0,1) fp32
  3      B=2^20 x 3    H ~ N(0, s^2), s in {10, 30, 100} (one sub-batch per s), G ~ N(0,1)
  4      B=2^24        H = bf16(N(0, 4)) stored as uint16 bit patterns, G ~ N(0,1) fp32
  5      B=2^22        per-matrix class (iid, so classes mix inside warps) and scale
                       sigma = exp(U(ln 0.1, ln 100)):
                         50 %   sigma * N(0,1)
                         25 %   N(0,1) with +8 on the 4 entries of a uniformly random permutation
                         12.5 % sigma * N(0,1) with one random row copied onto another
                         12.5 % sigma * N(0,1) with, in every row, the 2nd-largest entry set equal
                                to the largest (ties)
"""
import numpy as np

SEED = 20260607

DEFAULT_B = {1: 1 << 10, 2: 1 << 20, 3: 1 << 20, 4: 1 << 24, 5: 1 << 22}
CONFIG3_SCALES = (10.0, 30.0, 100.0)


def _rng(config, sub=0):
    return np.random.Generator(np.random.Philox(key=SEED + config + 1000 * sub))


def f32_to_bf16_bits(x):
    """round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (dtype conversion only)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b):
    """exact widening of bf16 bit patterns to fp32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal(B, scale=1.0, config=0, sub=0):
    """H, G: H ~ N(0, scale^2), G ~ N(0,1), both fp32 [B,4,4]."""
    rng = _rng(config, sub)
    H = rng.standard_normal((B, 4, 4), dtype=np.float32)
    if scale != 1.0:
        H *= np.float32(scale)
    G = rng.standard_normal((B, 4, 4), dtype=np.float32)
    return H, G


def uniform(B, half_width=1.0, config=0, sub=0):
    """H ~ Unif(-w, w) (the paper's second distribution), G ~ N(0,1)."""
    rng = _rng(config, sub)
    H = ((rng.random((B, 4, 4), dtype=np.float32) * 2 - 1) * np.float32(half_width)).astype(np.float32)
    G = rng.standard_normal((B, 4, 4), dtype=np.float32)
    return H, G


def normal_n(B, n, scale=1.0, config=8, sub=0):
    """H, G for the n x n Birkhoff projection (n = 4 or 8): H ~ N(0, scale^2), G ~ N(0,1), fp32 [B,n,n]."""
    rng = _rng(config, sub)
    H = rng.standard_normal((B, n, n), dtype=np.float32)
    if scale != 1.0:
        H *= np.float32(scale)
    G = rng.standard_normal((B, n, n), dtype=np.float32)
    return H, G


def ot_problem(B, n, m, scale=1.0, config=9, sub=0, uniform_marginals=False):
    """A batch of small entropic-OT problems: cost M ~ N(0, scale^2) [B,n,m], marginals a [B,n] and
    b [B,m] positive with equal sums (Gamma(4) draws, rescaled so that sum a = sum b = max(n, m); all ones when
    uniform_marginals and n == m), upstream gradient G ~ N(0,1).  All fp32; b is rescaled in fp64 and rounded, so the
    two sums agree to fp32 rounding."""
    rng = _rng(config, sub)
    M = (rng.standard_normal((B, n, m), dtype=np.float32) * np.float32(scale)).astype(np.float32)
    G = rng.standard_normal((B, n, m), dtype=np.float32)
    if uniform_marginals and n == m:
        return M, np.ones((B, n), np.float32), np.ones((B, m), np.float32), G
    a = rng.gamma(4.0, size=(B, n))
    b = rng.gamma(4.0, size=(B, m))
    tot = float(max(n, m))
    a = (a * (tot / a.sum(1, keepdims=True))).astype(np.float32)
    b = (b * (a.astype(np.float64).sum(1, keepdims=True) / b.sum(1, keepdims=True))).astype(np.float32)
    return M, a, b, G


def heterogeneous(B, config=5, sub=0, sort_by_class=False):
    """config 5.  Returns H, G, cls (0 scaled normal, 1 near-permutation, 2 duplicate row, 3 ties)."""
    rng = _rng(config, sub)
    H = rng.standard_normal((B, 4, 4), dtype=np.float32)
    G = rng.standard_normal((B, 4, 4), dtype=np.float32)
    cls = rng.choice(4, size=B, p=[0.5, 0.25, 0.125, 0.125]).astype(np.int8)
    sigma = np.exp(rng.uniform(np.log(0.1), np.log(100.0), size=B)).astype(np.float32)
    scaled = cls != 1
    H[scaled] *= sigma[scaled, None, None]
    # near-permutation: +8 on a uniformly random permutation's entries
    idx = np.nonzero(cls == 1)[0]
    perm = rng.permuted(np.tile(np.arange(4), (idx.size, 1)), axis=1)
    for i in range(4):
        H[idx, i, perm[:, i]] += np.float32(8.0)
    # duplicate rows: copy row src onto row dst != src
    idx = np.nonzero(cls == 2)[0]
    src = rng.integers(0, 4, size=idx.size)
    dst = (src + rng.integers(1, 4, size=idx.size)) % 4
    H[idx, dst, :] = H[idx, src, :]
    # ties: in every row the second-largest entry is set equal to the largest
    idx = np.nonzero(cls == 3)[0]
    sub_H = H[idx]
    order = np.argsort(sub_H, axis=2)
    top, second = order[:, :, 3], order[:, :, 2]
    ii, rr = np.meshgrid(np.arange(idx.size), np.arange(4), indexing="ij")
    sub_H[ii, rr, second] = sub_H[ii, rr, top]
    H[idx] = sub_H
    if sort_by_class:
        o = np.argsort(cls, kind="stable")
        H, G, cls = H[o], G[o], cls[o]
    return np.ascontiguousarray(H), np.ascontiguousarray(G), cls


def make(config, B=None, s=None, sort_by_class=False):
    """Inputs of BASELINE.json config `config` (1..5) as a dict: H (fp32, or uint16 bf16 bits for
    config 4 together with H_f32 = the exact widening), G (fp32), and the recipe parameters."""
    B = DEFAULT_B[config] if B is None else int(B)
    if config in (1, 2):
        H, G = normal(B, 1.0, config)
        return dict(config=config, B=B, H=H, G=G, scale=1.0)
    if config == 3:
        s = CONFIG3_SCALES[0] if s is None else float(s)
        sub = {10.0: 0, 30.0: 1, 100.0: 2}.get(s, 3)
        H, G = normal(B, s, config, sub)
        return dict(config=config, B=B, H=H, G=G, scale=s)
    if config == 4:
        H, G = normal(B, 2.0, config)
        bits = f32_to_bf16_bits(H)
        return dict(config=config, B=B, H=bits, H_f32=bf16_bits_to_f32(bits), G=G, scale=2.0)
    if config == 5:
        H, G, cls = heterogeneous(B, config, 0, sort_by_class)
        return dict(config=config, B=B, H=H, G=G, cls=cls)
    raise ValueError("config must be 1..5")
