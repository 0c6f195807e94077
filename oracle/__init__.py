"""fp64 CPU oracle for the batched 4x4 Birkhoff projection -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2606_07574_b200 (the CUDA path) and neither imports the
other.  See oracle/birkhoff4_oracle.c for what is computed and which passage of the paper
 each function follows; oracle/numpy_ref.py holds an independent numpy
statement of the same definitions, and oracle/paper_formulas.py the paper's closed forms in fp64.

All arrays are [B,4,4] (or [B,16]); inputs of any float dtype are widened exactly to float64.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        L.bk4o_num_threads.restype = ctypes.c_int
        L.bk4o_marginal_err.argtypes = [dp, dp, ctypes.c_int64]
        L.bk4o_marginal_err.restype = None
        L.bk4o_forward.argtypes = [dp, dp, ctypes.c_int64, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                   ctypes.c_double, ip, ip, ip, dp, ctypes.c_int]
        L.bk4o_forward.restype = ctypes.c_int64
        L.bk4o_backward.argtypes = [dp, dp, dp, ctypes.c_int64, ctypes.c_double, ctypes.c_int]
        L.bk4o_backward.restype = None
        L.bk4o_sinkhorn.argtypes = [dp, dp, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        L.bk4o_sinkhorn.restype = None
        _LIB = L
    return _LIB


def _as64(x):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if a.size % 16:
        raise ValueError("expected [B,4,4]")
    return a.reshape(-1, 4, 4)


def _p(a, t=ctypes.c_double):
    return a.ctypes.data_as(ctypes.POINTER(t))


def num_threads():
    return int(lib().bk4o_num_threads())


CERTIFY = 1e-12  # a matrix whose final Err exceeds this is "oracle-uncertified" (excluded from gating)


def forward(H, tol=1e-14, max_sweeps=200, max_newton=200, nthreads=0, return_info=False):
    """P = proj^KL_{B_4}(exp(H)) (eq. (1)).  Returns P[B,4,4] float64; with
    return_info also a dict of per-matrix tier / sweeps / newton steps / Err and the uncertified count."""
    H = _as64(H)
    B = H.shape[0]
    P = np.empty_like(H)
    tier = np.zeros(B, np.int32)
    sweeps = np.zeros(B, np.int32)
    newton = np.zeros(B, np.int32)
    err = np.zeros(B, np.float64)
    bad = lib().bk4o_forward(_p(H), _p(P), B, tol, max_sweeps, max_newton, CERTIFY,
                             _p(tier, ctypes.c_int32), _p(sweeps, ctypes.c_int32),
                             _p(newton, ctypes.c_int32), _p(err), nthreads)
    if return_info:
        return P, dict(tier=tier, sweeps=sweeps, newton=newton, err=err, uncertified=int(bad))
    return P


def backward(P, G, rcond=1e-13, nthreads=0):
    """dH = J^T vec(G): minimum-norm solve of the linearised KKT system (ungauged)."""
    P = _as64(P)
    G = _as64(G)
    if P.shape != G.shape:
        raise ValueError("P and G must have the same shape")
    dH = np.empty_like(P)
    lib().bk4o_backward(_p(P), _p(G), _p(dH), P.shape[0], rcond, nthreads)
    return dH


def sinkhorn(H, n_iter=20, nthreads=0):
    """exp(H) followed by n_iter x (row-normalise, column-normalise): eq. (2) PAPER.md:76."""
    H = _as64(H)
    T = np.empty_like(H)
    lib().bk4o_sinkhorn(_p(H), _p(T), H.shape[0], n_iter, nthreads)
    return T


def marginal_err(T):
    """Err(T) = ||T1-1||_1 + ||T^T1-1||_1 per matrix, evaluated in float64."""
    T = _as64(T)
    e = np.empty(T.shape[0], np.float64)
    lib().bk4o_marginal_err(_p(T), _p(e), T.shape[0])
    return e


def marginal_err_inf(T):
    """largest single marginal deviation per matrix (the Err_inf reported beside Err, S9)."""
    T = _as64(T)
    r = np.abs(T.sum(axis=2) - 1.0)
    c = np.abs(T.sum(axis=1) - 1.0)
    return np.maximum(r.max(axis=1), c.max(axis=1))
