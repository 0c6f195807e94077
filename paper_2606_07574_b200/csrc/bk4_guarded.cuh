// bk4_guarded.cuh -- the guarded Newton solver: the fallback for the few matrices the lean iteration
// (bk4_lean.cuh) leaves (a residual that stopped falling above the fp32 floor: none in a million N(0,1) matrices,
// about one in a thousand at N(0,30^2)), and the whole of birkhoff4_forward_guarded.  One matrix per thread, every
// lane in its own loop.
//
// It works, like the wide start of the lean iteration, on the matrix with its columns permuted so that the
// max-weight assignment sits on the diagonal (lp_dual in bk4_lean.cuh), from the LP dual potentials: there the
// exponentials, the residuals and the Hessian are all formed from differences and keep their relative accuracy
// however large the logits are (S9).
//
// Notation (paper): R = H (logits), U_ij = beta_j + R_ij, T = row-softmax(U) (eq. (10)),
// c = column sums, g = c_{1..3} - 1 (eq. (11)), Hessian = diag(c) - T_{-4}^T T_{-4}.
// T(beta) is evaluated incrementally: beta = beta0 + delta, E_ij = exp(U0_ij - U0_ii) at the base point beta0
// and v_j = exp(delta_j); T_ij = E_ij v_j / sum_k E_ik v_k is eq. (10) exactly and a Newton update is
// v_j *= exp(d_j).  When v leaves [2^-40, 2^40] the base is moved (beta0 += log v, E recomputed from the logits).
//
// Masks are 32-bit 0/1 words, never loop-carried `bool`s: for compute_100a nvcc 12.9 miscompiled an earlier form
// of this loop written with `bool` (the rejected-step path vanished from the PTX).
// tests/test_gpu_parity.py (test_guarded_solver_*) are the regression tests.
#pragma once
#include "bk4_solve.cuh"

namespace bk4 {

constexpr float kVHi = 1.099511627776e12f;      // 2^40: range of v before the base point is moved
constexpr float kVLo = 9.094947017729282e-13f;  // 2^-40

// E_im = 2^((Hc_im - Hc_ii) log2(e) + b_m - b_i), E_ii = 1: eq. (10) at the base point beta0 = b / log2(e) with the
// row shift mu_i = U_ii (the diagonal holds the assignment, which the LP potentials make the row maximum)
BK4_DEV void perm_exponentials(const float (&Hc)[16], const float (&b)[4], float (&E)[16]) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int m = 0; m < 4; ++m)
            E[4 * i + m] = (i == m) ? 1.0f : ex2_approx(fmaf(Hc[4 * i + m] - Hc[5 * i], kLog2e, b[m] - b[i]));
}

// Sinkhorn-Knopp column step (eq. (6) PAPER.md:108 with the gauge beta_4 = 0): ratio_j = c_4 / c_j from the
// column sums themselves, clamped so that the step stays finite when a column sum underflows.
BK4_DEV void column_ratios(const float (&T)[16], float (&ratio)[3]) {
    float cs[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) cs[j] = (T[j] + T[4 + j]) + (T[8 + j] + T[12 + j]);
#pragma unroll
    for (int j = 0; j < 3; ++j) ratio[j] = fminf(fmaxf(cs[3] * rcp_approx(cs[j]), kVLo), kVHi);
}

// Guarded Newton on f(beta_1..3) (eq. (8); iteration PAPER.md:164-168), S2:
//   start     the LP dual potentials xs (permuted column order, log2 units) and one Sinkhorn-Knopp column step
//   step      d = -Hessian^{-1} g  (eqs. (9), (11), (12))
//   guard     the full step stands iff the column residual err fell; otherwise back to the last accepted point
//             and a Sinkhorn column step from it, which never increases err in exact arithmetic
//   stop      err = |g1|+|g2|+|g3|+|g4| <= tol_i (rows are exact by eq. (10)); after max_iter
//             updates; or when a Sinkhorn step does not lower err either (fp32 floor).  What is emitted is always
//             an accepted point, never a rejected trial.
// Hc: the logits with permuted columns.  Gather(Hc) re-reads them when the base point moves; Emit(T, iters, converged)
// receives the result (still in the permuted column order).
template <class Gather, class Emit>
BK4_DEV void newton_guarded(const float (&Hc)[16], const float (&xs)[4], float tol_i, int max_iter, Gather&& gather,
                            Emit&& emit) {
    float E[16], T[16], c[4], v[3], b0[4] = {xs[0], xs[1], xs[2], xs[3]};
    perm_exponentials(Hc, b0, E);
    v[0] = v[1] = v[2] = 1.0f;
    eval_T<true>(E, v[0], v[1], v[2], T, c);
    column_ratios(T, v);

    float vprev[3] = {v[0], v[1], v[2]};
    float errprev = kInf;
    unsigned newton_trial = 0u, sink_trial = 0u;
    for (int it = 0;;) {
        eval_T<true>(E, v[0], v[1], v[2], T, c);  // c holds the residuals c_j - 1
        const float err = (fabsf(c[0]) + fabsf(c[1])) + (fabsf(c[2]) + fabsf(c[3]));
        const unsigned conv = err <= tol_i ? 1u : 0u;  // false for NaN
        const unsigned nan = err != err ? 1u : 0u;
        const unsigned worse = (newton_trial | sink_trial) & (err < errprev ? 0u : 1u) & (conv ^ 1u);
        if (worse) {
            if (newton_trial && it < max_iter) {
                // back to the last accepted point, Sinkhorn column step from it
                float ratio[3];
                eval_T<true>(E, vprev[0], vprev[1], vprev[2], T, c);
                column_ratios(T, ratio);
#pragma unroll
                for (int j = 0; j < 3; ++j) v[j] = vprev[j] * ratio[j];
                newton_trial = 0u, sink_trial = 1u;
                ++it;
                continue;
            }
            // neither step lowers err (fp32 floor), or no updates left: the last accepted point is the result
            eval_T<true>(E, vprev[0], vprev[1], vprev[2], T, c);
            emit(T, it, false);
            break;
        }
        if (conv | nan | (it >= max_iter ? 1u : 0u)) {
            emit(T, it, conv != 0u);
            break;
        }
        // accepted.  Far from the base: move the base there (beta0 += delta, E recomputed from H, v = 1); T, c and
        // the Newton direction do not depend on where the base is.
        if (fmaxf(fmaxf(v[0], v[1]), v[2]) > kVHi || fminf(fminf(v[0], v[1]), v[2]) < kVLo) {
            float Hr[16];
            gather(Hr);
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                b0[j] += lg2_approx(v[j]);
                v[j] = 1.0f;
            }
            perm_exponentials(Hr, b0, E);
        }
#pragma unroll
        for (int j = 0; j < 3; ++j) vprev[j] = v[j];
        errprev = err;
        float d1, d2, d3;
        newton_direction<true>(T, c[0], c[1], c[2], d1, d2, d3);
        // beta += d  <=>  v *= exp(d).  The step is clipped to |d| <= 41 (about 60 ln 2): a (near-)singular Hessian far
        // from the solution gives an unbounded direction; the guard then decides.  With |log2 v| <= 40 at accepted
        // points the trial stays inside the fp32 range.
        v[0] *= exp_step<true>(fminf(fmaxf(d1, -41.0f), 41.0f));
        v[1] *= exp_step<true>(fminf(fmaxf(d2, -41.0f), 41.0f));
        v[2] *= exp_step<true>(fminf(fmaxf(d3, -41.0f), 41.0f));
        newton_trial = 1u, sink_trial = 0u;
        ++it;
    }
}

}  // namespace bk4
