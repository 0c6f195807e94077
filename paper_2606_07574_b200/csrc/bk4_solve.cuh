// bk4_solve.cuh -- the 3x3 Newton / IFT system as a grounded graph Laplacian, the backward pass and the
// Sinkhorn-Knopp baseline, one matrix per thread, plain fp32 (the compiler may contract a*b+c into FFMA).
//
// Citations are to /root/reference/PAPER.md (arXiv 2606.07574); "DESIGN.md Sx" are the readings of the passages
// where the paper is silent or garbled.
#pragma once
#include "bk4_math.cuh"

namespace bk4 {

// Regularisation of the three ground weights of the Laplacian (S7).  A group of columns whose link to
// column 4 is weaker than lambda carries a residual below it, and without it the rounding noise of the right-hand
// side divided by a vanishing link would throw the whole group by 2^60.
//   forward   relative: 2^-22 of the sum of the six edge weights.  The residual g is formed without cancellation
//             (eval_T), so its noise is relative too, and a near-permutation T (all weights tiny) is solved as
//             accurately as a well-mixed one.
//   backward  absolute 2^-22: the right-hand side mu_c - P^T mu_r is computed from a P that was rounded to fp32
//             when it was stored, so its noise is 2^-24 |G| whatever the weights are.
constexpr float kLamRel = 2.384185791015625e-07f;
constexpr float kLamAbs = 2.384185791015625e-07f;
constexpr float kLamTiny = 1e-30f;  // keeps the pivots non-zero when T is exactly a permutation matrix

// Solve the grounded graph Laplacian system  L d = -g  (3 unknowns), L = [[a+b+p, -a, -b], [-a, a+c+q, -c],
// [-b, -c, b+c+r]].  This is the Newton system H d = -g of eq. (12) PAPER.md:223-233 (and Delta w = rhs of
// eq. (13)) with H = diag(c) - T_{-4}^T T_{-4} written through its six edge weights
// W_jk = sum_i T_ij T_ik >= 0: a,b,c = W12,W13,W23 and ground weights p,q,r = W14,W24,W34 (rows of T sum to 1,
// so h_jj = sum_{k != j} W_jk; no subtraction c_j - sum_i T_ij^2 is formed).  Node elimination: every pivot
// is a sum of non-negative terms (S7); the caller has regularised p, q, r.  3 reciprocals on the SFU.
BK4_DEV void solve_grounded_laplacian(float a, float b, float c, float p, float q, float r, float g1, float g2,
                                      float g3, float& d1, float& d2, float& d3) {
    // eliminate node 1
    const float i1 = rcp_approx((a + b) + p);
    const float ai = a * i1, bi = b * i1;
    const float c2 = fmaf(ai, b, c);
    const float q2 = fmaf(ai, p, q);
    const float r2 = fmaf(bi, p, r);
    const float g2p = fmaf(ai, g1, g2);
    const float g3p = fmaf(bi, g1, g3);
    // eliminate node 2
    const float i2 = rcp_approx(c2 + q2);
    const float ci = c2 * i2;
    const float r3 = fmaf(ci, q2, r2);
    const float g3pp = fmaf(ci, g2p, g3p);
    // back substitution
    d3 = -g3pp * rcp_approx(r3);
    d2 = fmaf(c2, d3, -g2p) * i2;
    d1 = (fmaf(a, d2, b * d3) - g1) * i1;
}

// edge weight W_jk = sum_i T_ij T_ik of the column graph (the p_jk dot products)
BK4_DEV float col_dot(const float (&T)[16], int j, int k) {
    return fmaf(T[12 + j], T[12 + k], fmaf(T[8 + j], T[8 + k], fmaf(T[4 + j], T[4 + k], T[j] * T[k])));
}

// Newton direction d = -Hessian^{-1} g at T (eq. (12) through the Laplacian form, S7), ground column 4
template <bool RELATIVE_LAMBDA>
BK4_DEV void newton_direction(const float (&T)[16], float g1, float g2, float g3, float& d1, float& d2, float& d3) {
    const float a = col_dot(T, 0, 1), b = col_dot(T, 0, 2), c = col_dot(T, 1, 2);
    float p = col_dot(T, 0, 3), q = col_dot(T, 1, 3), r = col_dot(T, 2, 3);
    const float lam = RELATIVE_LAMBDA ? fmaf(((a + b) + (c + p)) + (q + r), kLamRel, kLamTiny) : kLamAbs;
    p += lam, q += lam, r += lam;
    solve_grounded_laplacian(a, b, c, p, q, r, g1, g2, g3, d1, d2, d3);
}

// -------------------------------------------------------------------------------------------------
// T(beta) of eq. (10) from E and v = exp(beta - beta0), and the column residuals g_m = c_m - 1 of eq. (11) for
// m = 1..3 (ALL4: all four).  Neither a row nor a column is ever summed to 1 and compared with it (S9):
//   out_m = sum_{j != m} T_mj   (what row m gives to the other columns),   T_mm = 1 - out_m   (row m sums to 1),
//   in_m  = sum_{i != m} T_im   (what column m gets from the other rows),  g_m = in_m - out_m.
// When T is close to a permutation matrix on the diagonal (the wide start permutes the columns so that it is),
// in_m and out_m are sums of small numbers and g_m has their relative accuracy, where c_m - 1 would have
// cancelled against the 1; for a well-mixed T the two forms round alike.  REFINE (an evaluation that may be the
// result): one Newton-Raphson refinement of the SFU reciprocal.
template <bool REFINE, bool ALL4 = REFINE>
BK4_DEV void eval_T(const float (&E)[16], float v0, float v1, float v2, float (&T)[16], float (&g)[4]) {
    float out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float x[4] = {E[4 * i] * v0, E[4 * i + 1] * v1, E[4 * i + 2] * v2, E[4 * i + 3]};
        const int a = (i + 1) & 3, b = (i + 2) & 3, c = (i + 3) & 3;  // the three columns off the diagonal
        const float off = (x[a] + x[b]) + x[c];
        const float sum = x[i] + off;
        float r = rcp_approx(sum);
        if constexpr (REFINE) r = fmaf(r, fmaf(-sum, r, 1.0f), r);
        T[4 * i + a] = x[a] * r;
        T[4 * i + b] = x[b] * r;
        T[4 * i + c] = x[c] * r;
        out[i] = off * r;
        T[5 * i] = 1.0f - out[i];  // (may come out as -2^-25 of rounding when the entry is below 2^-24: clamp_diagonal)
    }
#pragma unroll
    for (int m = 0; m < (ALL4 ? 4 : 3); ++m) {
        const int a = (m + 1) & 3, b = (m + 2) & 3, c = (m + 3) & 3;
        g[m] = ((T[4 * a + m] + T[4 * b + m]) + T[4 * c + m]) - out[m];
    }
    if constexpr (!ALL4) g[3] = 0.0f;
}

// An evaluation that becomes the result: its diagonal entries 1 - out_m are not allowed below zero.
BK4_DEV void clamp_diagonal(float (&T)[16]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) T[5 * i] = fmaxf(T[5 * i], 0.0f);
}

// eval_T<true, false> for the lanes with `refine`, eval_T<false> for the others, bit for bit, in one instruction stream
// (a warp that holds both kinds of matrices: DESIGN.md S1): the refinement r += r (1 - sum r) is multiplied by 0 or 1.
BK4_DEV void eval_T_sel(const float (&E)[16], float v0, float v1, float v2, bool refine, float (&T)[16], float (&g)[4]) {
    const float m = refine ? 1.0f : 0.0f;
    float out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float x[4] = {E[4 * i] * v0, E[4 * i + 1] * v1, E[4 * i + 2] * v2, E[4 * i + 3]};
        const int a = (i + 1) & 3, b = (i + 2) & 3, c = (i + 3) & 3;
        const float off = (x[a] + x[b]) + x[c];
        const float sum = x[i] + off;
        float r = rcp_approx(sum);
        r = fmaf(r * m, fmaf(-sum, r, 1.0f), r);  // refine: fmaf(r, e, r); else: fmaf(0, e, r) = r
        T[4 * i + a] = x[a] * r;
        T[4 * i + b] = x[b] * r;
        T[4 * i + c] = x[c] * r;
        out[i] = off * r;
        T[5 * i] = 1.0f - out[i];
    }
#pragma unroll
    for (int mcol = 0; mcol < 3; ++mcol) {
        const int a = (mcol + 1) & 3, b = (mcol + 2) & 3, c = (mcol + 3) & 3;
        g[mcol] = ((T[4 * a + mcol] + T[4 * b + mcol]) + T[4 * c + mcol]) - out[mcol];
    }
    g[3] = 0.0f;
}

// beta += d  <=>  v *= exp(d).  ACCURATE (updates that may be the last): for |d| < 2^-8 the factor is
// 1 + d + d^2/2 (error below 2^-26) instead of the SFU's exp (relative error 2^-22, which at the end of the
// iteration is the largest error in v).
template <bool ACCURATE>
BK4_DEV float exp_step(float d) {
    const float e = ex2_approx(d * kLog2e);
    if constexpr (!ACCURATE) return e;
    const float p = fmaf(d, fmaf(d, 0.5f, 1.0f), 1.0f);
    return fabsf(d) < 0.00390625f ? p : e;
}
// exp_step<true> for the lanes with `accurate`, exp_step<false> for the others
BK4_DEV float exp_step_sel(float d, bool accurate) {
    const float e = ex2_approx(d * kLog2e);
    const float p = fmaf(d, fmaf(d, 0.5f, 1.0f), 1.0f);
    return (accurate && fabsf(d) < 0.00390625f) ? p : e;
}

// -------------------------------------------------------------------------------------------------
// Backward, PAPER.md:284-304 (section 4.2) with Delta solved as a grounded Laplacian (S6/S7):
//   Gamma = G o P, mu_r = Gamma 1, mu_c = (Gamma^T 1)_{1..3}, rhs = mu_c - P_{-4}^T mu_r,
//   Delta w = rhs, w_4 = 0, v = mu_r - P w, dH_ij = P_ij (G_ij - v_i - w_j)   ( = -D_ij, PAPER.md:302-304 )
BK4_DEV void backward_ift(const float (&P)[16], const float (&G)[16], float (&dH)[16]) {
    float mur[4], rhs[3];
#pragma unroll
    for (int i = 0; i < 4; ++i)
        mur[i] = fmaf(G[4 * i + 3], P[4 * i + 3],
                      fmaf(G[4 * i + 2], P[4 * i + 2], fmaf(G[4 * i + 1], P[4 * i + 1], G[4 * i] * P[4 * i])));
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const float muc = fmaf(G[12 + j], P[12 + j], fmaf(G[8 + j], P[8 + j], fmaf(G[4 + j], P[4 + j], G[j] * P[j])));
        const float pm = fmaf(P[12 + j], mur[3], fmaf(P[8 + j], mur[2], fmaf(P[4 + j], mur[1], P[j] * mur[0])));
        rhs[j] = muc - pm;
    }
    float w1, w2, w3;  // solve_grounded_laplacian returns -L^{-1} g: pass g = -rhs
    newton_direction<false>(P, -rhs[0], -rhs[1], -rhs[2], w1, w2, w3);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float vi = mur[i] - fmaf(P[4 * i + 2], w3, fmaf(P[4 * i + 1], w2, P[4 * i] * w1));
        dH[4 * i] = P[4 * i] * ((G[4 * i] - vi) - w1);
        dH[4 * i + 1] = P[4 * i + 1] * ((G[4 * i + 1] - vi) - w2);
        dH[4 * i + 2] = P[4 * i + 2] * ((G[4 * i + 2] - vi) - w3);
        dH[4 * i + 3] = P[4 * i + 3] * (G[4 * i + 3] - vi);
    }
}

// -------------------------------------------------------------------------------------------------
// Sinkhorn-Knopp baseline, eq. (2): K = exp(H), n_iter x (row normalise, column normalise).
// The row-max shift is cancelled by the first row normalisation (it only avoids fp32 overflow).
BK4_DEV void sinkhorn_knopp(const float (&H)[16], int n_iter, float (&T)[16]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float m = fmaxf(fmaxf(H[4 * i], H[4 * i + 1]), fmaxf(H[4 * i + 2], H[4 * i + 3]));
        const float t = m * -kLog2e;
#pragma unroll
        for (int j = 0; j < 4; ++j) T[4 * i + j] = ex2_approx(fmaf(H[4 * i + j], kLog2e, t));
    }
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float r = rcp_approx((T[4 * i] + T[4 * i + 1]) + (T[4 * i + 2] + T[4 * i + 3]));
#pragma unroll
            for (int j = 0; j < 4; ++j) T[4 * i + j] *= r;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float r = rcp_approx((T[j] + T[4 + j]) + (T[8 + j] + T[12 + j]));
#pragma unroll
            for (int i = 0; i < 4; ++i) T[4 * i + j] *= r;
        }
    }
}

}  // namespace bk4
