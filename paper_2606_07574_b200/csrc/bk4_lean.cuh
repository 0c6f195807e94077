// bk4_lean.cuh -- the lean Newton iteration: the path nearly every matrix takes.  One matrix per thread, the
// warp in lockstep, all state in registers; shared memory only as a per-thread scratch column for the
// data-dependent column permutation of the LP start (no thread reads another thread's slots: no barriers).
//
// Notation (paper): R = H (logits), U_ij = beta_j + R_ij, T = row-softmax(U) (eq. (10)),
// c = column sums, g = c_{1..3} - 1 (eq. (11)), Hessian = diag(c) - T_{-4}^T T_{-4}.
//
// How T(beta) is evaluated: write beta = beta0 + delta and keep
// E_ij = exp(U0_ij - mu_i) for the start point beta0 (16 exponentials, once) and v_j = exp(delta_j).  Then
// T_ij = E_ij v_j / sum_k E_ik v_k is eq. (10) exactly, a Newton update beta += d is v_j *= exp(d_j)
// (3 exponentials instead of 16), and the row shift mu_i keeps every exponential <= 1 as in PAPER.md:186-191.
//
// Two starts (S1), chosen per matrix by its largest in-row logit range (and wide, too, when exp(H) is
// a permutation matrix plus small entries):
//   narrow  beta0 = 0, E = exp(H - rowmax), three Sinkhorn-Knopp sweeps (eq. (2)) for v
//   wide    the dual potentials of the max-weight assignment (the LP limit eta -> 0 of (3)), with the
//           columns PERMUTED so that the assignment sits on the diagonal; the iteration then runs on the permuted
//           matrix (the projection commutes with column permutations) and the result is un-permuted when stored.
#pragma once
#include "bk4_solve.cuh"


namespace bk4 {

#ifndef BK4_THREADS
#define BK4_THREADS 128  // forward block size: 128 x 8 blocks per SM measured 1.5-2.5 % faster than 256 x 4
#endif
constexpr int kSmStride = BK4_THREADS;   // floats between consecutive entries of a thread's shared-memory column (= block size)
constexpr float kLeanFloor = 1e-5f;     // a residual that stalls below this is the fp32 floor, not a failure
constexpr int kLeanSweeps = 3;          // start-up Sinkhorn sweeps of the narrow start
constexpr int kLeanFree = 2;            // Newton updates taken before the first residual test
constexpr int kLeanFreeWide = 3;        // the same when every matrix of the warp took the wide start
static_assert(kLeanFree == 2, "lean_iterate spells the free updates out");
constexpr float kPeakedSum = 1.05f;     // every row sum of exp(H - rowmax) below this: wide start (see narrow_exponentials)
constexpr float kPolish = 1.5f;          // a residual within this factor of tol_i at the first test: polishing step (lean_iterate)
constexpr int kLeanNoisy = 4;            // tested updates during which a residual within 4 tol_i may rise
constexpr float kBalanceFloor = 3e-6f;  // floor of the flows in the balancing step after the LP start
constexpr unsigned kIdentityCode = 0x03020100u;  // column code: byte m = original column of permuted column m

constexpr unsigned kLeanConverged = 0u, kLeanStopped = 1u, kLeanFailed = 2u;

// -------------------------------------------------------------------------------------------------
// Narrow start, first half: E_ij = exp(H_ij - max_j H_ij) (eq. (10) at beta0 = 0) and its row sums.  max_i s_i is
// returned because it also decides the start: when every row's sum is within kPeakedSum of 1, exp(H) is a
// permutation matrix plus small entries and the matrix takes the wide start whatever its range is (S1).
BK4_DEV float narrow_exponentials(const float (&H)[16], const float (&rmax)[4], float (&E)[16], float (&s)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float t = rmax[i] * -kLog2e;
#pragma unroll
        for (int j = 0; j < 4; ++j) E[4 * i + j] = ex2_approx(fmaf(H[4 * i + j], kLog2e, t));
        s[i] = (E[4 * i] + E[4 * i + 1]) + (E[4 * i + 2] + E[4 * i + 3]);
    }
    return fmaxf(fmaxf(s[0], s[1]), fmaxf(s[2], s[3]));
}

// Narrow start, second half: kLeanSweeps Sinkhorn-Knopp sweeps in the scaling form of eq. (2) PAPER.md:76 with the
// gauge v_4 = 1: u = 1 / (E v), v_j = (E^T u)_4 / (E^T u)_j.  A sweep costs a third of a Newton update and cuts the
// residual about 4x on N(0,1) logits, which is what lets the second Newton update land below 1e-6 for 98 % of the
// matrices instead of 50 % (S1).
BK4_DEV void narrow_sweeps(const float (&E)[16], const float (&s0)[4], float& v0, float& v1, float& v2) {
    v0 = v1 = v2 = 1.0f;
#pragma unroll
    for (int k = 0; k < kLeanSweeps; ++k) {
        float u[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float s = k ? fmaf(E[4 * i], v0, fmaf(E[4 * i + 1], v1, fmaf(E[4 * i + 2], v2, E[4 * i + 3]))) : s0[i];
            u[i] = rcp_approx(s);
        }
        float q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) q[j] = fmaf(E[12 + j], u[3], fmaf(E[8 + j], u[2], fmaf(E[4 + j], u[1], E[j] * u[0])));
        v0 = q[3] * rcp_approx(q[0]);
        v1 = q[3] * rcp_approx(q[1]);
        v2 = q[3] * rcp_approx(q[2]);
    }
}

// -------------------------------------------------------------------------------------------------
// Wide start (S1).  As |H| grows the projection tends to the max-weight assignment (the LP limit
// eta -> 0 of (3)), and from beta = 0 both Newton and Sinkhorn need O(range) steps.  This start
// takes the LP's dual potentials instead:
//   1. sigma = argmax over the 24 permutations of sum_i H_{i,sigma(i)}: the six ways to split the columns between
//      rows {0,1} and rows {2,3}, each half in the better of its two orders;
//   2. the columns are permuted so that sigma is the diagonal (Hc_im = H_{i,sigma(m)}; the gather goes through the
//      thread's shared-memory column, which costs one issue slot per element where a select tree costs six);
//   3. x is dual-feasible iff x_j - x_k <= w_kj := Hc_kk - Hc_kj for all k != j (then every assigned entry is its
//      row's maximum of U = Hc + x); all-pairs shortest paths d of w (Floyd-Warshall, 4 nodes) give the feasible
//      extremes x = d[s][.] and x = -d[.][t]; their average over all s, t is feasible too and sits inside the dual
//      polytope, so that unassigned entries start e^{-slack} small instead of tied;
//   4. E_im = exp((x_m - x_i) - w_im) <= 1 with E_ii = 1, formed from differences (no rounding at |H|);
//   5. one balancing step for v: T is a permutation matrix plus small entries, where Sinkhorn sweeps barely move
//       and Newton's updates are of unit size (the residual falls by a factor e per update).  What
//      has to happen is that the small entries get balanced: column m's inflow in_m = c_m - T_mm against the
//      outflow out_m = 1 - T_mm of the row holding its assigned entry.  v_m = sqrt(out_m / in_m) (Osborne's
//      matrix-balancing update, gauge v_4 = 1) jumps there; flows are floored at kBalanceFloor.  Like every
//      start-up step it is judged by the tested iterations that follow.
// `sm` is this thread's scratch column (16 floats, stride kSmStride).  `code`: byte m = sigma(m).
BK4_DEV void gather_columns(const float* sm, unsigned code, float (&Hc)[16]);
BK4_DEV void lp_dual(const float (&H)[16], float* sm, float (&w)[4][4], float (&xs)[4], unsigned& code) {
    // 1. best split.  k: (a,b | c,d) = columns of rows {0,1} | rows {2,3}
    constexpr int SA[6] = {0, 0, 0, 1, 1, 2}, SB[6] = {1, 2, 3, 2, 3, 3}, SC[6] = {2, 1, 1, 0, 0, 0},
                  SD[6] = {3, 3, 2, 3, 2, 1};
    float tot[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float top = fmaxf(H[SA[k]] + H[4 + SB[k]], H[SB[k]] + H[4 + SA[k]]);
        const float bot = fmaxf(H[8 + SC[k]] + H[12 + SD[k]], H[8 + SD[k]] + H[12 + SC[k]]);
        tot[k] = top + bot;
    }
    const float best = fmaxf(fmaxf(fmaxf(tot[0], tot[1]), tot[2]), fmaxf(fmaxf(tot[3], tot[4]), tot[5]));
    code = (unsigned)SA[5] | (unsigned)SB[5] << 8 | (unsigned)SC[5] << 16 | (unsigned)SD[5] << 24;
#pragma unroll
    for (int k = 4; k >= 0; --k)
        code = tot[k] == best ? ((unsigned)SA[k] | (unsigned)SB[k] << 8 | (unsigned)SC[k] << 16 | (unsigned)SD[k] << 24)
                              : code;
    // 2. the logits into the scratch column; order of each half from its 2x2 block; gather
#pragma unroll
    for (int q = 0; q < 16; ++q) sm[q * kSmStride] = H[q];
    {
        const int a = code & 0xff, b = (code >> 8) & 0xff, c = (code >> 16) & 0xff, d = code >> 24;
        const float t0 = sm[a * kSmStride] + sm[(4 + b) * kSmStride], t1 = sm[b * kSmStride] + sm[(4 + a) * kSmStride];
        const float b0 = sm[(8 + c) * kSmStride] + sm[(12 + d) * kSmStride],
                    b1 = sm[(8 + d) * kSmStride] + sm[(12 + c) * kSmStride];
        code = __byte_perm(code, 0u, t1 > t0 ? 0x3201u : 0x3210u);
        code = __byte_perm(code, 0u, b1 > b0 ? 0x2310u : 0x3210u);
    }
    float Hc[16];
    gather_columns(sm, code, Hc);
    // 3. slack graph, all-pairs shortest paths, 8 x the centre of the dual polytope
    float d[4][4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int j = 0; j < 4; ++j) d[k][j] = w[k][j] = (k == j) ? 0.0f : Hc[5 * k] - Hc[4 * k + j];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (k != m && j != m && k != j) d[k][j] = fminf(d[k][j], d[k][m] + d[m][j]);
    const float e01 = d[0][1] - d[1][0], e02 = d[0][2] - d[2][0], e03 = d[0][3] - d[3][0], e12 = d[1][2] - d[2][1],
                e13 = d[1][3] - d[3][1], e23 = d[2][3] - d[3][2];
    const float sc = 0.125f * kLog2e;  // centre = x / 8; log2 units
    xs[0] = -((e01 + e02) + e03) * sc;
    xs[1] = ((e01 - e12) - e13) * sc;
    xs[2] = ((e02 + e12) - e23) * sc;
    xs[3] = ((e03 + e13) + e23) * sc;
}

// the logits of the thread's scratch column (written by lp_dual) with their columns permuted by `code`
BK4_DEV void gather_columns(const float* sm, unsigned code, float (&Hc)[16]) {
    const int c0 = code & 0xff, c1 = (code >> 8) & 0xff, c2 = (code >> 16) & 0xff, c3 = code >> 24;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        Hc[4 * i] = sm[(4 * i + c0) * kSmStride];
        Hc[4 * i + 1] = sm[(4 * i + c1) * kSmStride];
        Hc[4 * i + 2] = sm[(4 * i + c2) * kSmStride];
        Hc[4 * i + 3] = sm[(4 * i + c3) * kSmStride];
    }
}

BK4_DEV void wide_start(const float (&H)[16], float* sm, float (&E)[16], float& v0, float& v1, float& v2,
                        unsigned& code) {
    float w[4][4], xs[4];
    lp_dual(H, sm, w, xs, code);
    // 4. E in the permuted column order
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int m = 0; m < 4; ++m)
            E[4 * i + m] = (i == m) ? 1.0f : ex2_approx(fmaf(w[i][m], -kLog2e, xs[m] - xs[i]));
    // 5. balancing step
    float u[4], out[4], in[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        float off = 0.0f;
#pragma unroll
        for (int m = 0; m < 4; ++m)
            if (m != i) off += E[4 * i + m];
        u[i] = rcp_approx(1.0f + off);
        out[i] = fmaf(off, u[i], kBalanceFloor);
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        float s = kBalanceFloor;
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (i != m) s = fmaf(E[4 * i + m], u[i], s);
        in[m] = s;
    }
    // v_m = sqrt((out_m / in_m) / (out_4 / in_4))
    v0 = sqrt_approx((out[0] * in[3]) * rcp_approx(in[0] * out[3]));
    v1 = sqrt_approx((out[1] * in[3]) * rcp_approx(in[1] * out[3]));
    v2 = sqrt_approx((out[2] * in[3]) * rcp_approx(in[2] * out[3]));
}

// un-permute the columns of T through the thread's scratch column: out[i][sigma(m)] = T[i][m]
BK4_DEV void unpermute_columns(const float (&T)[16], unsigned code, float* sm, float (&out)[16]) {
    const int c0 = code & 0xff, c1 = (code >> 8) & 0xff, c2 = (code >> 16) & 0xff, c3 = code >> 24;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        sm[(4 * i + c0) * kSmStride] = T[4 * i];
        sm[(4 * i + c1) * kSmStride] = T[4 * i + 1];
        sm[(4 * i + c2) * kSmStride] = T[4 * i + 2];
        sm[(4 * i + c3) * kSmStride] = T[4 * i + 3];
    }
#pragma unroll
    for (int q = 0; q < 16; ++q) out[q] = sm[q * kSmStride];
}

// -------------------------------------------------------------------------------------------------
// Newton update beta += d <=> v *= exp(d), d from eq. (12) through the Laplacian form (S7); only where
// `go` (a lane whose matrix is finished keeps its v, and so its T)
template <bool ACCURATE>
BK4_DEV void lean_update(const float (&T)[16], const float (&g)[4], bool go, float& v0, float& v1, float& v2) {
    float d1, d2, d3;
    newton_direction<true>(T, g[0], g[1], g[2], d1, d2, d3);
    const float f0 = exp_step<ACCURATE>(d1), f1 = exp_step<ACCURATE>(d2), f2 = exp_step<ACCURATE>(d3);
    if (go) v0 *= f0, v1 *= f1, v2 *= f2;
}

// What the lean iteration reports for one matrix.
struct LeanResult {
    int it;          // updates taken
    bool stored;     // T is the result (converged, max_iter reached, or stalled at the fp32 floor)
    bool converged;  // the tested residual was <= tol_i
};

// Free updates and tested iterations in warp lockstep (PAPER.md:164-168 with the guard of DESIGN.md S2 reduced to its
// test: an update after which the column residual did not fall ends the lean iteration for that matrix).
//   - free updates, taken without looking at the residual (on well-scaled inputs no matrix is done before them, and
//     whatever they produce is judged by the tested iterations).  How many is a property of the MATRIX:
//       plain3 (wide start and max_iter >= kLeanFreeWide): kLeanFreeWide plain updates: after the wide start half of
//         the matrices need a third update and a quarter a fourth;
//       otherwise: min(kLeanFree, max_iter) updates, the last one refined (it is the last update of nearly every
//         well-scaled matrix: refined reciprocal and accurate exponential, or the 2^-23 of the SFU reciprocal is left
//         in the residual for the test to find).
//     A warp whose matrices all agree runs that schedule; a warp that holds both kinds runs the merged one, in which
//     every lane gets exactly the arithmetic of its own schedule (eval_T_sel, exp_step_sel), so a matrix's result does
//     not depend on its warp neighbours.
//   - then: evaluate, stop test, Newton update, until no lane is running.  A lane whose matrix is finished keeps its
//     v, so the last evaluation is every lane's result and T is handed back once.
// A lane that is not `active` only follows the warp.  `stored` is false for a matrix whose residual stopped falling
// above the fp32 floor (and for NaN): the guarded solver takes it.
// KIND: what the caller knows about the warp (no votes are spent on it, and a warp of wide matrices carries none of
// the narrow matrices' polishing step): kLeanNarrow = no wide matrix, kLeanWide = no narrow matrix (plain3 is then the
// same for every lane), kLeanMixed = both.
constexpr int kLeanNarrow = 0, kLeanMixed = 1, kLeanWide = 2;
template <int KIND>
BK4_DEV LeanResult lean_iterate(const float (&E)[16], float v0, float v1, float v2, bool active, bool plain3, bool polishable,
                                float tol_i, int max_iter, float (&T)[16]) {
    float g[4];
    int it = 0;  // this lane's update count
    const bool wide3 = KIND == kLeanWide && max_iter >= kLeanFreeWide;  // a warp of wide matrices: nothing to vote on
    const bool any3 = KIND == kLeanWide ? wide3 : KIND == kLeanMixed && __any_sync(0xffffffffu, plain3);
    const bool all3 = KIND == kLeanWide ? wide3 : KIND == kLeanMixed && any3 && __all_sync(0xffffffffu, plain3 || !active);
    if (any3 && all3) {
#pragma unroll 1
        for (; it < kLeanFreeWide; ++it) {
            eval_T<false>(E, v0, v1, v2, T, g);
            lean_update<false>(T, g, true, v0, v1, v2);
        }
    } else if (!any3 && max_iter >= kLeanFree) {
        eval_T<false>(E, v0, v1, v2, T, g);
        lean_update<false>(T, g, true, v0, v1, v2);
        eval_T<true, false>(E, v0, v1, v2, T, g);
        lean_update<true>(T, g, true, v0, v1, v2);
        it = kLeanFree;
    } else if (any3) {
        // merged schedule (max_iter >= kLeanFreeWide here): update 1 plain for everyone; update 2 plain for plain3 lanes,
        // refined for the others; update 3 for plain3 lanes only
        static_assert(kLeanFreeWide == kLeanFree + 1, "the merged schedule spells the updates out");
        eval_T<false>(E, v0, v1, v2, T, g);
        lean_update<false>(T, g, true, v0, v1, v2);
        eval_T_sel(E, v0, v1, v2, !plain3, T, g);
        {
            float d1, d2, d3;
            newton_direction<true>(T, g[0], g[1], g[2], d1, d2, d3);
            v0 *= exp_step_sel(d1, !plain3), v1 *= exp_step_sel(d2, !plain3), v2 *= exp_step_sel(d3, !plain3);
        }
        eval_T<false>(E, v0, v1, v2, T, g);
        lean_update<false>(T, g, plain3, v0, v1, v2);
        it = plain3 ? kLeanFreeWide : kLeanFree;
    } else {
        for (; it < max_iter; ++it) {
            eval_T<false>(E, v0, v1, v2, T, g);
            lean_update<false>(T, g, true, v0, v1, v2);
        }
    }
    LeanResult res = {it, false, false};
    float errprev = active ? kInf : -1.0f;  // negative: this lane is not, or no longer, running
    for (;; ++it) {
        eval_T<true>(E, v0, v1, v2, T, g);
        const float err = (fabsf(g[0]) + fabsf(g[1])) + (fabsf(g[2]) + fabsf(g[3]));
        const bool conv = err <= tol_i;  // false for NaN: a NaN matrix ends up in the guarded solver, which reports it
        // One more update as long as the residual falls.  Within 4 tol_i it may also rise: there the updates only
        // move the fp32 rounding noise of g around (each turns the noise of its evaluation into residual), and the
        // next evaluation is below tol_i more often than not (kLeanNoisy updates at most: a matrix whose noise sits
        // above tol_i would otherwise keep its whole warp until max_iter).
        const bool go = !conv && it < max_iter && (err < errprev || (err <= 4.0f * tol_i && it < kLeanFree + kLeanNoisy));
        if (errprev >= 0.0f && !go) {  // this lane's matrix is finished
            res.it = it;
            res.converged = conv;
            // (T is the evaluation at hand.  Out of updates: that is the last iterate.  Stalled: the evaluation is the one
            // at the trial that did not lower the residual, so it is the result only if it, too, is at the fp32 floor;
            // a trial that threw the residual back up goes to the guarded solver, which returns an accepted point.)
            res.stored = conv || (it >= max_iter && err < kInf) || (errprev < kLeanFloor && err < kLeanFloor);  // never a NaN
        }
        if (!__any_sync(0xffffffffu, go)) break;
        // The polishing step.  After the two untested updates a well-scaled matrix that fails its first test is as good
        // as converged: what is left is the fp32 error of the evaluation the second update started from (measured on
        // N(0,1): 82 % of them are within 2 tol_i).  Such a matrix (narrow start, in-row range at
        // most kPolishSpread, residual within kPolish tol_i) takes a Sinkhorn column step from the residuals at hand,
        // v_m *= c_4 / c_m = 1 + (g_4 - g_m) + O(g^2) (eq. (6) PAPER.md:108 with the gauge v_4 = 1), instead of a Newton
        // update; a warp in which no other matrix needs one skips the Hessian solve.  The choice is the matrix's own,
        // it is made once (a matrix that is still not there afterwards takes Newton updates), and it counts as an update.
        bool cheap = false, polish = false;
        if (KIND != kLeanWide) {
            cheap = go && polishable && it == kLeanFree && err <= kPolish * tol_i;
            polish = __any_sync(0xffffffffu, cheap);
        }
        if (!polish) {
            lean_update<true>(T, g, go, v0, v1, v2);
        } else {
            float f0 = 1.0f, f1 = 1.0f, f2 = 1.0f;
            if (__any_sync(0xffffffffu, go && !cheap)) {
                float d1, d2, d3;
                newton_direction<true>(T, g[0], g[1], g[2], d1, d2, d3);
                f0 = exp_step<true>(d1), f1 = exp_step<true>(d2), f2 = exp_step<true>(d3);
            }
            if (cheap) f0 = 1.0f + (g[3] - g[0]), f1 = 1.0f + (g[3] - g[1]), f2 = 1.0f + (g[3] - g[2]);
            if (go) v0 *= f0, v1 *= f1, v2 *= f2;
        }
        errprev = go ? err : -1.0f;
    }
    return res;
}

}  // namespace bk4
