// bk4_core.cuh -- per-matrix solvers of the batched 4x4 Birkhoff projection, written once for the value
// types of bk4_vec.cuh (float: one matrix per thread; float2: two matrices per thread, packed FP32).
//
// Citations are to /root/reference/PAPER.md (arXiv 2606.07574); "DESIGN.md Sx/Gx" are the readings of the
// passages where the paper is silent or garbled.
//
// Notation (paper): R = H (logits), U_ij = beta_j + R_ij, T = row-softmax(U) (eq. (10)), c = column sums,
// g = c_{1..3} - 1 (eq. (11)), Hessian = diag(c) - T_{-4}^T T_{-4}.
//
// How T(beta) is evaluated here: write beta = beta0 + delta and
// keep E_ij = exp(U0_ij - mu_i) for the base point beta0 (16 exponentials, once) and v_j = exp(delta_j).
// Then T_ij = E_ij v_j / sum_k E_ik v_k is eq. (10) exactly, a Newton update beta += d is v_j *= exp(d_j)
// (3 exponentials instead of 16), and the row-max shift mu_i keeps every exponential <= 1 as in PAPER.md:186-191.
// When |delta| grows past 2^40 the base is moved (beta0 += delta, E recomputed from H).
#pragma once
#include <type_traits>

#include "bk4_vec.cuh"

#ifndef BK4_TRACE  // development hook (host emulation of the solver); compiles to nothing in the library
#define BK4_TRACE(...)
#endif

namespace bk4 {

constexpr float kLog2e = 1.4426950408889634f;
#define kInf __int_as_float(0x7f800000)
#define kNaN __int_as_float(0x7fc00000)
constexpr float kVHi = 1.099511627776e12f;   // 2^40: range of v before the base point is moved
constexpr float kVLo = 9.094947017729282e-13f;  // 2^-40
// 2^-22 added to the three ground weights of the Laplacian (Hessian and Delta), S7: a group of columns
// whose link to column 4 is weaker than this carries a residual below it, and without it the rounding noise of
// g divided by a vanishing link would throw the whole group by 2^60.
constexpr float kLamGround = 2.384185791015625e-07f;

// -------------------------------------------------------------------------------------------------
// Solve the grounded graph Laplacian system  L d = -g  (3 unknowns), L = [[a+b+p, -a, -b], [-a, a+c+q, -c],
// [-b, -c, b+c+r]].  This is the Newton system H d = -g of eq. (12) PAPER.md:223-233 (and Delta w = rhs of
// eq. (13)) with H = diag(c) - T_{-4}^T T_{-4} written through its six edge weights
// W_jk = sum_i T_ij T_ik >= 0: a,b,c = W12,W13,W23 and ground weights p,q,r = W14,W24,W34 (rows of T sum to 1,
// so h_jj = sum_{k != j} W_jk; no subtraction c_j - sum_i T_ij^2 is formed).  Node elimination: every pivot
// is a sum of non-negative terms (S7); `lam` on the ground weights keeps them non-zero when T is a
// permutation matrix.  3 reciprocals on the SFU.
template <class V>
BK4_DEV void solve_grounded_laplacian(V a, V b, V c, V p, V q, V r, V g1, V g2, V g3, float lam, V& d1, V& d2,
                                      V& d3) {
    if (lam != 0.0f) {  // (folds away when the caller has put the regularisation into p, q, r itself)
        const V l = vsplat(V{}, lam);
        p = vadd(p, l);
        q = vadd(q, l);
        r = vadd(r, l);
    }
    // eliminate node 1
    const V i1 = vrcp(vadd(vadd(a, b), p));
    const V ai = vmul(a, i1), bi = vmul(b, i1);
    const V c2 = vfma(ai, b, c);
    const V q2 = vfma(ai, p, q);
    const V r2 = vfma(bi, p, r);
    const V g2p = vfma(ai, g1, g2);
    const V g3p = vfma(bi, g1, g3);
    // eliminate node 2
    const V i2 = vrcp(vadd(c2, q2));
    const V ci = vmul(c2, i2);
    const V r3 = vfma(ci, q2, r2);
    const V g3pp = vfma(ci, g2p, g3p);
    // back substitution
    d3 = vneg(vmul(g3pp, vrcp(r3)));
    d2 = vmul(vsub(vmul(c2, d3), g2p), i2);
    d1 = vmul(vsub(vfma(a, d2, vmul(b, d3)), g1), i1);
}

// six edge weights W_jk = sum_i T_ij T_ik of the column graph (the p_jk dot products)
template <class V>
BK4_DEV V col_dot(const V (&T)[16], int j, int k) {
    return vfma(T[12 + j], T[12 + k], vfma(T[8 + j], T[8 + k], vfma(T[4 + j], T[4 + k], vmul(T[j], T[k]))));
}

// E_ij = 2^(u_ij - mu_i), u_ij = H_ij log2(e) + b0_j, mu_i = max_j u_ij  (eq. (10) PAPER.md:186-191 at the base
// point beta0 = b0 / log2(e); b0_4 = 0 is the gauge PAPER.md:132).  First call (b0 = 0): `zero_base`.
template <class V>
BK4_DEV void base_exponentials(const V (&H)[16], const V (&b0)[3], bool zero_base, V (&E)[16]) {
    const V l2e = vsplat(V{}, kLog2e);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (zero_base) {
            const V m = vmax(vmax(H[4 * i], H[4 * i + 1]), vmax(H[4 * i + 2], H[4 * i + 3]));
            const V t = vmul(m, vsplat(V{}, -kLog2e));
#pragma unroll
            for (int j = 0; j < 4; ++j) E[4 * i + j] = vex2(vfma(H[4 * i + j], l2e, t));
        } else {
            V u[4];
#pragma unroll
            for (int j = 0; j < 3; ++j) u[j] = vfma(H[4 * i + j], l2e, b0[j]);
            u[3] = vmul(H[4 * i + 3], l2e);
            const V m = vmax(vmax(u[0], u[1]), vmax(u[2], u[3]));
#pragma unroll
            for (int j = 0; j < 4; ++j) E[4 * i + j] = vex2(vsub(u[j], m));
        }
    }
}

// T(beta) of eq. (10) from the base exponentials and v = exp(delta): rows normalised, plus the column residuals
// g_j = c_j - 1 for all four columns.  Two details keep the fp32 floor of Err below 1e-6 (S9):
// the SFU reciprocal (1 ulp) gets one Newton-Raphson refinement so that rows sum to 1 within rounding, and
// the residual is summed as sum_i (T_ij - 1/4), whose partial sums are small, instead of (sum_i T_ij) - 1.
template <class V>
BK4_DEV void eval_T(const V (&E)[16], const V (&v)[3], V (&T)[16], V (&g)[4]) {
    const V one = vsplat(V{}, 1.0f), mq = vsplat(V{}, -0.25f);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const V x0 = vmul(E[4 * i], v[0]), x1 = vmul(E[4 * i + 1], v[1]), x2 = vmul(E[4 * i + 2], v[2]);
        const V x3 = E[4 * i + 3];
        const V s = vadd(vadd(x0, x1), vadd(x2, x3));
        const V r0 = vrcp(s);
        const V r = vfma(r0, vfma(vneg(s), r0, one), r0);
        T[4 * i] = vmul(x0, r);
        T[4 * i + 1] = vmul(x1, r);
        T[4 * i + 2] = vmul(x2, r);
        T[4 * i + 3] = vmul(x3, r);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
        g[j] = vadd(vadd(vadd(T[j], mq), vadd(T[4 + j], mq)), vadd(vadd(T[8 + j], mq), vadd(T[12 + j], mq)));
}

template <class V>
BK4_DEV V clamp_ratio(V x) {
    // keeps a column step finite when a column sum underflows (NaN passes through vmin/vmax as the other operand,
    // which is fine: a NaN matrix is caught by the error test)
    return vmin(vmax(x, vsplat(V{}, kVLo)), vsplat(V{}, kVHi));
}

// Sinkhorn-Knopp column step (eq. (6) PAPER.md:108 with the gauge beta_4 = 0): ratio_j = c_4 / c_j, from the
// column sums themselves.  The residuals g_j = c_j - 1 of eval_T cannot be used here: a column that a bad
// Newton step has emptied (c_j ~ 1e-9) would come back from g_j + 1 as 0 or 6e-8 and the step would overshoot.
template <class V>
BK4_DEV void column_ratios(const V (&T)[16], V (&ratio)[3]) {
    V cs[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) cs[j] = vadd(vadd(T[j], T[4 + j]), vadd(T[8 + j], T[12 + j]));
#pragma unroll
    for (int j = 0; j < 3; ++j) ratio[j] = clamp_ratio(vmul(cs[3], vrcp(cs[j])));
}

// -------------------------------------------------------------------------------------------------
// Start point for large-magnitude logits (S1).  As |H| grows the projection tends to the
// max-weight assignment (the LP limit eta -> 0 of (3)), and from beta = 0 both Newton and Sinkhorn
// need O(range) steps.  This start takes the LP's dual potentials instead:
//   1. sigma = argmax over the 24 permutations of sum_i H_{i,sigma(i)}  (brute force, shared pair sums);
//   2. in the column order that puts sigma on the diagonal, x is dual-feasible iff x_j - x_k <= w_kj :=
//      H_kk - H_kj for all k != j (then every assigned entry is its row's maximum of U = H + x);
//      all-pairs shortest paths d of w (Floyd-Warshall, 4 nodes) give the feasible extremes x = d[s][.] and
//      x = -d[.][t]; their average over all s, t is feasible too and sits inside the dual polytope, so that
//      unassigned entries start e^{-slack} small instead of tied;
//   3. beta0_j = x_{sigma^{-1}(j)} - x_{sigma^{-1}(4)}   (gauge beta_4 = 0), returned in log2 units.
// Indices are carried as float values 0..3 so that the code is the same for both value types; everything is
// selects and static indexing (no local memory).
template <class V>
BK4_DEV void lp_dual_start(const V (&H)[16], V (&b0)[3]) {
    using M = typename vtraits<V>::mask;
    const V c0 = vsplat(V{}, 0.0f), c1 = vsplat(V{}, 1.0f), c2 = vsplat(V{}, 2.0f), c3 = vsplat(V{}, 3.0f);
    const V cidx[4] = {c0, c1, c2, c3};
    // 1. best permutation.  Rows 0,1 take the ordered pair (j0,j1); rows 2,3 take the other two columns in the
    //    better of their two orders.
    V best = vsplat(V{}, -kInf), s0 = c0, s1 = c1, s2 = c2, s3 = c3;
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = a + 1; b < 4; ++b) {
            // complement pair {a,b} for rows 2,3
            const V bab = vadd(H[8 + a], H[12 + b]), bba = vadd(H[8 + b], H[12 + a]);
            const M f = vgt(bba, bab);
            const V bb = vmax(bab, bba);
            const V t2 = vsel(f, cidx[b], cidx[a]), t3 = vsel(f, cidx[a], cidx[b]);
            int p = 0, q = 0;  // the two columns left for rows 0,1
            for (int j = 0, n = 0; j < 4; ++j)
                if (j != a && j != b) {
                    if (n++ == 0) p = j;
                    else q = j;
                }
#pragma unroll
            for (int o = 0; o < 2; ++o) {
                const int j0 = o ? q : p, j1 = o ? p : q;
                const V S = vadd(vadd(H[j0], H[4 + j1]), bb);
                const M m = vgt(S, best);
                best = vsel(m, S, best);
                s0 = vsel(m, cidx[j0], s0);
                s1 = vsel(m, cidx[j1], s1);
                s2 = vsel(m, t2, s2);
                s3 = vsel(m, t3, s3);
            }
        }
    // 2. columns reordered so that the assignment is the diagonal: Hc[i][m] = H[i][sigma(m)]
    const V sg[4] = {s0, s1, s2, s3};
    M eq[4][3];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int j = 0; j < 3; ++j) eq[m][j] = veq(sg[m], cidx[j]);
    V Hc[16];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int m = 0; m < 4; ++m)
            Hc[4 * i + m] = vsel(eq[m][0], H[4 * i], vsel(eq[m][1], H[4 * i + 1], vsel(eq[m][2], H[4 * i + 2], H[4 * i + 3])));
    V d[4][4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int j = 0; j < 4; ++j) d[k][j] = (k == j) ? c0 : vsub(Hc[5 * k], Hc[4 * k + j]);
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (k != m && j != m && k != j) d[k][j] = vmin(d[k][j], vadd(d[k][m], d[m][j]));
    V x[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        V acc = c0;
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (k != j) acc = vadd(acc, vsub(d[k][j], d[j][k]));
        x[j] = acc;  // 8 x the centre
    }
    // 3. back to the original column order, gauge, log2 units
    V beta[4];
#pragma unroll
    for (int j = 0; j < 3; ++j) beta[j] = vsel(eq[0][j], x[0], vsel(eq[1][j], x[1], vsel(eq[2][j], x[2], x[3])));
    {
        const M e0 = mor(mor(eq[0][0], eq[0][1]), eq[0][2]), e1 = mor(mor(eq[1][0], eq[1][1]), eq[1][2]),
                e2 = mor(mor(eq[2][0], eq[2][1]), eq[2][2]);
        beta[3] = vsel(e0, vsel(e1, vsel(e2, x[3], x[2]), x[1]), x[0]);
    }
    const V sc = vsplat(V{}, 0.125f * kLog2e);
#pragma unroll
    for (int j = 0; j < 3; ++j) b0[j] = vmul(vsub(beta[j], beta[3]), sc);
}

// -------------------------------------------------------------------------------------------------
// Guarded Newton on f(beta_1..3) (eq. (8); iteration PAPER.md:164-168).
//
//   start     beta0 = 0, or the LP dual start above for the matrices flagged `hard` (large logit range),
//             followed by one Sinkhorn-Knopp column step (eq. (6)) -- DESIGN.md S1
//   step      d = -Hessian^{-1} g  (eq. (9),(11),(12))
//   guard     accept the full step iff the column residual err decreased; otherwise go back and take a
//             Sinkhorn column step beta_j -= log(c_j / c_4), which never increases err -- DESIGN.md S2
//   stop      err = |g1|+|g2|+|g3|+|g1+g2+g3| <= tol_i (rows are exact by eq. (10)) -- S3;
//             after max_iter updates -- S4; or when neither step lowers err (fp32 floor) -- S5
//
// `any_hard` must be uniform over the threads that execute together (it only selects the cheaper start-up
// code when no matrix needs the LP start).  Reload(H) re-reads the logits (used when the base point moves);
// Emit(half, T, iters, converged) receives the result of one matrix as soon as it is final.
// `skip` marks matrices this call must leave alone (already finished by lean_iterate, or padding): they start out
// `done`, nothing is emitted for them and their arithmetic is ignored.
// LANE_INDEPENDENT: a matrix's arithmetic does not depend on which other matrices share its warp (the cheaper
// start-up code for warps without a `hard` matrix rounds differently), at the cost of a few instructions.
template <class V, bool LANE_INDEPENDENT = false, class Reload, class Emit>
BK4_DEV void newton_forward(const V (&H)[16], typename vtraits<V>::mask hard, bool any_hard,
                            typename vtraits<V>::mask skip, float tol_i, int max_iter, Reload&& reload,
                            Emit&& emit) {
    using M = typename vtraits<V>::mask;
    constexpr int NL = vtraits<V>::lanes;
    const V one = vsplat(V{}, 1.0f), zero = vsplat(V{}, 0.0f);

    V E[16], T[16], c[4], v[3], b0[3];
    b0[0] = b0[1] = b0[2] = zero;
    if (any_hard) {
        V bl[3];
        lp_dual_start(H, bl);
#pragma unroll
        for (int j = 0; j < 3; ++j) b0[j] = vsel(hard, bl[j], zero);
        base_exponentials(H, b0, false, E);
    } else {
        base_exponentials(H, b0, !LANE_INDEPENDENT, E);
    }

    // start-up column step (v = 1): v_j = c_4 / c_j
    v[0] = v[1] = v[2] = one;
    eval_T(E, v, T, c);
    column_ratios(T, v);

    V vprev[3] = {v[0], v[1], v[2]};
    V errprev = vsplat(V{}, kInf);
    M newton_trial = msplat(V{}, false), sink_trial = msplat(V{}, false), done = skip;
    int it[NL];
#pragma unroll
    for (int k = 0; k < NL; ++k) it[k] = 0;
    const V tolv = vsplat(V{}, tol_i);

    for (;;) {
        eval_T(E, v, T, c);  // c holds the residuals c_j - 1
        const V g1 = c[0], g2 = c[1], g3 = c[2];
        const V err = vadd(vadd(vabs(g1), vabs(g2)), vadd(vabs(g3), vabs(c[3])));
        const M conv = mnot(vgt(err, tolv));  // NaN counts as "stop"
        const M improved = vlt(err, errprev);
        const M rej = mand(mand(newton_trial, mnot(improved)), mnot(conv));
        const M stag = mand(mand(sink_trial, mnot(improved)), mnot(conv));
        M capped;
        if constexpr (NL == 1) capped = M(it[0] >= max_iter);
        else capped = M(it[0] >= max_iter, it[1] >= max_iter);
        const M fin = mor(mor(conv, capped), stag);
        BK4_TRACE("it %d err %.3e errprev %.3e v %.3e %.3e %.3e c %.4f %.4f %.4f %.4f rej %d stag %d\n", it[0],
                  vget(err, 0), vget(errprev, 0), vget(v[0], 0), vget(v[1], 0), vget(v[2], 0), 1 + vget(c[0], 0),
                  1 + vget(c[1], 0), 1 + vget(c[2], 0), 1 + vget(c[3], 0), (int)mget(rej, 0), (int)mget(stag, 0));
#pragma unroll
        for (int k = 0; k < NL; ++k)
            if (mget(fin, k) && !mget(done, k)) emit(k, T, it[k], mget(conv, k));
        done = mor(done, fin);
        if (mall(done)) break;

        const M act = mnot(done);
        const M rejected = mand(rej, act);
        const M accepted = mand(mnot(rej), act);

        // accepted point far from the base: move the base there (beta0 += delta, E recomputed from H, v = 1).
        // T, c and the Newton direction below do not depend on where the base is.
        {
            const V vmx = vmax(vmax(v[0], v[1]), v[2]), vmn = vmin(vmin(v[0], v[1]), v[2]);
            const M far = mand(accepted, mor(vgt(vmx, vsplat(V{}, kVHi)), vlt(vmn, vsplat(V{}, kVLo))));
            if (many(far)) {
                V Hr[16];
                reload(Hr);
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    b0[j] = vsel(far, vadd(b0[j], vlg2(v[j])), b0[j]);
                    v[j] = vsel(far, one, v[j]);
                }
                base_exponentials(Hr, b0, false, E);
            }
        }

        V vn[3] = {v[0], v[1], v[2]};
        if (many(accepted)) {
            // Newton direction at the accepted point (eq. (12) through the Laplacian form, S7)
            V d1, d2, d3;
            solve_grounded_laplacian(col_dot(T, 0, 1), col_dot(T, 0, 2), col_dot(T, 1, 2), col_dot(T, 0, 3),
                                     col_dot(T, 1, 3), col_dot(T, 2, 3), g1, g2, g3, kLamGround, d1, d2, d3);
            // beta += d  <=>  v *= exp(d).  The step is clipped to |d| <= 60 ln 2: a (near-)singular Hessian far
            // from the solution gives an unbounded direction; the guard then decides.  With |log2 v| <= 40 at
            // accepted points the trial stays inside the fp32 range.
            const V l2e = vsplat(V{}, kLog2e), hi = vsplat(V{}, 60.0f), lo = vsplat(V{}, -60.0f);
            vn[0] = vmul(v[0], vex2(vmin(vmax(vmul(d1, l2e), lo), hi)));
            vn[1] = vmul(v[1], vex2(vmin(vmax(vmul(d2, l2e), lo), hi)));
            vn[2] = vmul(v[2], vex2(vmin(vmax(vmul(d3, l2e), lo), hi)));
        }
        if (many(rejected)) {
            // back to the last accepted point (T is re-evaluated there: rare path, and T is dead until the next
            // eval_T), Sinkhorn column step from it
            V ratio[3], gdead[4];
            eval_T(E, vprev, T, gdead);
            column_ratios(T, ratio);
#pragma unroll
            for (int j = 0; j < 3; ++j) vn[j] = vsel(rejected, vmul(vprev[j], ratio[j]), vn[j]);
        }
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            vprev[j] = vsel(accepted, v[j], vprev[j]);
            v[j] = vsel(act, vn[j], v[j]);
        }
        errprev = vsel(accepted, err, errprev);
        newton_trial = accepted;
        sink_trial = rejected;
#pragma unroll
        for (int k = 0; k < NL; ++k) it[k] += mget(act, k) ? 1 : 0;
    }
}

// -------------------------------------------------------------------------------------------------
// Lean Newton (one matrix per thread, the whole warp in lockstep): the path nearly every matrix takes.
//
// Same iteration as newton_forward -- eq. (10) for T, eq. (11) for g, the Laplacian form of eq. (12) for the
// direction; start beta0 = 0, or the LP dual start for matrices whose largest in-row logit range exceeds
// `lp_range`, followed by Sinkhorn column steps (S1) -- with the guard of DESIGN.md S2 reduced to its
// test: a step after which the column residual did not fall ends the lean iteration for that matrix, which is
// then (status kLeanFailed) solved from scratch by newton_forward, whose guard can go back and take Sinkhorn
// steps.  Measured on B200: that happens to 0 of 2^20 N(0,1) matrices and to about 1 in 1000 at N(0,30^2).  So
// the common path carries no trial/rollback state, no re-basing and no per-lane stores: a finished lane freezes
// its v and keeps re-evaluating the same T until the warp is through, and the caller stores all results at once.
// A matrix's arithmetic does not depend on the other matrices of its warp.
//
//   active    lanes holding a matrix (the others only follow the warp's votes)
//   returns   kLeanConverged, kLeanStopped (max_iter reached, or the residual stalled at the fp32 floor:
//             result valid, counted as unconverged) or kLeanFailed (T is not a result)
constexpr unsigned kLeanConverged = 0u, kLeanStopped = 1u, kLeanFailed = 2u;
constexpr float kLeanFloor = 1e-5f;  // a residual that stalls below this is the fp32 floor, not a failure
constexpr float kLeanFloorTol = 2e-7f;  // internal tolerances below this are below the fp32 floor of the residual
constexpr int kLeanSweeps = 3;       // start-up Sinkhorn column steps
constexpr int kLeanFree = 2;         // Newton updates taken before the first residual test
constexpr float kBalanceFloor = 3e-6f;  // floor of the flows in the balancing step after the LP start

// State of one matrix inside the lean iteration.
struct LeanState {
    float E[16];        // exp(beta0_j + H_ij - mu_i), fixed after the start
    float v0, v1, v2;   // exp(beta_j - beta0_j)
    float errprev;      // residual of the last update's starting point (kInf before the first tested update)
    int it;             // updates taken
    unsigned running;   // 1 while the matrix is being iterated
    unsigned status;    // kLean* once it is not
};

// T(beta) of eq. (10) and g_j = c_j - 1 of eq. (11).  REFINE (an evaluation that may be the result): one
// Newton-Raphson refinement of the SFU reciprocal, so that the rows sum to 1 within rounding, and the residual of
// all four columns summed as two halves started from -1/2, which keeps every partial sum below 1/2 (S9).
template <bool REFINE>
BK4_DEV void lean_eval(const LeanState& s, float (&T)[16], float& g0, float& g1, float& g2, float& g3) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float x0 = s.E[4 * i] * s.v0, x1 = s.E[4 * i + 1] * s.v1, x2 = s.E[4 * i + 2] * s.v2, x3 = s.E[4 * i + 3];
        const float sum = (x0 + x1) + (x2 + x3);
        float r = rcp_approx(sum);
        if constexpr (REFINE) r = fmaf(r, fmaf(-sum, r, 1.0f), r);
        T[4 * i] = x0 * r;
        T[4 * i + 1] = x1 * r;
        T[4 * i + 2] = x2 * r;
        T[4 * i + 3] = x3 * r;
    }
    if constexpr (REFINE) {
        g0 = ((T[0] - 0.5f) + T[4]) + ((T[8] - 0.5f) + T[12]);
        g1 = ((T[1] - 0.5f) + T[5]) + ((T[9] - 0.5f) + T[13]);
        g2 = ((T[2] - 0.5f) + T[6]) + ((T[10] - 0.5f) + T[14]);
        g3 = ((T[3] - 0.5f) + T[7]) + ((T[11] - 0.5f) + T[15]);
    } else {
        g0 = (((T[0] - 1.0f) + T[4]) + T[8]) + T[12];
        g1 = (((T[1] - 1.0f) + T[5]) + T[9]) + T[13];
        g2 = (((T[2] - 1.0f) + T[6]) + T[10]) + T[14];
        g3 = 0.0f;
    }
}

// Newton update beta += d <=> v *= exp(d), d from eq. (12) through the Laplacian form (S7); the ground
// regularisation rides on the first product of each ground weight's FMA chain.
BK4_DEV void lean_update(LeanState& s, const float (&T)[16], float g0, float g1, float g2, bool apply) {
    auto ground = [&](int j) {
        return fmaf(T[12 + j], T[15], fmaf(T[8 + j], T[11], fmaf(T[4 + j], T[7], fmaf(T[j], T[3], kLamGround))));
    };
    float d1, d2, d3;
    solve_grounded_laplacian<float>(col_dot(T, 0, 1), col_dot(T, 0, 2), col_dot(T, 1, 2), ground(0), ground(1), ground(2),
                                    g0, g1, g2, 0.0f, d1, d2, d3);
    if (apply) {  // a finished lane keeps its v (and so its T)
        s.v0 *= ex2_approx(d1 * kLog2e);
        s.v1 *= ex2_approx(d2 * kLog2e);
        s.v2 *= ex2_approx(d3 * kLog2e);
    }
}

// Start: E at beta0 (0, or the LP dual start when the largest in-row range exceeds lp_range), then kLeanSweeps
// Sinkhorn column steps (beta0 = 0) or one balancing step (LP start), then min(kLeanFree, max_iter) untested Newton
// updates.  Returns false when the warp has nothing to do.
BK4_DEV bool lean_start(const float (&H)[16], bool active, float lp_range, int max_iter, LeanState& s) {
    // row maxima (the shift of eq. (10)) and the largest in-row range, which decides the start.
    // A NaN logit is skipped by fmaxf/fminf: such a matrix fails the first residual test and ends up in
    // newton_forward, which reports it; an infinite logit makes the range infinite and is sent there at once.
    float rmax[4], spread = 0.0f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        rmax[i] = fmaxf(fmaxf(H[4 * i], H[4 * i + 1]), fmaxf(H[4 * i + 2], H[4 * i + 3]));
        const float rmin = fminf(fminf(H[4 * i], H[4 * i + 1]), fminf(H[4 * i + 2], H[4 * i + 3]));
        spread = fmaxf(spread, rmax[i] - rmin);
    }
    const bool narrow = active && spread <= lp_range, wide = active && !narrow && spread <= 3.0e38f;
    active = narrow || wide;  // an infinite (or inf - inf = NaN) range is newton_forward's to report
    s.running = active ? 1u : 0u;
    s.status = kLeanFailed;
    s.errprev = kInf;
    s.it = 0;
    if (!__any_sync(0xffffffffu, active)) return false;
    if (__any_sync(0xffffffffu, narrow)) {
        // E_ij = exp(H_ij - max_j H_ij): eq. (10) at beta0 = 0
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float t = rmax[i] * -kLog2e;
#pragma unroll
            for (int j = 0; j < 4; ++j) s.E[4 * i + j] = ex2_approx(fmaf(H[4 * i + j], kLog2e, t));
        }
    }
    if (__any_sync(0xffffffffu, wide)) {
        // E at the LP dual start beta0 (log2 units), S1
        float b0[3], Eg[16];
        lp_dual_start<float>(H, b0);
        base_exponentials<float>(H, b0, false, Eg);
#pragma unroll
        for (int q = 0; q < 16; ++q) s.E[q] = wide ? Eg[q] : s.E[q];
    }
    // kLeanSweeps Sinkhorn column steps from beta0 (eq. (6) PAPER.md:108 with the gauge beta_4 = 0; rows are
    // normalised inside each step, eq. (5)): v_j *= c_4 / c_j.  Each costs a third of a Newton update and cuts the
    // residual about 4x on N(0,1) logits, which is what lets the second Newton update land below 1e-6 for 99 % of
    // the matrices instead of 50 % (S1).
    s.v0 = s.v1 = s.v2 = 1.0f;
    const bool any_narrow = __any_sync(0xffffffffu, narrow), any_wide = __any_sync(0xffffffffu, wide);
#pragma unroll
    for (int k = 0; k < kLeanSweeps; ++k) {
        if (!any_narrow) break;  // matrices with the LP start take the balancing step below instead
        float c0 = 0.0f, c1 = 0.0f, c2 = 0.0f, c3 = 0.0f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float x0 = k ? s.E[4 * i] * s.v0 : s.E[4 * i], x1 = k ? s.E[4 * i + 1] * s.v1 : s.E[4 * i + 1],
                        x2 = k ? s.E[4 * i + 2] * s.v2 : s.E[4 * i + 2], x3 = s.E[4 * i + 3];
            const float r = rcp_approx((x0 + x1) + (x2 + x3));
            c0 = fmaf(x0, r, c0);
            c1 = fmaf(x1, r, c1);
            c2 = fmaf(x2, r, c2);
            c3 = fmaf(x3, r, c3);
        }
        const float f0 = c3 * rcp_approx(c0), f1 = c3 * rcp_approx(c1), f2 = c3 * rcp_approx(c2);
        if (narrow) s.v0 *= f0, s.v1 *= f1, s.v2 *= f2;
    }
    // Matrices with the LP start: their T is a permutation matrix plus small entries, where column steps barely
    // move (Sinkhorn's slow regime) and Newton's updates are of unit size, so that the residual
    // falls by a factor e per update only.  What has to happen is that the small entries get balanced: column
    // j's inflow in_j = c_j - max_i T_ij against the outflow out_j = 1 - max_i T_ij of the row holding its
    // dominant entry.  One balancing step beta_j += (1/2) log(out_j / in_j) (Osborne's matrix-balancing update,
    // gauge beta_4 = 0) jumps there; flows are floored at kBalanceFloor, above the fp32 noise of 1 - max.  It is
    // a start-up step like the column steps: whatever it produces is judged by the tested iterations.  Measured
    // (S1): the mean over warps of the largest update count falls from 6.8 to 4.5 at N(0,100^2).
    if (any_wide) {
        float c[4] = {0.0f, 0.0f, 0.0f, 0.0f}, m[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float x0 = s.E[4 * i] * s.v0, x1 = s.E[4 * i + 1] * s.v1, x2 = s.E[4 * i + 2] * s.v2, x3 = s.E[4 * i + 3];
            const float r = rcp_approx((x0 + x1) + (x2 + x3));
            const float t[4] = {x0 * r, x1 * r, x2 * r, x3 * r};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                c[j] += t[j];
                m[j] = fmaxf(m[j], t[j]);
            }
        }
        float in[4], out[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            in[j] = fmaxf(c[j] - m[j], 0.0f) + kBalanceFloor;
            out[j] = fmaxf(1.0f - m[j], 0.0f) + kBalanceFloor;
        }
        // v_j *= sqrt((out_j / in_j) / (out_4 / in_4))
        const float num = in[3], den = out[3];
        const float q0 = (out[0] * num) * rcp_approx(in[0] * den), q1 = (out[1] * num) * rcp_approx(in[1] * den),
                    q2 = (out[2] * num) * rcp_approx(in[2] * den);
        if (wide) {
            s.v0 *= sqrt_approx(q0);
            s.v1 *= sqrt_approx(q1);
            s.v2 *= sqrt_approx(q2);
        }
    }
    // the first kLeanFree updates are taken without looking at the residual: on well-scaled inputs no matrix is
    // done before them, and whatever they produce is judged by the tested iterations of lean_iterate
    const int n_free = max_iter < kLeanFree ? max_iter : kLeanFree;
    for (int k = 0; k < n_free; ++k) {
        float T[16], g0, g1, g2, g3;
        lean_eval<false>(s, T, g0, g1, g2, g3);
        lean_update(s, T, g0, g1, g2, true);
    }
    s.it = n_free;
    return true;
}

// Tested iterations in warp lockstep: evaluate, stop test, Newton update, until no lane is running.
// T holds the last evaluation of every lane: the result of the lanes whose status is not kLeanFailed.
BK4_DEV void lean_iterate(LeanState& s, float tol_i, int max_iter, float (&T)[16]) {
    for (;;) {
        float g0, g1, g2, g3;
        lean_eval<true>(s, T, g0, g1, g2, g3);
        const float err = (fabsf(g0) + fabsf(g1)) + (fabsf(g2) + fabsf(g3));
        const bool conv = err <= tol_i;  // false for NaN: a NaN ends up in newton_forward
        const bool improved = err < s.errprev;
        if (s.running && (conv || !improved || s.it >= max_iter)) {
            s.running = 0u;
            // a residual that no longer falls: the fp32 floor if the caller asked for less than fp32 can give,
            // otherwise newton_forward's Sinkhorn steps may still get below tol
            s.status = conv ? kLeanConverged
                            : (improved || (s.errprev < kLeanFloor && tol_i < kLeanFloorTol)) ? kLeanStopped : kLeanFailed;
        }
        if (!__any_sync(0xffffffffu, s.running != 0u)) break;
        lean_update(s, T, g0, g1, g2, s.running != 0u);
        if (s.running) {
            s.errprev = err;
            ++s.it;
        }
    }
}

// -------------------------------------------------------------------------------------------------
// Backward, PAPER.md:284-304 (section 4.2) with Delta solved as a grounded Laplacian (S6/S7):
//   Gamma = G o P, mu_r = Gamma 1, mu_c = (Gamma^T 1)_{1..3}, rhs = mu_c - P_{-4}^T mu_r,
//   Delta w = rhs, w_4 = 0, v = mu_r - P w, dH_ij = P_ij (G_ij - v_i - w_j)   ( = -D_ij, PAPER.md:302-304 )
template <class V>
BK4_DEV void backward_ift(const V (&P)[16], const V (&G)[16], V (&dH)[16]) {
    V mur[4], muc[3], rhs[3];
#pragma unroll
    for (int i = 0; i < 4; ++i)
        mur[i] = vfma(G[4 * i + 3], P[4 * i + 3],
                      vfma(G[4 * i + 2], P[4 * i + 2], vfma(G[4 * i + 1], P[4 * i + 1], vmul(G[4 * i], P[4 * i]))));
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        muc[j] = vfma(G[12 + j], P[12 + j], vfma(G[8 + j], P[8 + j], vfma(G[4 + j], P[4 + j], vmul(G[j], P[j]))));
        const V pm = vfma(P[12 + j], mur[3], vfma(P[8 + j], mur[2], vfma(P[4 + j], mur[1], vmul(P[j], mur[0]))));
        rhs[j] = vsub(muc[j], pm);
    }
    V w1, w2, w3;  // solve_grounded_laplacian returns -L^{-1} g: pass g = -rhs
    solve_grounded_laplacian(col_dot(P, 0, 1), col_dot(P, 0, 2), col_dot(P, 1, 2), col_dot(P, 0, 3), col_dot(P, 1, 3),
                             col_dot(P, 2, 3), vneg(rhs[0]), vneg(rhs[1]), vneg(rhs[2]), kLamGround, w1, w2, w3);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const V vi = vsub(mur[i], vfma(P[4 * i + 2], w3, vfma(P[4 * i + 1], w2, vmul(P[4 * i], w1))));
        dH[4 * i] = vmul(P[4 * i], vsub(vsub(G[4 * i], vi), w1));
        dH[4 * i + 1] = vmul(P[4 * i + 1], vsub(vsub(G[4 * i + 1], vi), w2));
        dH[4 * i + 2] = vmul(P[4 * i + 2], vsub(vsub(G[4 * i + 2], vi), w3));
        dH[4 * i + 3] = vmul(P[4 * i + 3], vsub(G[4 * i + 3], vi));
    }
}

// -------------------------------------------------------------------------------------------------
// Sinkhorn-Knopp baseline, eq. (2): K = exp(H), n_iter x (row normalise, column normalise).
// The row-max shift is cancelled by the first row normalisation (it only avoids fp32 overflow).
template <class V>
BK4_DEV void sinkhorn_knopp(const V (&H)[16], int n_iter, V (&T)[16]) {
    V b0[3] = {vsplat(V{}, 0.0f), vsplat(V{}, 0.0f), vsplat(V{}, 0.0f)};
    base_exponentials(H, b0, true, T);
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const V r = vrcp(vadd(vadd(T[4 * i], T[4 * i + 1]), vadd(T[4 * i + 2], T[4 * i + 3])));
#pragma unroll
            for (int j = 0; j < 4; ++j) T[4 * i + j] = vmul(T[4 * i + j], r);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const V r = vrcp(vadd(vadd(T[j], T[4 + j]), vadd(T[8 + j], T[12 + j])));
#pragma unroll
            for (int i = 0; i < 4; ++i) T[4 * i + j] = vmul(T[4 * i + j], r);
        }
    }
}

}  // namespace bk4
