// bk_ot.cuh -- small entropic-regularised optimal transport, N x M with N, M <= 8, one problem per thread: the
// general problem of PAPER.md section 2.3 / 3.1 of which the 4x4 Birkhoff projection is the special case, and in
// particular the n = 8 Birkhoff projection.  SURVEY.md 8(f) NEXT-1 and NEXT-3.
//
//   forward   T = argmin_{T in Pi(a,b)} <T, C> - eta h(T)   (eq. (3)) by Newton's method on the
//             (M-1)-variable dual f(beta_{-M}) (eq. (8)) with gradient and Hessian of eq. (9)
//             PAPER.md:144-147, T_i. = a_i Softmax(U_i. / eta), a guarded step
//             and a stop on the marginal error (PAPER.md:323 with the marginals a, b).
//   backward  D = dl/dC from T and G = dl/dT by eq. (13) PAPER.md:273-280.
//
// What is the same as in the 4x4 kernels (bk4_*.cuh): incremental exponentials (E = exp(U0/eta - mu) once per
// base point, v_j = exp(delta_j/eta), a Newton update is v_j *= exp(d_j)); the Hessian written as the Laplacian of
// the column graph with edge weights W_jk = sum_i T_ij T_ik / a_i, grounded at column M and solved by node
// elimination (every pivot a sum of non-negative terms; S7); the residual-decrease guard with a
// Sinkhorn column step as fallback (S2).
// What is different: rows are streamed (T is never held whole: with N M = 64 entries the registers hold E, the
// column sums and the M(M-1)/2 edge weights); there is no LP start (an assignment problem for N = M = 8 has no
// 24-permutation brute force): wide costs are reached by continuation in eta (eps-scaling): the problem is solved
// at eta 2^K, ..., 2 eta, eta with 2^K eta ~ range / 16, each stage started from the potentials of the one before.
#pragma once
#include <type_traits>

#include "bk4_math.cuh"

namespace bkot {

using namespace bk4;

constexpr float kOtLam = 2.384185791015625e-07f;  // ground regularisation, relative to the mean row marginal
constexpr int kOtSweeps = 3;                     // Sinkhorn sweeps at the start of every continuation stage
constexpr float kOtStageRange = 16.0f;           // a stage's scaled costs span at most this (8 / 12 / 16 / 20 / 24 measured: DESIGN.md)
constexpr int kOtHalvings = 4;                   // step halvings before the Sinkhorn fallback
constexpr float kOtTiny = 1e-30f;                // floor of a row sum s_i and of a column sum q_j before their reciprocals
constexpr float kOtStageTol = 1e-2f;             // relative marginal error at which an intermediate stage is left

// vector load/store of one row of K floats (K = 4: 128 bits, K = 8: 256 bits, else scalar)
template <int K>
BK4_DEV void load_row(const float* p, float (&r)[K]) {
    if constexpr (K == 8) {
        ld256(p, r);
    } else if constexpr (K == 4) {
        const float4 t = *reinterpret_cast<const float4*>(p);
        r[0] = t.x, r[1] = t.y, r[2] = t.z, r[3] = t.w;
    } else {
#pragma unroll
        for (int j = 0; j < K; ++j) r[j] = p[j];
    }
}
template <int K>
BK4_DEV void store_row(float* p, const float (&r)[K]) {
    if constexpr (K == 8) {
        stg256(p, r);
    } else if constexpr (K == 4) {
        *reinterpret_cast<float4*>(p) = make_float4(r[0], r[1], r[2], r[3]);
    } else {
#pragma unroll
        for (int j = 0; j < K; ++j) p[j] = r[j];
    }
}

// all N rows of one problem: the loads are issued back to back (a load followed by arithmetic on it, row after row,
// would leave one row in flight per thread and bind the kernel by latency)
template <int N, int M>
BK4_DEV void load_all(const float* p, float (&X)[N * M]) {
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float r[M];
        load_row<M>(p + i * M, r);
#pragma unroll
        for (int j = 0; j < M; ++j) X[i * M + j] = r[j];
    }
}

// ---- sizes other than {4, 8} x {4, 8} (PAD instances): an n x m problem, 2 <= n <= N, 2 <= m <= M, sits in the N x M
// register tile.  Rows i >= n are padding with mass a_i = 0; the last real column, m-1, sits in slot M-1 (the ground
// of the gauge and of the Laplacian must be a real column) and the slots m-1 .. M-2 are padding with b_j = 0 and
// E_ij = 0: a zero marginal is outside the domain of eq. (5), so such rows and columns are not run
// through the formulas but carry no mass by construction (T_ij = 0 exactly) and are never stored.
struct OtShape {
    int n, m;
};
template <int M>
BK4_DEV bool pad_slot(OtShape sh, int j) { return j >= sh.m - 1 && j < M - 1; }
template <int M>
BK4_DEV int slot_column(OtShape sh, int j) { return j == M - 1 ? sh.m - 1 : j; }

// the costs of an n x m problem ([n][m] row-major, scalar loads: rows of odd length are not aligned) into the tile;
// a padding entry repeats the first entry of its row (of row 0 for a padding row): finite whenever the problem is,
// inside the problem's range, and never the row's only maximum
template <int N, int M>
BK4_DEV void load_padded(const float* p, OtShape sh, float (&X)[N * M]) {
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const float* row = p + (i < sh.n ? i : 0) * sh.m;
#pragma unroll
        for (int j = 0; j < M; ++j) X[i * M + j] = row[pad_slot<M>(sh, j) ? 0 : slot_column<M>(sh, j)];
    }
}
// T or G of the backward: padding entries are zero
template <int N, int M>
BK4_DEV void load_padded_zero(const float* p, OtShape sh, float (&X)[N * M]) {
#pragma unroll
    for (int i = 0; i < N; ++i)
#pragma unroll
        for (int j = 0; j < M; ++j)
            X[i * M + j] = (i < sh.n && !pad_slot<M>(sh, j)) ? p[i * sh.m + slot_column<M>(sh, j)] : 0.0f;
}
template <int M>
BK4_DEV void store_padded_row(float* p, OtShape sh, int i, const float (&x)[M]) {
    if (i >= sh.n) return;
#pragma unroll
    for (int j = 0; j < M; ++j)
        if (!pad_slot<M>(sh, j)) p[i * sh.m + slot_column<M>(sh, j)] = x[j];
}

// index of the edge weight W_jk, j < k < M, in the packed upper triangle
template <int M>
BK4_DEV constexpr int tri(int j, int k) {
    return j * M - j * (j + 1) / 2 + (k - j - 1);
}

// compile-time loop: f(integral_constant<int, I>) for I = Begin .. End-1.  (With a plain `#pragma unroll` nest nvcc 12.9
// gives up on the elimination below for M = 8 and indexes W in local memory.)
template <int I, int End, class F>
BK4_DEV void static_for(F&& f) {
    if constexpr (I < End) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, End>(f);
    }
}

// Solve the grounded Laplacian system L d = -g, L_jk = -W_jk (j != k), L_jj = sum_{k != j} W_jk, unknowns j < M-1,
// ground = column M-1 (its links get `lam`), by node elimination in the order 0, 1, ...  W (packed) is destroyed.
// Eliminating node p gives its neighbours j, k > p the weight W_jk += W_pj W_pk / deg_p; the new degree of j is
// recomputed as the sum of its remaining weights, all non-negative: no subtraction anywhere (S7).
template <int M>
BK4_DEV void solve_laplacian(float (&W)[M * (M - 1) / 2], const float (&g)[M], float lam, float (&d)[M - 1]) {
    constexpr int K = M - 1;
    float deg[K], rhs[K], inv[K];
    static_for<0, K>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        W[tri<M>(j, K)] += lam;
    });
    static_for<0, K>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        float s = 0.0f;
        static_for<0, M>([&](auto kc) {
            constexpr int k = decltype(kc)::value;
            if constexpr (k != j) s += W[k > j ? tri<M>(j, k) : tri<M>(k, j)];
        });
        deg[j] = s;
        rhs[j] = -g[j];
    });
    static_for<0, K>([&](auto pc) {
        constexpr int p = decltype(pc)::value;
        inv[p] = rcp_approx(deg[p]);
        static_for<p + 1, K>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            const float f = W[tri<M>(p, j)] * inv[p];
            static_for<j + 1, M>([&](auto kc) {
                constexpr int k = decltype(kc)::value;
                W[tri<M>(j, k)] = fmaf(f, W[tri<M>(p, k)], W[tri<M>(j, k)]);
            });
            rhs[j] = fmaf(f, rhs[p], rhs[j]);
        });
        static_for<p + 1, K>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            float s = 0.0f;
            static_for<p + 1, M>([&](auto kc) {
                constexpr int k = decltype(kc)::value;
                if constexpr (k != j) s += W[k > j ? tri<M>(j, k) : tri<M>(k, j)];
            });
            deg[j] = s;
        });
    });
    // back substitution: d_p = (rhs_p + sum_{k > p, k < K} W_pk d_k) / deg_p
    static_for<0, K>([&](auto qc) {
        constexpr int p = K - 1 - decltype(qc)::value;
        float s = rhs[p];
        static_for<p + 1, K>([&](auto kc) {
            constexpr int k = decltype(kc)::value;
            s = fmaf(W[tri<M>(p, k)], d[k], s);
        });
        d[p] = s * inv[p];
    });
}

// One streamed evaluation at v: column sums c_j = sum_i T_ij, and (HESS) the packed edge weights
// W_jk = sum_i T_ij T_ik / a_i, with T_ij = a_i E_ij v_j / sum_k E_ik v_k and v_{M-1} = 1.
template <int N, int M, bool UNIT, bool HESS, bool PAD = false>
BK4_DEV void ot_eval(const float (&E)[N * M], const float (&v)[M - 1], const float (&a)[N], float (&c)[M],
                     float (&W)[M * (M - 1) / 2]) {
#pragma unroll
    for (int j = 0; j < M; ++j) c[j] = 0.0f;
    if constexpr (HESS) {
#pragma unroll
        for (int q = 0; q < M * (M - 1) / 2; ++q) W[q] = 0.0f;
    }
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float x[M], s = E[i * M + M - 1];
        x[M - 1] = s;
#pragma unroll
        for (int j = 0; j < M - 1; ++j) {
            x[j] = E[i * M + j] * v[j];
            s += x[j];
        }
        s = fmaxf(s, kOtTiny);  // a row whose every term underflowed: a finite (huge) residual instead of Inf * 0 = NaN
        float r = rcp_approx(s);
        r = fmaf(r, fmaf(-s, r, 1.0f), r);
        const float ar = UNIT ? r : a[i] * r;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            x[j] *= ar;  // T_ij
            c[j] += x[j];
        }
        if constexpr (HESS) {
            float ia = UNIT ? 1.0f : rcp_approx(a[i]);
            if constexpr (PAD) ia = a[i] > 0.0f ? ia : 0.0f;  // a padding row: T_i. = 0, and 0 x (1 / 0) must stay 0
#pragma unroll
            for (int j = 0; j < M - 1; ++j) {
                const float tj = UNIT ? x[j] : x[j] * ia;
#pragma unroll
                for (int k = j + 1; k < M; ++k) W[tri<M>(j, k)] = fmaf(tj, x[k], W[tri<M>(j, k)]);
            }
        }
    }
}

// E_ij = exp((beta_j - C_ij) / eta - mu_i) for the base potentials beta (beta_{M-1} = 0), mu_i the row maximum; E holds
// the raw costs (or logits) on entry.  sign = -1 for costs C (entropic OT), +1 for logits H = -C (Birkhoff
// projection).  Returns false if a NaN/Inf was met.
template <int N, int M>
BK4_DEV bool ot_exponentials(float sign_over_eta, const float (&beta_over_eta)[M - 1], float (&E)[N * M]) {
    float poison = 0.0f;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float u[M];
        float mx = -kInf;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            const float c = E[i * M + j];
            poison = __fmaf_rn(c, 0.0f, poison);
            u[j] = j < M - 1 ? fmaf(c, sign_over_eta * kLog2e, beta_over_eta[j]) : c * (sign_over_eta * kLog2e);
            mx = fmaxf(mx, u[j]);
        }
#pragma unroll
        for (int j = 0; j < M; ++j) E[i * M + j] = ex2_approx(u[j] - mx);
    }
    return poison == 0.0f;
}

// One Sinkhorn sweep in scaling form: u_i = a_i / sum_j E_ij v_j, q_j = sum_i E_ij u_i, v_j = (b_j / q_j) / (b_M / q_M).
template <int N, int M, bool UNIT>
BK4_DEV void ot_sweep(const float (&E)[N * M], float (&v)[M - 1], const float (&a)[N], const float (&b)[M]) {
    float q[M];
#pragma unroll
    for (int j = 0; j < M; ++j) q[j] = 0.0f;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float s = E[i * M + M - 1];
#pragma unroll
        for (int j = 0; j < M - 1; ++j) s = fmaf(E[i * M + j], v[j], s);
        s = fmaxf(s, kOtTiny);
        const float u = UNIT ? rcp_approx(s) : a[i] * rcp_approx(s);
#pragma unroll
        for (int j = 0; j < M; ++j) q[j] = fmaf(E[i * M + j], u, q[j]);
    }
    // (a column of E that underflowed to zero, e.g. under a tiny b_j late in the continuation, gives q_j = 0: clamped,
    // so that v_j becomes large and finite instead of Inf and the guard can still judge the step; bk4_guarded.cuh
    // clamps its column ratios for the same reason)
    const float t = UNIT ? fmaxf(q[M - 1], kOtTiny) : fmaxf(q[M - 1], kOtTiny) * rcp_approx(b[M - 1]);  // 1 / v_M before the gauge
#pragma unroll
    for (int j = 0; j < M - 1; ++j) v[j] = (UNIT ? t : b[j] * t) * rcp_approx(fmaxf(q[j], kOtTiny));
}

struct OtStats {
    int iters;
    bool converged;
};

// The whole forward for one problem.  Cg: this problem's N x M costs (or logits) in global memory, a, b: its
// marginals in registers (ignored when UNIT), T: where the result goes.  tol_rel: the stop threshold on
// Err_ab / sum(a) ... as an absolute threshold on the column part of Err_ab (rows are exact by construction).
template <int N, int M, bool UNIT, bool PAD = false>
BK4_DEV OtStats ot_forward_one(const float* Cg, float sign, float eta, const float (&a)[N], const float (&b)[M], float tol_abs,
                               int max_iter, float* Tg, OtShape sh = OtShape{N, M}) {
    static_assert(!(UNIT && PAD), "a padded problem carries its marginals (zeros on the padding)");
    float E[N * M], v[M - 1], vprev[M - 1], bl[M - 1], c[M], W[M * (M - 1) / 2];
    auto load_costs = [&](float(&X)[N * M]) {
        if constexpr (PAD) load_padded<N, M>(Cg, sh, X);
        else load_all<N, M>(Cg, X);
    };
    auto store_result_row = [&](int i, const float(&x)[M]) {
        if constexpr (PAD) store_padded_row<M>(Tg, sh, i, x);
        else store_row<M>(Tg + i * M, x);
    };
    // range of the costs decides the continuation schedule
    float lo = kInf, hi = -kInf, suma = 0.0f;
    load_costs(E);
#pragma unroll
    for (int i = 0; i < N; ++i) {
#pragma unroll
        for (int j = 0; j < M; ++j) {
            lo = fminf(lo, E[i * M + j]);
            hi = fmaxf(hi, E[i * M + j]);
        }
        suma += UNIT ? 1.0f : a[i];
    }
    if (!((hi - lo) < kInf)) {
        // an Inf among the costs: there is no finite range to build a continuation schedule on (it would run all 24
        // stages before the NaN came out); the result is the all-NaN matrix the header promises, at once
        float x[M];
#pragma unroll
        for (int j = 0; j < M; ++j) x[j] = kNaN;
#pragma unroll
        for (int i = 0; i < N; ++i) store_result_row(i, x);
        return OtStats{0, false};
    }
    const float lam = kOtLam * suma * (1.0f / N);
    float eta_s = eta;
    int stages = 0;
    while ((hi - lo) > kOtStageRange * eta_s && stages < 24) {
        eta_s *= 2.0f;
        ++stages;
    }
#pragma unroll
    for (int j = 0; j < M - 1; ++j) bl[j] = 0.0f;  // base potentials / eta_s in log2 units
    OtStats st = {0, false};
    bool finite = true;
    for (bool first = true;; eta_s *= 0.5f, --stages, first = false) {
        if (!first) load_costs(E);  // a later stage: the costs again (through L2)
        finite = ot_exponentials<N, M>(sign / eta_s, bl, E) && finite;
        if constexpr (PAD) {  // a padding column carries no mass
#pragma unroll
            for (int j = 0; j < M - 1; ++j)
                if (pad_slot<M>(sh, j)) {
#pragma unroll
                    for (int i = 0; i < N; ++i) E[i * M + j] = 0.0f;
                }
        }
#pragma unroll
        for (int j = 0; j < M - 1; ++j) v[j] = 1.0f;
        // Sinkhorn sweeps in the scaling form of eq. (2) PAPER.md:76 with marginals: u = a / (E v), v = b / (E^T u), gauge
        // v_M = 1 (two fused multiply-adds per entry; T itself is not formed)
        for (int k = 0; k < kOtSweeps; ++k) ot_sweep<N, M, UNIT>(E, v, a, b);
        const float tol_s = stages > 0 ? kOtStageTol * suma : tol_abs;
        float errprev = kInf, tstep = 1.0f, d[M - 1];
        unsigned newton_trial = 0u, sink_trial = 0u;
        int halvings = 0;
#pragma unroll
        for (int j = 0; j < M - 1; ++j) {
            vprev[j] = v[j];
            d[j] = 0.0f;
        }
        for (;;) {
            ot_eval<N, M, UNIT, true, PAD>(E, v, a, c, W);
            float g[M], err = 0.0f;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                g[j] = c[j] - (UNIT ? 1.0f : b[j]);
                err += fabsf(g[j]);
            }
            const bool conv = err <= tol_s;
            if ((newton_trial | sink_trial) && !(err < errprev) && !conv) {
                // the trial did not lower the residual (a line search decides the step size):
                // halve the Newton step up to kOtHalvings times, then a Sinkhorn column step, from the last accepted point
                if (st.iters < max_iter && newton_trial && halvings < kOtHalvings) {
                    tstep *= 0.5f;
                    ++halvings;
#pragma unroll
                    for (int j = 0; j < M - 1; ++j) v[j] = vprev[j] * ex2_approx(tstep * d[j]);
                    ++st.iters;
                    continue;
                }
                if (st.iters < max_iter && newton_trial) {
                    ot_eval<N, M, UNIT, false, PAD>(E, vprev, a, c, W);
                    const float t = (UNIT ? 1.0f : b[M - 1]) * rcp_approx(c[M - 1]);
#pragma unroll
                    for (int j = 0; j < M - 1; ++j) {
                        v[j] = vprev[j] * ((UNIT ? 1.0f : b[j]) * rcp_approx(c[j] * t));
                        if constexpr (PAD) v[j] = pad_slot<M>(sh, j) ? vprev[j] : v[j];  // c_j = b_j = 0 there
                    }
                    newton_trial = 0u, sink_trial = 1u;
                    ++st.iters;
                    continue;
                }
#pragma unroll
                for (int j = 0; j < M - 1; ++j) v[j] = vprev[j];  // nothing helps (fp32 floor), or no updates left
                break;
            }
            if (conv || !(err == err) || st.iters >= max_iter) {
                st.converged = conv && stages == 0;
                break;
            }
#pragma unroll
            for (int j = 0; j < M - 1; ++j) vprev[j] = v[j];
            errprev = err;
            solve_laplacian<M>(W, g, lam, d);
#pragma unroll
            for (int j = 0; j < M - 1; ++j) {
                d[j] = fminf(fmaxf(d[j], -30.0f), 30.0f) * kLog2e;  // kept in log2 units for the halvings
                v[j] *= ex2_approx(d[j]);
            }
            tstep = 1.0f, halvings = 0;
            newton_trial = 1u, sink_trial = 0u;
            ++st.iters;
        }
        if (stages <= 0) break;
        // next stage: eta halves, so potentials / eta double: beta/eta <- 2 (beta/eta + log2 v)
#pragma unroll
        for (int j = 0; j < M - 1; ++j) {
            bl[j] = 2.0f * (bl[j] + lg2_approx(v[j]));
            if constexpr (PAD) bl[j] = pad_slot<M>(sh, j) ? 0.0f : bl[j];  // (a sweep leaves v_j = 0 on a padding column)
        }
    }
    // the result: rows at the final v
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float x[M], s = E[i * M + M - 1];
        x[M - 1] = s;
#pragma unroll
        for (int j = 0; j < M - 1; ++j) {
            x[j] = E[i * M + j] * v[j];
            s += x[j];
        }
        float r = rcp_approx(s);
        r = fmaf(r, fmaf(-s, r, 1.0f), r);
        const float ar = UNIT ? r : a[i] * r;
#pragma unroll
        for (int j = 0; j < M; ++j) x[j] = finite ? x[j] * ar : kNaN;
        store_result_row(i, x);
    }
    st.converged = st.converged && finite;
    return st;
}

// Backward, eq. (13):  Gamma = G o T, mu_r = Gamma 1, mu_c = Gamma^T 1,
// Delta w = mu_c - T_{-M}^T (mu_r / a), w_M = 0, Delta = diag(c) - T_{-M}^T diag(a)^{-1} T_{-M} as a grounded Laplacian,
// D_ij = out_scale T_ij ((mu_r_i - (T w)_i) / a_i + w_j - G_ij),  out_scale = 1/eta for dl/dC, -1 for dl/dH of the
// Birkhoff projection.  The row marginals a are those of the given T.
template <int N, int M, bool PAD = false>
BK4_DEV void ot_backward_one(const float* Tg, const float* Gg, float out_scale, float* Dg, OtShape sh = OtShape{N, M}) {
    float T[N * M], G[N * M], W[M * (M - 1) / 2], mur[N], ia[N], rhs[M], w[M - 1];
    if constexpr (PAD) {
        load_padded_zero<N, M>(Tg, sh, T);
        load_padded_zero<N, M>(Gg, sh, G);
    } else {
        load_all<N, M>(Tg, T);
        load_all<N, M>(Gg, G);  // D may alias G: all of G is in registers before anything is written
    }
#pragma unroll
    for (int q = 0; q < M * (M - 1) / 2; ++q) W[q] = 0.0f;
#pragma unroll
    for (int j = 0; j < M; ++j) rhs[j] = 0.0f;
    float suma = 0.0f;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float ai = 0.0f, mr = 0.0f;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            ai += T[i * M + j];
            mr = fmaf(G[i * M + j], T[i * M + j], mr);
        }
        suma += ai;
        ia[i] = rcp_approx(ai);
        ia[i] = fmaf(ia[i], fmaf(-ai, ia[i], 1.0f), ia[i]);
        if constexpr (PAD) ia[i] = ai > 0.0f ? ia[i] : 0.0f;  // a padding row: everything it contributes is 0
        mur[i] = mr;
        const float mra = mr * ia[i];
#pragma unroll
        for (int j = 0; j < M; ++j) rhs[j] += fmaf(G[i * M + j], T[i * M + j], -T[i * M + j] * mra);  // mu_c_j - sum_i T_ij mu_r_i / a_i
#pragma unroll
        for (int j = 0; j < M - 1; ++j) {
            const float tj = T[i * M + j] * ia[i];
#pragma unroll
            for (int k = j + 1; k < M; ++k) W[tri<M>(j, k)] = fmaf(tj, T[i * M + k], W[tri<M>(j, k)]);
        }
    }
    float gneg[M];
#pragma unroll
    for (int j = 0; j < M; ++j) gneg[j] = -rhs[j];
    solve_laplacian<M>(W, gneg, kOtLam * suma * (1.0f / N), w);
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float tw = 0.0f, d[M];
#pragma unroll
        for (int j = 0; j < M - 1; ++j) tw = fmaf(T[i * M + j], w[j], tw);
        const float vi = (mur[i] - tw) * ia[i];
#pragma unroll
        for (int j = 0; j < M; ++j) d[j] = out_scale * T[i * M + j] * ((vi - G[i * M + j]) + (j < M - 1 ? w[j] : 0.0f));
        if constexpr (PAD) store_padded_row<M>(Dg, sh, i, d);
        else store_row<M>(Dg + i * M, d);
    }
}

}  // namespace bkot
