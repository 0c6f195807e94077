/*
 * birkhoff4_oracle.c -- fp64 CPU ORACLE for the batched 4x4 Birkhoff (KL / entropic-OT) projection.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2606_07574_b200/csrc/ and is never a
 * fallback for it.
 *
 * What it computes, and where the paper defines it:
 *
 *   forward   P = proj^KL_{B_4}(exp(H)): the unique P_ij = exp(a_i + H_ij + b_j) with unit row and
 *             column sums (eq. (1); Sinkhorn's theorem PAPER.md:62; KKT form
 *             PAPER.md:428-432).  The method reaches this P exactly, so the oracle is the plain
 *             definition, found by
 *               tier 1: Sinkhorn-Knopp in the log domain, eq. (2) PAPER.md:76 written with the
 *                       partial maximisers (5),(6) at eta=1, a=b=1, i.e. BCA (7),
 *                       run until Err(P) <= tol (Err: PAPER.md:323), tol = 1e-14 by default;
 *               tier 2: only for matrices tier 1 leaves above tol after `max_sweeps` sweeps (Sinkhorn
 *                       converges slowly at large |H|): damped Newton on the FULL
 *                       8-variable dual (4) with a generic pseudo-inverse solve
 *                       (Jacobi eigen-decomposition), reached by continuation in the regularisation
 *                       parameter eta of (3)/(4).  Different formulation from the GPU's 3-variable path.
 *             Whichever tier produced it the output is self-certifying: it has the scaling form by
 *             construction and its measured Err is returned per matrix (uniqueness => it is the
 *             projection).
 *
 *   backward  dH = J^T vec(G), J = d vec(P) / d vec(H), by solving the linearised KKT system of
 *             the projection directly (the derivation of PAPER.md:527-563 BEFORE the gauge is
 *             fixed):  [diag(r) P; P^T diag(c)] [v; w] = [(G o P) 1; (G o P)^T 1]  in the
 *             minimum-norm sense (the matrix is singular along (1,-1)), then
 *             dH_ij = P_ij (G_ij - v_i - w_j)   ( = -D of PAPER.md:302-304, sign for R = -M).
 *
 *   sinkhorn  K = exp(H); n_iter x (row-normalise, column-normalise): the "Sinkhorn-20" recipe of
 *             Xie et al. the paper benchmarks against (eq. (2) with v0 = 1).
 *
 *   marginal_err  Err(T) = ||T1 - 1||_1 + ||T^T 1 - 1||_1.
 *
 * Pins (tests/test_oracle_*.py, all CPU): P = 1/4 for additively separable H; permutation
 * equivariance; rank-2 additivity of log P - H; unit marginals; the 2x2 closed form embedded in a
 * 4x4; max-weight assignment support as s -> inf; backward == central finite differences of forward;
 * dH row/col sums zero; the paper's closed form (13) == this KKT solve; Sinkhorn-20 statistics of
 * PAPER.md Table 2.
 *
 * Layout: [B][4][4] row-major doubles (fp32/bf16 inputs are widened exactly by the caller).
 * Plain C99 + OpenMP over the batch; no SIMD intrinsics, no fast-math.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define N4 4

/* ---- Err(T), PAPER.md:323 -------------------------------------------------------------------- */
static double err_one(const double *T)
{
    double e = 0.0;
    for (int i = 0; i < N4; ++i) {
        double r = 0.0;
        for (int j = 0; j < N4; ++j) r += T[4 * i + j];
        e += fabs(r - 1.0);
    }
    for (int j = 0; j < N4; ++j) {
        double c = 0.0;
        for (int i = 0; i < N4; ++i) c += T[4 * i + j];
        e += fabs(c - 1.0);
    }
    return e;
}

/* max-shifted log-sum-exp of 4 numbers */
static double lse4(const double *x)
{
    double m = x[0];
    for (int k = 1; k < N4; ++k) if (x[k] > m) m = x[k];
    if (!(m > -INFINITY && m < INFINITY)) return m; /* all -inf, or +inf/NaN: propagate */
    double s = 0.0;
    for (int k = 0; k < N4; ++k) s += exp(x[k] - m);
    return m + log(s);
}

/* alpha*(beta), eq. (5) PAPER.md:103 with eta=1, a=1, M=-H:  a_i = -LSE_j(H_ij + b_j) */
static void alpha_star(const double *H, const double *b, double *a)
{
    for (int i = 0; i < N4; ++i) {
        double x[4];
        for (int j = 0; j < N4; ++j) x[j] = H[4 * i + j] + b[j];
        a[i] = -lse4(x);
    }
}

/* beta*(alpha), eq. (6):  b_j = -LSE_i(H_ij + a_i) */
static void beta_star(const double *H, const double *a, double *b)
{
    for (int j = 0; j < N4; ++j) {
        double x[4];
        for (int i = 0; i < N4; ++i) x[i] = H[4 * i + j] + a[i];
        b[j] = -lse4(x);
    }
}

/* primal recovery T_ij = exp(a_i + b_j - M_ij) */
static void primal(const double *H, const double *a, const double *b, double *P)
{
    for (int i = 0; i < N4; ++i)
        for (int j = 0; j < N4; ++j) P[4 * i + j] = exp(a[i] + H[4 * i + j] + b[j]);
}

/* -L(alpha, beta) of the dual (4), a=b=1, for the cost M = -H (H already divided by eta;
 * the problem at regularisation eta is the eta=1 problem for H/eta with duals alpha/eta, beta/eta) */
static double neg_dual(const double *H, const double *a, const double *b)
{
    double s = 0.0;
    for (int i = 0; i < N4; ++i)
        for (int j = 0; j < N4; ++j) s += exp(a[i] + H[4 * i + j] + b[j]);
    for (int k = 0; k < N4; ++k) s -= a[k] + b[k];
    return s;
}

/* cyclic Jacobi eigen-decomposition of a symmetric n x n matrix (n <= 8): A = V diag(w) V^T */
static void jacobi_eig(int n, double *A, double *V, double *w)
{
    for (int p = 0; p < n; ++p)
        for (int q = 0; q < n; ++q) V[p * n + q] = (p == q) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 64; ++sweep) {
        double off = 0.0, dia = 0.0;
        for (int p = 0; p < n; ++p)
            for (int q = 0; q < n; ++q) {
                if (p == q) dia += A[p * n + p] * A[p * n + p];
                else off += A[p * n + q] * A[p * n + q];
            }
        if (off <= 1e-60 * dia || off == 0.0) break;
        for (int p = 0; p < n - 1; ++p)
            for (int q = p + 1; q < n; ++q) {
                double apq = A[p * n + q];
                if (apq == 0.0) continue;
                double theta = (A[q * n + q] - A[p * n + p]) / (2.0 * apq);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double cs = 1.0 / sqrt(t * t + 1.0), sn = t * cs;
                for (int k = 0; k < n; ++k) { /* columns p,q of A */
                    double akp = A[k * n + p], akq = A[k * n + q];
                    A[k * n + p] = cs * akp - sn * akq;
                    A[k * n + q] = sn * akp + cs * akq;
                }
                for (int k = 0; k < n; ++k) { /* rows p,q of A */
                    double apk = A[p * n + k], aqk = A[q * n + k];
                    A[p * n + k] = cs * apk - sn * aqk;
                    A[q * n + k] = sn * apk + cs * aqk;
                }
                for (int k = 0; k < n; ++k) {
                    double vkp = V[k * n + p], vkq = V[k * n + q];
                    V[k * n + p] = cs * vkp - sn * vkq;
                    V[k * n + q] = sn * vkp + cs * vkq;
                }
            }
    }
    for (int p = 0; p < n; ++p) w[p] = A[p * n + p];
}

/* y = K^+ rhs for a symmetric 8x8 K via its eigen-decomposition; eigenvalues <= rcond*max dropped */
static void pinv_apply(const double *Kin, const double *rhs, double *y, double rcond)
{
    double K[64], V[64], w[8];
    memcpy(K, Kin, sizeof K);
    jacobi_eig(8, K, V, w);
    double wmax = 0.0;
    for (int k = 0; k < 8; ++k) if (fabs(w[k]) > wmax) wmax = fabs(w[k]);
    memset(y, 0, 8 * sizeof(double));
    for (int k = 0; k < 8; ++k) {
        if (!(fabs(w[k]) > rcond * wmax)) continue;
        double proj = 0.0;
        for (int p = 0; p < 8; ++p) proj += V[p * 8 + k] * rhs[p];
        proj /= w[k];
        for (int p = 0; p < 8; ++p) y[p] += V[p * 8 + k] * proj;
    }
}

/* the KKT matrix [diag(r) P; P^T diag(c)] = Hessian of -L of the dual (4); r, c = marginals of P */
static void kkt_matrix(const double *P, double *K, double *r, double *c)
{
    memset(K, 0, 64 * sizeof(double));
    for (int k = 0; k < N4; ++k) r[k] = c[k] = 0.0;
    for (int i = 0; i < N4; ++i)
        for (int j = 0; j < N4; ++j) {
            double p = P[4 * i + j];
            r[i] += p;
            c[j] += p;
            K[i * 8 + 4 + j] = p;
            K[(4 + j) * 8 + i] = p;
        }
    for (int k = 0; k < N4; ++k) { K[k * 8 + k] = r[k]; K[(4 + k) * 8 + 4 + k] = c[k]; }
}

/*
 * Damped Newton on the full 8-variable dual (4) for the cost -Hs, from the column potentials b
 * (updated in place).  Each step: rows made exact (alpha*(beta), eq. (5)), step = K^+ [1-r; 1-c]
 * (minimum-norm: the gauge direction PAPER.md:132 is the null vector), backtracking on -L.
 * Stops at Err <= tol, after max_newton steps, or when Err has stopped improving.
 * Leaves the best P seen in P and returns its Err; *steps += steps taken.
 */
static double newton_full_dual(const double *Hs, double *b, double *P, double tol, int max_newton, int *steps)
{
    double a[4], bestP[16], bestb[4], beste;
    alpha_star(Hs, b, a);
    primal(Hs, a, b, P);
    beste = err_one(P);
    memcpy(bestP, P, sizeof bestP);
    memcpy(bestb, b, sizeof bestb);
    int stall = 0;
    for (int it = 0; it < max_newton && beste > tol; ++it) {
        double K[64], rhs[8], y[8], r[4], c[4];
        kkt_matrix(P, K, r, c);
        for (int k = 0; k < N4; ++k) { rhs[k] = 1.0 - r[k]; rhs[4 + k] = 1.0 - c[k]; }
        pinv_apply(K, rhs, y, 1e-15);
        double slope = 0.0; /* grad(-L)^T step <= 0 */
        for (int k = 0; k < 8; ++k) slope -= rhs[k] * y[k];
        double f0 = neg_dual(Hs, a, b), t = 1.0, an[4], bn[4];
        int ok = 0;
        for (int h = 0; h < 60; ++h) {
            for (int k = 0; k < N4; ++k) { an[k] = a[k] + t * y[k]; bn[k] = b[k] + t * y[4 + k]; }
            double f1 = neg_dual(Hs, an, bn);
            if (f1 <= f0 + 1e-4 * t * slope + 1e-13 * (1.0 + fabs(f0))) { ok = 1; break; }
            t *= 0.5;
        }
        if (!ok) break;
        memcpy(b, bn, 4 * sizeof(double));
        alpha_star(Hs, b, a); /* exact maximisation over alpha: never increases -L; rows exact */
        primal(Hs, a, b, P);
        double e = err_one(P);
        ++*steps;
        if (e != e) { beste = e; memcpy(bestP, P, sizeof bestP); break; }
        if (e < beste) {
            stall = (e > 0.5 * beste) ? stall + 1 : 0;
            beste = e; memcpy(bestP, P, sizeof bestP); memcpy(bestb, b, sizeof bestb);
        } else {
            ++stall;
        }
        if (stall >= 4 && beste < 1e-10) break; /* at the fp64 floor for this magnitude */
    }
    memcpy(P, bestP, sizeof bestP);
    memcpy(b, bestb, 4 * sizeof(double));
    return beste;
}

/*
 * forward for one matrix.  Returns the tier that produced P (1 or 2); *sweeps = Sinkhorn sweeps
 * used, *newton = tier-2 Newton steps used, *err = Err(P) of the returned P.
 */
static int forward_one(const double *H, double *P, double tol, int max_sweeps, int max_newton,
                       int *sweeps, int *newton, double *err)
{
    double a[4], b[4] = {0.0, 0.0, 0.0, 0.0};
    double e = INFINITY;
    int k = 0;
    *newton = 0;
    *sweeps = 0;
    for (int q = 0; q < 16; ++q)
        if (!(fabs(H[q]) < INFINITY)) { /* NaN/Inf logit: the projection is undefined -> all NaN */
            for (int p = 0; p < 16; ++p) P[p] = NAN;
            *err = NAN;
            return 1;
        }
    /* tier 1: BCA (7) PAPER.md:113 == Sinkhorn-Knopp (2).  alpha is updated last so that rows are
     * exact when P is formed; Err is then the column residual plus rounding. */
    for (;;) {
        alpha_star(H, b, a);
        primal(H, a, b, P);
        e = err_one(P);
        if (!(e > tol) || k >= max_sweeps) break; /* also leaves on NaN */
        beta_star(H, a, b);
        ++k;
    }
    *sweeps = k;
    *err = e;
    if (!(e > tol) || e != e) return 1;

    /* tier 2: continuation in the regularisation parameter eta of (3)/(4), from an
     * eta at which the scaled logits H/eta span <= 8 down to eta = 1 by halving; at each eta damped
     * Newton on the full dual, warm-started from the previous stage's potentials (which scale as
     * 1/eta).  Intermediate stages are solved loosely, the last one to `tol`. */
    double lo = H[0], hi = H[0];
    for (int q = 1; q < 16; ++q) { if (H[q] < lo) lo = H[q]; if (H[q] > hi) hi = H[q]; }
    double eta = 1.0;
    while ((hi - lo) / eta > 8.0) eta *= 2.0;
    for (int q = 0; q < N4; ++q) b[q] = 0.0;
    for (;;) {
        double Hs[16];
        for (int q = 0; q < 16; ++q) Hs[q] = H[q] / eta;
        e = newton_full_dual(Hs, b, P, eta > 1.0 ? 1e-9 : tol, max_newton, newton);
        if (!(eta > 1.0)) break;
        eta *= 0.5;
        for (int q = 0; q < N4; ++q) b[q] *= 2.0;
    }
    *err = e;
    return 2;
}

/* backward for one matrix: minimum-norm solve of the linearised KKT system (see header) */
static void backward_one(const double *P, const double *G, double *dH, double rcond)
{
    double K[64], rhs[8], y[8], r[4], c[4];
    kkt_matrix(P, K, r, c);
    memset(rhs, 0, sizeof rhs);
    for (int i = 0; i < N4; ++i)
        for (int j = 0; j < N4; ++j) {
            double gm = G[4 * i + j] * P[4 * i + j];
            rhs[i] += gm;     /* mu_r = (G o P) 1, */
            rhs[4 + j] += gm; /* mu_c = (G o P)^T 1 (all 4 columns: no gauge fixed yet) */
        }
    pinv_apply(K, rhs, y, rcond);
    for (int i = 0; i < N4; ++i)
        for (int j = 0; j < N4; ++j)
            dH[4 * i + j] = P[4 * i + j] * (G[4 * i + j] - y[i] - y[4 + j]);
}

/* ================================ exported batch entry points ================================= */

int bk4o_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void bk4o_marginal_err(const double *T, double *err, int64_t B)
{
    for (int64_t b = 0; b < B; ++b) err[b] = err_one(T + 16 * b);
}

/*
 * forward.  H,P: [B][16].  tier/sweeps/newton/err: [B] or NULL.  nthreads<=0: all OpenMP threads.
 * Returns the number of matrices whose final Err exceeds `certify` (pass 1e-12).
 */
int64_t bk4o_forward(const double *H, double *P, int64_t B, double tol, int max_sweeps, int max_newton,
                     double certify, int32_t *tier, int32_t *sweeps, int32_t *newton, double *err,
                     int nthreads)
{
    int64_t bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads) reduction(+ : bad)
#endif
    for (int64_t b = 0; b < B; ++b) {
        int sw, nw;
        double e;
        int t = forward_one(H + 16 * b, P + 16 * b, tol, max_sweeps, max_newton, &sw, &nw, &e);
        if (tier) tier[b] = t;
        if (sweeps) sweeps[b] = sw;
        if (newton) newton[b] = nw;
        if (err) err[b] = e;
        if (!(e <= certify)) ++bad;
    }
    return bad;
}

void bk4o_backward(const double *P, const double *G, double *dH, int64_t B, double rcond, int nthreads)
{
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (int64_t b = 0; b < B; ++b) backward_one(P + 16 * b, G + 16 * b, dH + 16 * b, rcond);
}

/* Sinkhorn-Knopp, eq. (2) PAPER.md:76 in matrix form: K = exp(H); n_iter x (rows /= sum, cols /= sum) */
void bk4o_sinkhorn(const double *H, double *T, int64_t B, int n_iter, int nthreads)
{
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (int64_t b = 0; b < B; ++b) {
        const double *h = H + 16 * b;
        double *t = T + 16 * b;
        for (int k = 0; k < 16; ++k) t[k] = exp(h[k]);
        for (int it = 0; it < n_iter; ++it) {
            for (int i = 0; i < N4; ++i) {
                double s = 0.0;
                for (int j = 0; j < N4; ++j) s += t[4 * i + j];
                for (int j = 0; j < N4; ++j) t[4 * i + j] /= s;
            }
            for (int j = 0; j < N4; ++j) {
                double s = 0.0;
                for (int i = 0; i < N4; ++i) s += t[4 * i + j];
                for (int i = 0; i < N4; ++i) t[4 * i + j] /= s;
            }
        }
    }
}
