/*
 * ot_oracle.c -- fp64 CPU ORACLE for small batched entropic-regularised optimal transport, n x m with
 * n, m <= OT_MAX: the general problem of which the 4x4 Birkhoff projection is a special case
 * (section 2.3), and in particular the n = 8 Birkhoff projection.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may build, load or call it.  It shares no code, header, table or helper with
 * the CUDA path under paper_2606_07574_b200/csrc/ and is never a fallback for it.  It is a second, independent
 * file next to birkhoff4_oracle.c (which stays as committed in round 1); tests/test_oracle_ot.py checks that the
 * two agree where they overlap (n = m = 4, a = b = 1, eta = 1, M = -H).
 *
 * What it computes, and where the paper defines it:
 *
 *   forward   T = argmin_{T in Pi(a,b)} <T, M> - eta h(T)  (eq. (3)), the unique
 *             T_ij = exp((alpha_i + beta_j - M_ij) / eta) with T 1 = a, T^T 1 = b, found by
 *               tier 1: block coordinate ascent (7) PAPER.md:113 with the partial maximisers (5), (6)
 *                       (PAPER.md:103, 108), i.e. Sinkhorn-Knopp (2) in the log domain, until
 *                       Err_ab(T) = ||T1 - a||_1 + ||T^T1 - b||_1 <= tol * sum(a)  (Err: PAPER.md:323 with the
 *                       marginals a, b in place of 1);
 *               tier 2: only for problems tier 1 leaves above tol after `max_sweeps` sweeps (slow Sinkhorn,
 *                       PAPER.md:32): damped Newton on the FULL (n+m)-variable dual (4) PAPER.md:97 with a
 *                       pseudo-inverse solve (Jacobi eigen-decomposition), reached by continuation in eta.
 *             The output is self-certifying: scaling form by construction, measured Err_ab returned.
 *
 *   backward  D = dl/dM from G = dl/dT (eq. (13)), computed WITHOUT the gauge and without the
 *             paper's closed form: the linearised optimality system of PAPER.md:527-563 before beta_m is fixed,
 *               [diag(r) T; T^T diag(c)] [v; w] = [(G o T) 1; (G o T)^T 1]   (minimum-norm: singular along (1,-1)),
 *               D_ij = T_ij (v_i + w_j - G_ij) / eta,
 *             r, c the marginals of the given T.
 *
 * Pins (tests/test_oracle_ot.py, all CPU): T = a b^T / sum(a) for separable M; permutation equivariance; scaling
 * form + marginals; the 2x2 closed form with general marginals; eta-scaling and mass-scaling laws; the assignment
 * limit; agreement with birkhoff4_oracle.c; backward == central finite differences; the paper's closed form (13)
 * == this solve; an 80-digit solve at large scale.
 *
 * Layout: M, T, G, D: [B][n][m] row-major doubles; a: [B][n] or NULL (all ones); b: [B][m] or NULL.
 * Plain C99 + OpenMP over the batch; no SIMD intrinsics, no fast-math.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OT_MAX 16
#define KK (2 * OT_MAX)

typedef struct {
    int n, m;
    double eta;
    const double *M, *a, *b; /* a, b: this problem's marginals (never NULL here) */
} Prob;

/* Err_ab(T), PAPER.md:323 with marginals a, b */
static double err_ab(const Prob *p, const double *T)
{
    double e = 0.0;
    for (int i = 0; i < p->n; ++i) {
        double r = 0.0;
        for (int j = 0; j < p->m; ++j) r += T[i * p->m + j];
        e += fabs(r - p->a[i]);
    }
    for (int j = 0; j < p->m; ++j) {
        double c = 0.0;
        for (int i = 0; i < p->n; ++i) c += T[i * p->m + j];
        e += fabs(c - p->b[j]);
    }
    return e;
}

static double lse(const double *x, int k)
{
    double mx = x[0];
    for (int q = 1; q < k; ++q) if (x[q] > mx) mx = x[q];
    if (!(mx > -INFINITY && mx < INFINITY)) return mx;
    double s = 0.0;
    for (int q = 0; q < k; ++q) s += exp(x[q] - mx);
    return mx + log(s);
}

/* alpha*(beta), eq. (5):  alpha_i = eta log a_i - eta LSE_j((beta_j - M_ij) / eta) */
static void alpha_star(const Prob *p, double eta, const double *beta, double *alpha)
{
    double x[OT_MAX];
    for (int i = 0; i < p->n; ++i) {
        for (int j = 0; j < p->m; ++j) x[j] = (beta[j] - p->M[i * p->m + j]) / eta;
        alpha[i] = eta * log(p->a[i]) - eta * lse(x, p->m);
    }
}

/* beta*(alpha), eq. (6) */
static void beta_star(const Prob *p, double eta, const double *alpha, double *beta)
{
    double x[OT_MAX];
    for (int j = 0; j < p->m; ++j) {
        for (int i = 0; i < p->n; ++i) x[i] = (alpha[i] - p->M[i * p->m + j]) / eta;
        beta[j] = eta * log(p->b[j]) - eta * lse(x, p->n);
    }
}

/* primal recovery T_ij = exp((alpha_i + beta_j - M_ij) / eta) */
static void primal(const Prob *p, double eta, const double *alpha, const double *beta, double *T)
{
    for (int i = 0; i < p->n; ++i)
        for (int j = 0; j < p->m; ++j) T[i * p->m + j] = exp((alpha[i] + beta[j] - p->M[i * p->m + j]) / eta);
}

/* -L(alpha, beta) of the dual (4) */
static double neg_dual(const Prob *p, double eta, const double *alpha, const double *beta)
{
    double s = 0.0;
    for (int i = 0; i < p->n; ++i)
        for (int j = 0; j < p->m; ++j) s += eta * exp((alpha[i] + beta[j] - p->M[i * p->m + j]) / eta);
    for (int i = 0; i < p->n; ++i) s -= alpha[i] * p->a[i];
    for (int j = 0; j < p->m; ++j) s -= beta[j] * p->b[j];
    return s;
}

/* cyclic Jacobi eigen-decomposition of a symmetric k x k matrix: A = V diag(w) V^T */
static void jacobi_eig(int k, double *A, double *V, double *w)
{
    for (int p = 0; p < k; ++p)
        for (int q = 0; q < k; ++q) V[p * k + q] = (p == q) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 100; ++sweep) {
        double off = 0.0, dia = 0.0;
        for (int p = 0; p < k; ++p)
            for (int q = 0; q < k; ++q) {
                if (p == q) dia += A[p * k + p] * A[p * k + p];
                else off += A[p * k + q] * A[p * k + q];
            }
        if (off <= 1e-60 * dia || off == 0.0) break;
        for (int p = 0; p < k - 1; ++p)
            for (int q = p + 1; q < k; ++q) {
                double apq = A[p * k + q];
                if (apq == 0.0) continue;
                double theta = (A[q * k + q] - A[p * k + p]) / (2.0 * apq);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double cs = 1.0 / sqrt(t * t + 1.0), sn = t * cs;
                for (int r = 0; r < k; ++r) {
                    double arp = A[r * k + p], arq = A[r * k + q];
                    A[r * k + p] = cs * arp - sn * arq;
                    A[r * k + q] = sn * arp + cs * arq;
                }
                for (int r = 0; r < k; ++r) {
                    double apr = A[p * k + r], aqr = A[q * k + r];
                    A[p * k + r] = cs * apr - sn * aqr;
                    A[q * k + r] = sn * apr + cs * aqr;
                }
                for (int r = 0; r < k; ++r) {
                    double vrp = V[r * k + p], vrq = V[r * k + q];
                    V[r * k + p] = cs * vrp - sn * vrq;
                    V[r * k + q] = sn * vrp + cs * vrq;
                }
            }
    }
    for (int p = 0; p < k; ++p) w[p] = A[p * k + p];
}

/* y = K^+ rhs for a symmetric k x k K; eigenvalues <= rcond * max dropped */
static void pinv_apply(int k, const double *Kin, const double *rhs, double *y, double rcond)
{
    double K[KK * KK], V[KK * KK], w[KK];
    memcpy(K, Kin, sizeof(double) * k * k);
    jacobi_eig(k, K, V, w);
    double wmax = 0.0;
    for (int q = 0; q < k; ++q) if (fabs(w[q]) > wmax) wmax = fabs(w[q]);
    for (int q = 0; q < k; ++q) y[q] = 0.0;
    for (int q = 0; q < k; ++q) {
        if (!(fabs(w[q]) > rcond * wmax)) continue;
        double proj = 0.0;
        for (int r = 0; r < k; ++r) proj += V[r * k + q] * rhs[r];
        proj /= w[q];
        for (int r = 0; r < k; ++r) y[r] += V[r * k + q] * proj;
    }
}

/* [diag(r) T; T^T diag(c)], r, c the marginals of T: eta times the Hessian of -L */
static void kkt_matrix(int n, int m, const double *T, double *K, double *r, double *c)
{
    int k = n + m;
    memset(K, 0, sizeof(double) * k * k);
    for (int i = 0; i < n; ++i) r[i] = 0.0;
    for (int j = 0; j < m; ++j) c[j] = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < m; ++j) {
            double t = T[i * m + j];
            r[i] += t;
            c[j] += t;
            K[i * k + n + j] = t;
            K[(n + j) * k + i] = t;
        }
    for (int i = 0; i < n; ++i) K[i * k + i] = r[i];
    for (int j = 0; j < m; ++j) K[(n + j) * k + n + j] = c[j];
}

/* damped Newton on the full dual at regularisation eta, from beta (updated in place); leaves the best T seen */
static double newton_full_dual(const Prob *p, double eta, double *beta, double *T, double tol, int max_newton, int *steps)
{
    int n = p->n, m = p->m, k = n + m;
    double alpha[OT_MAX], bestT[OT_MAX * OT_MAX], bestb[OT_MAX], beste;
    alpha_star(p, eta, beta, alpha);
    primal(p, eta, alpha, beta, T);
    beste = err_ab(p, T);
    memcpy(bestT, T, sizeof(double) * n * m);
    memcpy(bestb, beta, sizeof(double) * m);
    int stall = 0;
    for (int it = 0; it < max_newton && beste > tol; ++it) {
        double K[KK * KK], rhs[KK], y[KK], r[OT_MAX], c[OT_MAX];
        kkt_matrix(n, m, T, K, r, c);
        for (int i = 0; i < n; ++i) rhs[i] = p->a[i] - r[i];
        for (int j = 0; j < m; ++j) rhs[n + j] = p->b[j] - c[j];
        pinv_apply(k, K, rhs, y, 1e-15);
        double slope = 0.0;
        for (int q = 0; q < k; ++q) slope -= rhs[q] * y[q] * eta;
        double f0 = neg_dual(p, eta, alpha, beta), t = 1.0, an[OT_MAX], bn[OT_MAX];
        int ok = 0;
        for (int h = 0; h < 60; ++h) {
            for (int i = 0; i < n; ++i) an[i] = alpha[i] + t * eta * y[i];
            for (int j = 0; j < m; ++j) bn[j] = beta[j] + t * eta * y[n + j];
            double f1 = neg_dual(p, eta, an, bn);
            if (f1 <= f0 + 1e-4 * t * slope + 1e-13 * (1.0 + fabs(f0))) { ok = 1; break; }
            t *= 0.5;
        }
        if (!ok) break;
        memcpy(beta, bn, sizeof(double) * m);
        alpha_star(p, eta, beta, alpha);
        primal(p, eta, alpha, beta, T);
        double e = err_ab(p, T);
        ++*steps;
        if (e != e) { beste = e; memcpy(bestT, T, sizeof(double) * n * m); break; }
        if (e < beste) {
            stall = (e > 0.5 * beste) ? stall + 1 : 0;
            beste = e;
            memcpy(bestT, T, sizeof(double) * n * m);
            memcpy(bestb, beta, sizeof(double) * m);
        } else {
            ++stall;
        }
        if (stall >= 4 && beste < 1e-10) break;
    }
    memcpy(T, bestT, sizeof(double) * n * m);
    memcpy(beta, bestb, sizeof(double) * m);
    return beste;
}

static int forward_one(const Prob *p, double *T, double tol, int max_sweeps, int max_newton, int *sweeps, int *newton,
                       double *err)
{
    int n = p->n, m = p->m;
    double alpha[OT_MAX], beta[OT_MAX], suma = 0.0, e = INFINITY;
    *sweeps = 0;
    *newton = 0;
    int bad = !(p->eta > 0.0 && p->eta < INFINITY);
    for (int q = 0; q < n * m; ++q) if (!(fabs(p->M[q]) < INFINITY)) bad = 1;
    for (int i = 0; i < n; ++i) { if (!(p->a[i] > 0.0 && p->a[i] < INFINITY)) bad = 1; suma += p->a[i]; }
    for (int j = 0; j < m; ++j) if (!(p->b[j] > 0.0 && p->b[j] < INFINITY)) bad = 1;
    if (bad) {
        for (int q = 0; q < n * m; ++q) T[q] = NAN;
        *err = NAN;
        return 1;
    }
    tol *= suma;
    for (int j = 0; j < m; ++j) beta[j] = 0.0;
    int k = 0;
    for (;;) { /* tier 1: BCA (7) */
        alpha_star(p, p->eta, beta, alpha);
        primal(p, p->eta, alpha, beta, T);
        e = err_ab(p, T);
        if (!(e > tol) || k >= max_sweeps) break;
        beta_star(p, p->eta, alpha, beta);
        ++k;
    }
    *sweeps = k;
    *err = e;
    if (!(e > tol) || e != e) return 1;
    /* tier 2: continuation in eta from a value at which the scaled costs span <= 8, halving down to eta */
    double lo = p->M[0], hi = p->M[0];
    for (int q = 1; q < n * m; ++q) { if (p->M[q] < lo) lo = p->M[q]; if (p->M[q] > hi) hi = p->M[q]; }
    double eta = p->eta;
    while ((hi - lo) / eta > 8.0) eta *= 2.0;
    for (int j = 0; j < m; ++j) beta[j] = 0.0;
    for (;;) {
        e = newton_full_dual(p, eta, beta, T, eta > p->eta ? 1e-9 * suma : tol, max_newton, newton);
        if (!(eta > p->eta)) break;
        eta *= 0.5;
        if (eta < p->eta) eta = p->eta;
        /* the potentials of the entropic problem tend to those of the LP as eta -> 0: warm start unchanged */
    }
    *err = e;
    return 2;
}

static void backward_one(int n, int m, double eta, const double *T, const double *G, double *D, double rcond)
{
    int k = n + m;
    double K[KK * KK], rhs[KK], y[KK], r[OT_MAX], c[OT_MAX];
    kkt_matrix(n, m, T, K, r, c);
    for (int q = 0; q < k; ++q) rhs[q] = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < m; ++j) {
            double gm = G[i * m + j] * T[i * m + j];
            rhs[i] += gm;     /* mu_r = (G o T) 1 */
            rhs[n + j] += gm; /* mu_c over ALL columns: no gauge fixed */
        }
    pinv_apply(k, K, rhs, y, rcond);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < m; ++j) D[i * m + j] = T[i * m + j] * (y[i] + y[n + j] - G[i * m + j]) / eta;
}

/* ================================ exported batch entry points ================================= */
static const double ONES[OT_MAX] = {1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1};

int oto_max_dim(void) { return OT_MAX; }

/* returns the number of problems whose final Err_ab exceeds certify * sum(a); -1 for bad dimensions */
int64_t oto_forward(const double *M, const double *a, const double *b, double *T, int64_t B, int n, int m, double eta,
                    double tol, int max_sweeps, int max_newton, double certify, int32_t *tier, double *err, int nthreads)
{
    if (n < 1 || m < 1 || n > OT_MAX || m > OT_MAX) return -1;
    int64_t bad = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads) reduction(+ : bad)
#endif
    for (int64_t q = 0; q < B; ++q) {
        Prob p = {n, m, eta, M + q * n * m, a ? a + q * n : ONES, b ? b + q * m : ONES};
        int sw, nw;
        double e;
        int t = forward_one(&p, T + q * n * m, tol, max_sweeps, max_newton, &sw, &nw, &e);
        double suma = 0.0;
        for (int i = 0; i < n; ++i) suma += p.a[i];
        if (tier) tier[q] = t;
        if (err) err[q] = e;
        if (!(e <= certify * suma)) ++bad;
    }
    return bad;
}

void oto_backward(const double *T, const double *G, double *D, int64_t B, int n, int m, double eta, double rcond, int nthreads)
{
    if (n < 1 || m < 1 || n > OT_MAX || m > OT_MAX) return;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (int64_t q = 0; q < B; ++q) backward_one(n, m, eta, T + q * n * m, G + q * n * m, D + q * n * m, rcond);
}

/* Err_ab per problem */
void oto_marginal_err(const double *T, const double *a, const double *b, double *err, int64_t B, int n, int m)
{
    for (int64_t q = 0; q < B; ++q) {
        Prob p = {n, m, 1.0, NULL, a ? a + q * n : ONES, b ? b + q * m : ONES};
        err[q] = err_ab(&p, T + q * n * m);
    }
}
