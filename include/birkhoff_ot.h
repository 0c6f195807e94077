/*
 * birkhoff_ot.h -- C ABI (part of libbirkhoff4.so) of the widenings of the 4x4 hot path that the paper itself
 * names: the n = 8 Birkhoff projection ("n = 4 or 8") and small general entropic-regularised
 * optimal transport with arbitrary marginals a, b and regularisation eta (PAPER.md:83-168 forward, eq. (13)
 * PAPER.md:255-282 backward).  SURVEY.md 8(f) NEXT-1 and NEXT-3.
 *
 *   forward   T = argmin_{T in Pi(a,b)} <T, C> - eta h(T)  (eq. (3)) by Newton's method on the
 *             (m-1)-variable dual (eq. (8), gradient and Hessian eq. (9)),
 *             guarded step, stop on the marginal error.  Wide costs are reached by continuation
 *             in eta.  The n x n Birkhoff projection of exp(H) is the case C = -H, eta = 1,
 *             a = b = 1.
 *   backward  D = dl/dC from T and G = dl/dT by eq. (13) PAPER.md:273-280 (for Birkhoff: dl/dH = -D).
 *
 * Conventions (all entry points)
 *   layout     [B][n][m] row-major contiguous; marginals a [B][n], b [B][m].
 *   sizes      any 2 <= n, m <= 8; anything else returns BIRKHOFF_OT_EINVAL.  The four sizes {4, 8} x {4, 8} have
 *              kernels of their own (vector loads, tuned register budgets).  Every other size runs inside the
 *              next of those tiles: rows beyond n carry mass 0 and columns beyond m carry mass 0 and no entries
 *              (a zero marginal is outside the domain of eq. (5), so the padding is kept out of
 *              the formulas by construction rather than passed through them), scalar loads and stores; correct
 *              to the same gates, not tuned.
 *   pointers   DEVICE pointers owned by the caller; the library neither allocates nor synchronises; every call
 *              is asynchronous on `stream` (a cudaStream_t; 0 = the legacy default stream).
 *   alignment  every matrix pointer must be 32-byte aligned for the sizes {4, 8} x {4, 8} (256-bit accesses); the
 *              other sizes are accessed float by float and need 4-byte alignment only (else BIRKHOFF_OT_EINVAL).
 *   aliasing   T == C and D == G are allowed as exact aliases; partial overlap is undefined.
 *   marginals  a and b both NULL: all ones (needs n == m).  Otherwise both given, positive, sum a = sum b
 *              (PAPER.md:91-93); not checked.
 *   tol        stop when Err_ab(T) = ||T1 - a||_1 + ||T^T1 - b||_1 (PAPER.md:323 with marginals a, b) <= tol.
 *              Rows equal a by construction, so the kernel tests the column part against tol / 2.  fp32 floor:
 *              about 2.5e-7 per unit of sum(a) / 4 (so 1e-6 is reachable for 4x4 with unit marginals, 2e-6 for 8x8).
 *   max_iter   maximum number of updates of beta over all continuation stages.  An update is a Newton step, a
 *              retry of a Newton step at half its length (up to four per step, when the step did not lower the
 *              residual) or a fallback Sinkhorn step; `iters` counts the same.  The three Sinkhorn sweeps that
 *              start each stage are not counted.
 *   regime     costs of any finite range: a range wider than 16 eta is reached by continuation (eta 2^K, ..., 2 eta,
 *              eta, at most 24 halvings, i.e. range / eta up to 2.7e8), every stage drawing on the same max_iter;
 *              a problem that runs out of updates on the way is written as it stands (rows equal to a) and counted
 *              in n_unconverged.  Tested against the oracle for range / eta up to about 1000 (n = 8 logits
 *              N(0,100^2); costs N(0,3^2) at eta = 0.1) and for marginals down to 1e-6 of the total mass, where 60
 *              to 80 updates suffice; max_iter = 40 covers range / eta up to about 100.
 *   NaN/Inf    a problem holding a NaN or Inf cost gives an all-NaN T for that problem only.
 *   errors     0 on success; BIRKHOFF_OT_EINVAL for bad sizes, a null or misaligned pointer with B > 0, B < 0,
 *              tol < 0 or NaN, max_iter < 0, eta <= 0 or not finite, exactly one of a, b NULL;
 *              BIRKHOFF_OT_ECUDA_BASE + cudaError_t if the launch failed.  B == 0 is a successful no-op.
 *   precision  fp32 storage and arithmetic, exp on the SFU.  No CPU fallback.
 */
#ifndef BIRKHOFF_OT_H
#define BIRKHOFF_OT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BIRKHOFF_OT_OK 0
#define BIRKHOFF_OT_EINVAL 1
#define BIRKHOFF_OT_ECUDA_BASE 1000

typedef struct CUstream_st* birkhoff_ot_stream_t; /* identical to cudaStream_t */

/*
 * n = 8 Birkhoff projection P = proj^KL_{B_8}(exp(H)) (eq. (1) PAPER.md:72 at n = 8).  H, P: fp32 [B][8][8].
 * iters (int32 [B], updates taken) and n_unconverged (uint64 [1], accumulated) are nullable diagnostics.
 */
int birkhoff8_forward(const float* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                      unsigned long long* n_unconverged, birkhoff_ot_stream_t stream);

/* dH = dL/dH from P and dP = dL/dP, fp32 [B][8][8] (eq. (13) with a = b = 1, eta = 1; dL/dH = -D) */
int birkhoff8_backward(const float* P, const float* dP, float* dH, int64_t B, birkhoff_ot_stream_t stream);

/* General small entropic OT, forward: costs C [B][n][m], marginals a [B][n], b [B][m] (or both NULL), T [B][n][m]. */
int entropic_ot_forward(const float* C, const float* a, const float* b, float* T, int64_t B, int n, int m, float eta,
                        float tol, int max_iter, int32_t* iters, unsigned long long* n_unconverged,
                        birkhoff_ot_stream_t stream);

/* General small entropic OT, backward: D = dl/dC [B][n][m] from T and G = dl/dT; the row marginals are read off T. */
int entropic_ot_backward(const float* T, const float* G, float* D, int64_t B, int n, int m, float eta,
                         birkhoff_ot_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* BIRKHOFF_OT_H */
