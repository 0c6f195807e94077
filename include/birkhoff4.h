/*
 * birkhoff4.h -- C ABI of libbirkhoff4.so: batched 4x4 Birkhoff (KL / entropic-OT) projection on one B200.
 *
 * Source of every operation: arXiv 2606.07574 ("PAPER.md" = /root/reference/PAPER.md at build time).
 *
 *   forward   P = proj^KL_{B_4}(exp(H)) = diag(u) exp(H) diag(v), unit row and column sums
 *             (eq. (1); Sinkhorn's theorem PAPER.md:62), found by Newton's method on the
 *             gauge-fixed 3-variable dual f(beta_1..3) (eq. (8)) with the closed-form
 *             gradient and 3x3 Hessian (eq. (9)-(11) PAPER.md:144-221), a guarded step
 *             and a stop on marginal error.
 *   backward  dL/dH from P and dL/dP by the implicit-function-theorem formula, no stored iterates
 *             (eq. (13), 4x4 case PAPER.md:284-304; dL/dH = -D).
 *   sinkhorn  K = exp(H), n_iter x (row-normalise, column-normalise): the Sinkhorn-20 baseline the
 *             paper compares against (eq. (2)).
 *
 * Conventions (all entry points)
 *   layout     [B][4][4] row-major contiguous: element (i,j) of matrix b at 16*b + 4*i + j.
 *              H is the paper's R = -M.
 *   pointers   DEVICE pointers unless the name ends in _host; owned by the caller.  The library never
 *              allocates or frees device memory in the device-pointer calls and never synchronises:
 *              every call is asynchronous on `stream` (a cudaStream_t; 0 = the legacy default stream).
 *   alignment  every matrix pointer must be 32-byte aligned (else BIRKHOFF4_EINVAL; there is no slow path): a
 *              thread moves its 64-byte matrix with two 256-bit loads or stores (ld/st.global.v8.f32), which
 *              need their address aligned to 32 bytes.  (SURVEY.md 8(b) proposed 16, the 128-bit rule.)
 *   aliasing   P == H and dH == dP are allowed as exact aliases; partial overlap is undefined.
 *   errors     return 0 on success; BIRKHOFF4_EINVAL for a null pointer with B > 0, B < 0, tol < 0 or NaN,
 *              max_iter < 0, n_iter < 0 or a misaligned pointer; BIRKHOFF4_ECUDA_BASE + cudaError_t if
 *              the launch failed.  B == 0 is a successful no-op.
 *   NaN/Inf    a matrix holding a NaN or Inf gives an all-NaN output for that matrix only; the loops
 *              are bounded by max_iter, so nothing hangs.
 *   precision  fp32 storage and arithmetic (exp on the SFU via ex2.approx); bf16 inputs are widened
 *              exactly to fp32.
 *
 * There is no CPU fallback: without a CUDA device every compute call returns an error.
 */
#ifndef BIRKHOFF4_H
#define BIRKHOFF4_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BIRKHOFF4_OK 0
#define BIRKHOFF4_EINVAL 1
#define BIRKHOFF4_ETOOBIG 2 /* birkhoff4_forward_host_static only: B > BIRKHOFF4_STATIC_MAX */
#define BIRKHOFF4_ECUDA_BASE 1000 /* return value = BIRKHOFF4_ECUDA_BASE + cudaError_t */

#define BIRKHOFF4_HIST_BINS 64
#define BIRKHOFF4_STATIC_MAX 65536 /* matrices per call of birkhoff4_forward_host_static (4 MiB of device memory) */

typedef struct CUstream_st* birkhoff4_stream_t; /* identical to cudaStream_t */

/*
 * Forward projection (section 3).  H, P: device, fp32 [B][4][4].
 *   tol       stop when the marginal error Err(T) = ||T1-1||_1 + ||T^T1-1||_1 of the
 *             current iterate is <= tol.  Rows of T are normalised by construction (eq. (10)), so the
 *             kernel tests the column part |g1|+|g2|+|g3|+|g4|, g = c - 1 (eq. (11)), in fp32
 *             against an internal threshold max(tol/2, tol - 7e-7) that leaves room for the fp32
 *             rounding of the stored entries (S3/S9).  tol = 0 runs to the fp32 floor.
 *   max_iter  maximum number of updates of beta per matrix (Newton steps, the one Sinkhorn column step
 *             a nearly converged well-scaled matrix may take instead, and the guarded solver's fallback
 *             column steps; PAPER.md:319 uses 20).  The start-up steps (three Sinkhorn sweeps
 *             for well-scaled logits, one balancing step after the LP start otherwise; S1) are
 *             not counted: function evaluations <= max_iter + 4 for a matrix the lean iteration finishes.  (One
 *             it hands to the guarded solver starts again there: the start-up evaluations are spent a second
 *             time and every rejected trial step costs one more, so only the update count is bounded for it.)
 *             The first updates are taken without
 *             testing the residual: min(2, max_iter) for a matrix that starts from beta = 0, 3 for one
 *             that takes the LP start (if max_iter >= 3), so a matrix reports at least that many; the
 *             count is a property of the matrix, not of the batch it is in (S2).
 *             A matrix that the lean iteration hands to the guarded solver (S2) is solved again
 *             with the updates that are left, and reports the sum.  max_iter = 0 is accepted (start
 *             point only, rows normalised).
 * A matrix that has not converged after max_iter updates gets its last iterate (rows still
 * normalised); this is not an error (Table 2 reports such iterates too).
 */
int birkhoff4_forward(const float* H, float* P, int64_t B, float tol, int max_iter, birkhoff4_stream_t stream);

/*
 * Forward with diagnostics.  Extra outputs, each nullable:
 *   iters          int32 [B]: updates of beta taken by each matrix (0..max_iter)
 *   hist           uint64 [BIRKHOFF4_HIST_BINS]: hist[k] += #matrices with min(iters, 63) == k
 *                  (accumulated with atomics: zero it before the call)
 *   n_unconverged  uint64 [1]: += #matrices that stopped on max_iter or at the fp32 floor with the
 *                  tested error still above the internal threshold
 */
int birkhoff4_forward_ex(const float* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                         unsigned long long* hist, unsigned long long* n_unconverged,
                         birkhoff4_stream_t stream);

/*
 * The guarded solver (residual-decrease guard with Sinkhorn fallback steps, S2) applied to EVERY
 * matrix instead of only to those the lean iteration leaves: the plain, slower statement of the method, exported
 * so that the default path can be validated against it.  Same arguments and diagnostics as birkhoff4_forward_ex.
 */
int birkhoff4_forward_guarded(const float* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                              unsigned long long* hist, unsigned long long* n_unconverged,
                              birkhoff4_stream_t stream);

/* Forward for logits stored as bf16 bit patterns (uint16 [B][4][4], 32 B per matrix); P is fp32. */
int birkhoff4_forward_bf16(const uint16_t* H, float* P, int64_t B, float tol, int max_iter,
                           birkhoff4_stream_t stream);
/* The same with the diagnostics of birkhoff4_forward_ex (each nullable). */
int birkhoff4_forward_bf16_ex(const uint16_t* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                              unsigned long long* hist, unsigned long long* n_unconverged,
                              birkhoff4_stream_t stream);

/*
 * Backward (section 4.2).  P: the forward output; dP = dL/dP; dH = dL/dH, all
 * device fp32 [B][4][4].  Gamma = dP o P, mu_r = Gamma 1, mu_c = Gamma^T 1, w_{1..3} from the 3x3
 * system Delta w = mu_c - P_{-4}^T mu_r (w_4 = 0), v = mu_r - P w, dH_ij = P_ij (dP_ij - v_i - w_j).
 * Delta is formed and solved as a grounded graph Laplacian by node elimination (S7), which
 * stays finite when P is (near) a permutation.
 */
int birkhoff4_backward(const float* P, const float* dP, float* dH, int64_t B, birkhoff4_stream_t stream);

/*
 * Fused forward + backward for recompute-style training (the backward needs nothing of the
 * forward but its result): one kernel projects H and differentiates the result while it is still in registers.
 * H, dP = dL/dP, dH = dL/dH: device fp32 [B][4][4]; P: device fp32 [B][4][4] or NULL (then the projection is never
 * written: 64 + 64 bytes in and 64 out per matrix instead of the 320 of the two separate calls).  Aliases allowed:
 * dH == dP, P == H.  P and dH are bit-identical to birkhoff4_forward followed by birkhoff4_backward.
 */
int birkhoff4_forward_backward(const float* H, const float* dP, float* P, float* dH, int64_t B, float tol, int max_iter,
                               birkhoff4_stream_t stream);

/*
 * Fused consumer: the residual-stream mix of PAPER.md:46-50 with its mixing matrix
 * projected in the same kernel,
 *     Y_b = P_b X_b,   P_b = proj^KL_{B_4}(exp(H_b)),   b = 0..B-1 (tokens),
 * X, Y: device [B][4][C] row-major (stream j of token b at (4 b + j) C), fp32 or bf16 bit patterns (fp32
 * accumulation, round-to-nearest-even on store); C a multiple of 4 (fp32) or 8 (bf16); X, Y 16-byte aligned; Y must
 * not alias X.  P: device fp32 [B][4][4] or NULL: written only if given (the backward pass needs it).  P never
 * makes the round trip through HBM that birkhoff4_forward followed by a separate mix pays.
 */
int birkhoff4_forward_mix(const float* H, const float* X, float* Y, float* P, int64_t B, int C, float tol, int max_iter,
                          birkhoff4_stream_t stream);
int birkhoff4_forward_mix_bf16(const float* H, const uint16_t* X, uint16_t* Y, float* P, int64_t B, int C, float tol,
                               int max_iter, birkhoff4_stream_t stream);

/*
 * Backward of the fused consumer: everything the training step needs from the mix Y_b = P_b X_b in one
 * kernel, with P_b = proj^KL_{B_4}(exp(H_b)) projected again from the logits (recompute-style), so
 * that neither P nor dL/dP ever goes through HBM:
 *     dX_b = P_b^T dY_b,     G_b = dY_b X_b^T  (= dL/dP_b, a 4 x 4 matrix of C-long dot products, fp32 accumulation),
 *     dH_b = dL/dH_b from (P_b, G_b) by the formula of birkhoff4_backward.
 * H: device fp32 [B][4][4]; X, dY, dX: device [B][4][C] row-major, fp32 or bf16 bit patterns (round-to-nearest-even on
 * store), 16-byte aligned, C a multiple of 4 (fp32) or 8 (bf16); dX must not alias X or dY; dH: device fp32 [B][4][4]
 * (dH == H is allowed); P: device fp32 [B][4][4] or NULL, written only if given.  tol, max_iter as in birkhoff4_forward:
 * with the same values P equals birkhoff4_forward's bit for bit.  Errors as for birkhoff4_forward_mix.
 */
int birkhoff4_backward_mix(const float* H, const float* X, const float* dY, float* dX, float* dH, float* P, int64_t B, int C,
                           float tol, int max_iter, birkhoff4_stream_t stream);
int birkhoff4_backward_mix_bf16(const float* H, const uint16_t* X, const uint16_t* dY, uint16_t* dX, float* dH, float* P,
                                int64_t B, int C, float tol, int max_iter, birkhoff4_stream_t stream);

/*
 * Sinkhorn-Knopp baseline (eq. (2)): K = exp(H) (row-max shifted, which the first row
 * normalisation cancels), then n_iter x (rows /= row sums; columns /= column sums).  n_iter = 20 is the
 * "Sinkhorn-20" of PAPER.md:32, 319.  Reported baseline only.
 */
int birkhoff4_sinkhorn(const float* H, float* P, int64_t B, int n_iter, birkhoff4_stream_t stream);

/*
 * Host-buffer convenience calls (end-to-end path): H_host/dP_host/P_host/dH_host are HOST pointers
 * (pinned memory recommended; pageable works but copies then serialise).  The batch is cut into
 * chunks that are copied to the device, processed and copied back on a small ring of internal
 * streams and device buffers (allocated on first use, released by birkhoff4_host_release()).
 * These calls are synchronous: they return when the outputs are in host memory.
 *   birkhoff4_forward_host           H_host -> P_host
 *   birkhoff4_backward_host          P_host, dP_host -> dH_host
 *   birkhoff4_forward_backward_host  H_host, dP_host -> P_host (nullable), dH_host
 *                                    (one fused kernel per chunk: P goes from the projection to its
 *                                    derivative in registers)
 * The ring belongs to the device that is current when it is first used (a call under another current
 * device rebuilds it); calls are serialised by a mutex.  On an error the call still waits for every copy
 * it has started, so no transfer into the caller's buffers is in flight when it returns.
 */
int birkhoff4_forward_host(const float* H_host, float* P_host, int64_t B, float tol, int max_iter);
int birkhoff4_backward_host(const float* P_host, const float* dP_host, float* dH_host, int64_t B);
int birkhoff4_forward_backward_host(const float* H_host, const float* dP_host, float* P_host, float* dH_host,
                                    int64_t B, float tol, int max_iter);
void birkhoff4_host_release(void);

/*
 * birkhoff4_forward_host for callers that must not allocate device memory: H_host -> P_host, the same forward
 * kernel and the same results as birkhoff4_forward / birkhoff4_forward_host, but no cudaMalloc, cudaFree, stream
 * creation or other allocating call is ever made, on the first call or on a later one.
 *
 * Who needs it.  birkhoff4_forward_host keeps its device copy of the batch in buffers it gets from cudaMalloc on
 * first use.  That is unusable when the process has already handed all of the GPU's memory to a pool of its own
 * (a serving engine that sizes its KV cache to what is free, a training job whose caching allocator has grown to
 * the card): cudaMalloc then fails although the job itself is far from full.  It is also unusable where a
 * device-wide stall is not acceptable (cudaMalloc and cudaFree may synchronise the whole device), and in a process
 * where another thread is recording a CUDA graph in the default (global) capture mode, during which cudaMalloc
 * from any thread is an error.
 *
 * How.  The device copy lives in a fixed array inside the library: BIRKHOFF4_STATIC_MAX matrices, 4 MiB, which
 * every GPU that loads libbirkhoff4.so holds from the moment the library's code is loaded on it until the process
 * exits, whether or not this call is ever made.  The logits are copied into it, projected in place and copied
 * out, all on `stream` (the caller's; 0 = the legacy default stream), and the call returns after waiting for
 * `stream`, when P_host holds the result.  P_host == H_host is allowed.  Pinned host memory is recommended;
 * pageable memory works.
 *
 *   B > BIRKHOFF4_STATIC_MAX   returns BIRKHOFF4_ETOOBIG (nothing is copied or launched; birkhoff4_strerror names
 *                              the limit).  Split the batch into several calls, or use birkhoff4_forward_host.
 *   first call on a device     looks up the array's address on the device that is current (once per device, under a
 *                              lock; the address is kept).  This may make the driver load the library's device
 *                              code, so make one call (B = 1 will do) on each device you will use before you begin
 *                              any stream capture there.
 *   one array per device       every call on a device uses the same array, from every thread and every stream.  The
 *                              library does NOT serialise them: two calls whose work overlaps on the GPU (two
 *                              host threads, hence two calls in flight at once) overwrite each other's matrices.
 *                              Issue the calls for one device from one thread, or put your own lock around them.
 *                              Each process has its own copy, so separate processes do not interfere.
 *   stale contents             the array keeps whatever the last call left in it.  No call depends on that: the
 *                              first B matrices are overwritten before the kernel reads them and no others are
 *                              touched, so nothing needs clearing between calls.
 * Other errors as for birkhoff4_forward (BIRKHOFF4_EINVAL for a null pointer with B > 0, B < 0, bad tol or
 * max_iter; BIRKHOFF4_ECUDA_BASE + cudaError_t for a failed copy or launch).  B == 0 is a successful no-op.
 */
int birkhoff4_forward_host_static(const float* H_host, float* P_host, int64_t B, float tol, int max_iter,
                                  birkhoff4_stream_t stream);

const char* birkhoff4_strerror(int code);
int birkhoff4_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BIRKHOFF4_H */
