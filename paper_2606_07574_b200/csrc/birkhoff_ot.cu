// birkhoff_ot.cu -- kernels and C ABI of the n = 8 Birkhoff projection and of small general entropic OT
// (include/birkhoff_ot.h).  Part of libbirkhoff4.so.  sm_100a only.
//
// One thread owns one problem; rows are streamed (bk_ot.cuh).  An 8 x 8 matrix is 256 bytes = eight 32-byte
// sectors, moved row by row with 256-bit LDG/STG.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/birkhoff_ot.h"
#include "bk_ot.cuh"

namespace bkot {

constexpr int kOtThreads = 128;

template <class... KArgs, class... Args>
static cudaError_t launch(void (*kernel)(KArgs...), unsigned grid, unsigned block, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// blocks per SM the forward is compiled for: 3 for 8 x 8 (168 registers instead of 198: 54.5 -> 46.3 us at N(0,1), bit-identical),
// 4 for the rectangular sizes (128 registers), the compiler's choice for 4 x 4 (0 = no bound)
template <int N, int M>
constexpr int kOtFwdBlocks = N * M > 32 ? 3 : N * M > 16 ? 4 : 0;
template <int N, int M, bool UNIT>
__global__ void __launch_bounds__(kOtThreads, kOtFwdBlocks<N, M>) ot_forward_kernel(const float* __restrict__ C, const float* __restrict__ a,
                                                                const float* __restrict__ b, float* __restrict__ T, int64_t B,
                                                                float sign, float eta, float tol_abs, int max_iter,
                                                                int32_t* iters, unsigned long long* n_unconverged) {
    pdl_wait_and_trigger();
    const int64_t q = (int64_t)blockIdx.x * kOtThreads + threadIdx.x;
    if (q >= B) return;
    float av[N], bv[M];
    if constexpr (!UNIT) {
#pragma unroll
        for (int i = 0; i < N; ++i) av[i] = a[q * N + i];
#pragma unroll
        for (int j = 0; j < M; ++j) bv[j] = b[q * M + j];
    }
    const OtStats st = ot_forward_one<N, M, UNIT>(C + q * (N * M), sign, eta, av, bv, tol_abs, max_iter, T + q * (N * M));
    if (iters) iters[q] = st.iters;
    if (n_unconverged && !st.converged) atomicAdd(n_unconverged, 1ull);
}

// An n x m problem with 2 <= n, m <= 8 other than the four sizes above, in the N x M tile that holds it (bk_ot.cuh, PAD).
// The marginals are read into the tile's slots (zeros on the padding; all ones on the real rows and columns when a, b
// are null).  Scalar loads and stores: these sizes are served for completeness, not tuned.
template <int N, int M>
__global__ void __launch_bounds__(kOtThreads) ot_forward_padded_kernel(
    const float* __restrict__ C, const float* __restrict__ a, const float* __restrict__ b, float* __restrict__ T, int64_t B, OtShape sh,
    float sign, float eta, float tol_abs, int max_iter, int32_t* iters, unsigned long long* n_unconverged) {
    pdl_wait_and_trigger();
    const int64_t q = (int64_t)blockIdx.x * kOtThreads + threadIdx.x;
    if (q >= B) return;
    float av[N], bv[M];
#pragma unroll
    for (int i = 0; i < N; ++i) av[i] = i < sh.n ? (a ? a[q * sh.n + i] : 1.0f) : 0.0f;
#pragma unroll
    for (int j = 0; j < M; ++j) bv[j] = pad_slot<M>(sh, j) ? 0.0f : (b ? b[q * sh.m + slot_column<M>(sh, j)] : 1.0f);
    const OtStats st = ot_forward_one<N, M, false, true>(C + q * (sh.n * sh.m), sign, eta, av, bv, tol_abs, max_iter,
                                                         T + q * (sh.n * sh.m), sh);
    if (iters) iters[q] = st.iters;
    if (n_unconverged && !st.converged) atomicAdd(n_unconverged, 1ull);
}

template <int N, int M>
__global__ void __launch_bounds__(kOtThreads) ot_backward_padded_kernel(const float* __restrict__ T, const float* __restrict__ G,
                                                                        float* __restrict__ D, int64_t B, OtShape sh, float out_scale) {
    pdl_wait_and_trigger();
    const int64_t q = (int64_t)blockIdx.x * kOtThreads + threadIdx.x;
    if (q >= B) return;
    const int64_t off = q * (sh.n * sh.m);
    ot_backward_one<N, M, true>(T + off, G + off, out_scale, D + off, sh);
}

// (the 8 x 8 backward keeps T, G and the edge weights in 214 registers, 2 blocks per SM: compiled for 3 it spills 392 bytes and
// takes 54 us instead of 43.6)
template <int N, int M>
__global__ void __launch_bounds__(kOtThreads) ot_backward_kernel(const float* __restrict__ T, const float* __restrict__ G,
                                                                 float* __restrict__ D, int64_t B, float out_scale) {
    pdl_wait_and_trigger();
    const int64_t q = (int64_t)blockIdx.x * kOtThreads + threadIdx.x;
    if (q >= B) return;
    ot_backward_one<N, M>(T + q * (N * M), G + q * (N * M), out_scale, D + q * (N * M));
}

static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) != 0; }
static inline bool misaligned4(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 3u) != 0; }  // scalar float access
static inline int cuda_rc(cudaError_t e) { return e == cudaSuccess ? BIRKHOFF_OT_OK : BIRKHOFF_OT_ECUDA_BASE + (int)e; }
static inline unsigned grid_for(int64_t B) { return (unsigned)((B + kOtThreads - 1) / kOtThreads); }

template <int N, int M>
static int launch_fwd(const float* C, const float* a, const float* b, float* T, int64_t B, float sign, float eta, float tol,
                      int max_iter, int32_t* iters, unsigned long long* unc, cudaStream_t st) {
    const float tol_abs = 0.5f * tol;  // the column part of Err_ab; the rows and the rounding of the result get the rest
    if (a)
        return cuda_rc(launch(ot_forward_kernel<N, M, false>, grid_for(B), kOtThreads, st, C, a, b, T, B, sign, eta, tol_abs,
                              max_iter, iters, unc));
    return cuda_rc(launch(ot_forward_kernel<N, M, true>, grid_for(B), kOtThreads, st, C, a, b, T, B, sign, eta, tol_abs,
                          max_iter, iters, unc));
}

static int forward_dispatch(const float* C, const float* a, const float* b, float* T, int64_t B, int n, int m, float sign,
                            float eta, float tol, int max_iter, int32_t* iters, unsigned long long* unc, cudaStream_t st) {
    if (B < 0 || !(tol >= 0.0f) || max_iter < 0 || !(eta > 0.0f) || !(eta < 3.0e38f)) return BIRKHOFF_OT_EINVAL;
    if ((a == nullptr) != (b == nullptr)) return BIRKHOFF_OT_EINVAL;
    if (!a && n != m) return BIRKHOFF_OT_EINVAL;  // unit marginals need a square problem (sum a = sum b)
    if (n < 2 || n > 8 || m < 2 || m > 8) return BIRKHOFF_OT_EINVAL;
    if (B == 0) return BIRKHOFF_OT_OK;
    const bool tile = (n == 4 || n == 8) && (m == 4 || m == 8);  // a size with a kernel of its own (256- or 128-bit accesses)
    if (!C || !T || (tile ? misaligned(C) || misaligned(T) : misaligned4(C) || misaligned4(T) || misaligned4(a) || misaligned4(b)))
        return BIRKHOFF_OT_EINVAL;
    if (!tile) {
        const OtShape sh{n, m};
        const float tol_abs = 0.5f * tol;
        if (n <= 4 && m <= 4)
            return cuda_rc(launch(ot_forward_padded_kernel<4, 4>, grid_for(B), kOtThreads, st, C, a, b, T, B, sh, sign, eta, tol_abs, max_iter, iters, unc));
        if (n <= 4)
            return cuda_rc(launch(ot_forward_padded_kernel<4, 8>, grid_for(B), kOtThreads, st, C, a, b, T, B, sh, sign, eta, tol_abs, max_iter, iters, unc));
        if (m <= 4)
            return cuda_rc(launch(ot_forward_padded_kernel<8, 4>, grid_for(B), kOtThreads, st, C, a, b, T, B, sh, sign, eta, tol_abs, max_iter, iters, unc));
        return cuda_rc(launch(ot_forward_padded_kernel<8, 8>, grid_for(B), kOtThreads, st, C, a, b, T, B, sh, sign, eta, tol_abs, max_iter, iters, unc));
    }
    if (n == 4 && m == 4) return launch_fwd<4, 4>(C, a, b, T, B, sign, eta, tol, max_iter, iters, unc, st);
    if (n == 8 && m == 8) return launch_fwd<8, 8>(C, a, b, T, B, sign, eta, tol, max_iter, iters, unc, st);
    if (n == 4 && m == 8) return launch_fwd<4, 8>(C, a, b, T, B, sign, eta, tol, max_iter, iters, unc, st);
    return launch_fwd<8, 4>(C, a, b, T, B, sign, eta, tol, max_iter, iters, unc, st);
}

static int backward_dispatch(const float* T, const float* G, float* D, int64_t B, int n, int m, float out_scale,
                             cudaStream_t st) {
    if (B < 0) return BIRKHOFF_OT_EINVAL;
    if (n < 2 || n > 8 || m < 2 || m > 8) return BIRKHOFF_OT_EINVAL;
    if (B == 0) return BIRKHOFF_OT_OK;
    const bool tile = (n == 4 || n == 8) && (m == 4 || m == 8);
    if (!T || !G || !D || (tile ? misaligned(T) || misaligned(G) || misaligned(D) : misaligned4(T) || misaligned4(G) || misaligned4(D)))
        return BIRKHOFF_OT_EINVAL;
    if (!tile) {
        const OtShape sh{n, m};
        if (n <= 4 && m <= 4) return cuda_rc(launch(ot_backward_padded_kernel<4, 4>, grid_for(B), kOtThreads, st, T, G, D, B, sh, out_scale));
        if (n <= 4) return cuda_rc(launch(ot_backward_padded_kernel<4, 8>, grid_for(B), kOtThreads, st, T, G, D, B, sh, out_scale));
        if (m <= 4) return cuda_rc(launch(ot_backward_padded_kernel<8, 4>, grid_for(B), kOtThreads, st, T, G, D, B, sh, out_scale));
        return cuda_rc(launch(ot_backward_padded_kernel<8, 8>, grid_for(B), kOtThreads, st, T, G, D, B, sh, out_scale));
    }
    if (n == 4 && m == 4) return cuda_rc(launch(ot_backward_kernel<4, 4>, grid_for(B), kOtThreads, st, T, G, D, B, out_scale));
    if (n == 8 && m == 8) return cuda_rc(launch(ot_backward_kernel<8, 8>, grid_for(B), kOtThreads, st, T, G, D, B, out_scale));
    if (n == 4 && m == 8) return cuda_rc(launch(ot_backward_kernel<4, 8>, grid_for(B), kOtThreads, st, T, G, D, B, out_scale));
    return cuda_rc(launch(ot_backward_kernel<8, 4>, grid_for(B), kOtThreads, st, T, G, D, B, out_scale));
}

}  // namespace bkot

using namespace bkot;

extern "C" {

int birkhoff8_forward(const float* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                      unsigned long long* n_unconverged, birkhoff_ot_stream_t stream) {
    return forward_dispatch(H, nullptr, nullptr, P, B, 8, 8, 1.0f, 1.0f, tol, max_iter, iters, n_unconverged,
                            (cudaStream_t)stream);
}

int birkhoff8_backward(const float* P, const float* dP, float* dH, int64_t B, birkhoff_ot_stream_t stream) {
    return backward_dispatch(P, dP, dH, B, 8, 8, -1.0f, (cudaStream_t)stream);
}

int entropic_ot_forward(const float* C, const float* a, const float* b, float* T, int64_t B, int n, int m, float eta,
                        float tol, int max_iter, int32_t* iters, unsigned long long* n_unconverged,
                        birkhoff_ot_stream_t stream) {
    return forward_dispatch(C, a, b, T, B, n, m, -1.0f, eta, tol, max_iter, iters, n_unconverged, (cudaStream_t)stream);
}

int entropic_ot_backward(const float* T, const float* G, float* D, int64_t B, int n, int m, float eta,
                         birkhoff_ot_stream_t stream) {
    if (!(eta > 0.0f) || !(eta < 3.0e38f)) return BIRKHOFF_OT_EINVAL;
    return backward_dispatch(T, G, D, B, n, m, 1.0f / eta, (cudaStream_t)stream);
}

}  // extern "C"
