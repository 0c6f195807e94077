// birkhoff4.cu -- kernels and C ABI of libbirkhoff4.so (include/birkhoff4.h).  sm_100a only.
//
// Mapping: one thread owns one matrix.  A 64-byte matrix is two 32-byte DRAM sectors, so each thread moves its
// matrix with 256-bit LDG/STG (bk4_math.cuh).  All intermediates live in registers; the forward
// kernel's shared memory is a per-thread scratch column for the column permutation of the wide start.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include <mutex>

#include "../../include/birkhoff4.h"
#include "bk4_mix.cuh"
#include "bk4_project.cuh"

namespace bk4 {

constexpr int kThreads = BK4_THREADS;  // forward kernels
constexpr int kThreadsBwd = 256;       // backward and Sinkhorn kernels
static_assert(kThreads == kSmStride, "the scratch column stride is the block size");

#ifdef BK4_EXPERIMENTS
static float lp_range_exp() { const char* e = getenv("BK4_LPRANGE"); return e ? (float)atof(e) : kLpRange; }
#endif

struct FwdDiag {
    int32_t* iters;
    unsigned long long* hist;
    unsigned long long* n_unconverged;
};

// ---------------------------------------------------------------- launch with programmatic dependent launch
template <class... KArgs, class... Args>
static cudaError_t launch(void (*kernel)(KArgs...), unsigned grid, unsigned block, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---------------------------------------------------------------- forward kernel
// Every matrix first runs the lean iteration in warp lockstep (bk4_lean.cuh).  What that leaves (NaN/Inf, a residual that stopped falling above the fp32 floor) runs the
// guarded solver afterwards, in a branch a warp skips when it has none.  A matrix's result depends on that matrix
// alone, not on which matrices share its warp.
// GUARDED_ONLY (birkhoff4_forward_guarded): the lean part is skipped and every matrix takes the guarded solver.
// FUSED_BWD (birkhoff4_forward_backward): the backward pass runs on the result while it is still in
// registers: dH from P and dP = dL/dP; P itself is written only if the pointer is not null.
struct FusedBwd {
    const float* dP;
    float* dH;
};
template <bool BF16, bool DIAG, bool GUARDED_ONLY = false, bool FUSED_BWD = false>
__global__ void __launch_bounds__(kThreads, 1024 / kThreads) forward_kernel(const void* __restrict__ H, float* __restrict__ P, int64_t B,
                                                              float tol_i, int max_iter, float lp_range, FwdDiag diag,
                                                              FusedBwd bwd) {
    pdl_wait_and_trigger();
    __shared__ float s_col[16 * kThreads];
    __shared__ unsigned int s_hist[DIAG ? BIRKHOFF4_HIST_BINS : 1];
    __shared__ unsigned int s_unc;
    if constexpr (DIAG) {
        if (threadIdx.x < BIRKHOFF4_HIST_BINS) s_hist[threadIdx.x] = 0;
        if (threadIdx.x == 0) s_unc = 0;
        __syncthreads();
    }
    float* const sm = s_col + threadIdx.x;
    const int64_t b = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    const bool valid = b < B;
    const int64_t idx = valid ? b : B - 1;  // padding lanes shadow the last matrix and store nothing
    auto record = [&](int iters, bool converged) {
        if constexpr (DIAG) {
            if (diag.iters) diag.iters[idx] = iters;
            atomicAdd(&s_hist[min(iters, BIRKHOFF4_HIST_BINS - 1)], 1u);
            if (!converged) atomicAdd(&s_unc, 1u);
        }
    };
    // the result of this thread's matrix (original column order): store it and, when fused, differentiate it
    auto commit = [&](const float(&out)[16]) {
        // (the matrix index is formed again from the special registers: kept from the top of the kernel it is the one
        // value that does not fit 64 registers, and its spill costs every thread 8 bytes of L2 write traffic)
        unsigned cta, tid;
        asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(cta));
        asm volatile("mov.u32 %0, %%tid.x;" : "=r"(tid));
        const int64_t b2 = (int64_t)cta * kThreads + tid;
        const int64_t idx = b2 < B ? b2 : B - 1;
        if (!FUSED_BWD || P) store_matrix(P + 16 * idx, out);
        if constexpr (FUSED_BWD) {
            float g[16], d[16];
            load_matrix(bwd.dP + 16 * idx, g);  // dH may alias dP: coherent load
            backward_ift(out, g, d);
            store_matrix(bwd.dH + 16 * idx, d);
        }
    };
    auto load = [&](float(&h)[16]) { load_logits<BF16>(H, idx, h); };
    project_one<GUARDED_ONLY>(load, valid, sm, tol_i, max_iter, lp_range, commit, record);
    if constexpr (DIAG) {
        __syncthreads();
        if (diag.hist && threadIdx.x < BIRKHOFF4_HIST_BINS && s_hist[threadIdx.x])
            atomicAdd(&diag.hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
        if (diag.n_unconverged && threadIdx.x == 0 && s_unc) atomicAdd(diag.n_unconverged, (unsigned long long)s_unc);
    }
}

// ---------------------------------------------------------------- fused consumer: projection + residual-stream mix
template <bool XBF16>
__global__ void __launch_bounds__(kThreads, 512 / kThreads) forward_mix_kernel(
    const float* __restrict__ H, const typename MixVec<XBF16>::elem* __restrict__ X, typename MixVec<XBF16>::elem* __restrict__ Y,
    float* __restrict__ P, int64_t B, int C, float tol_i, int max_iter, float lp_range) {
    pdl_wait_and_trigger();
    __shared__ float s_col[16 * kThreads];
    float* const sm = s_col + threadIdx.x;
    const int64_t tok0 = (int64_t)blockIdx.x * kMixTokens;
    const int64_t b = tok0 + threadIdx.x;
    const bool valid = b < B;
    const int64_t idx = valid ? b : B - 1;
    // phase 1: thread t projects token t; the result stays in the thread's shared-memory column
    auto load = [&](float(&h)[16]) { load_matrix(H + 16 * idx, h); };
    auto commit = [&](const float(&out)[16]) {
        if (P) store_matrix(P + 16 * idx, out);
#pragma unroll
        for (int q = 0; q < 16; ++q) sm[q * kSmStride] = out[q];
    };
    auto record = [](int, bool) {};
    project_one<false>(load, valid, sm, tol_i, max_iter, lp_range, commit, record);
    __syncthreads();
    // phase 2: the block streams its tokens' 4 x C activations
    const int ntok = (int)((B - tok0 < kMixTokens) ? B - tok0 : kMixTokens);
    for (int t = 0; t < ntok; t += kMixGroup)
        mix_tokens<XBF16>(s_col, t, ntok - t, X + (size_t)(tok0 + t) * 4 * C, Y + (size_t)(tok0 + t) * 4 * C, C);
}

// ---------------------------------------------------------------- backward of the fused consumer
// One block = kMixTokens tokens, as in forward_mix_kernel.  Phase 1: thread t projects token t's logits again
// (recompute-style: the backward needs nothing of the forward but its result) and leaves P_t in its
// shared-memory column.  Phase 2: each of the block's warps takes every fourth token and streams its x and dy once:
// dx = P^T dy goes out as it is formed, G = dy x^T = dL/dP is summed over the warp and left in shared memory.
// Phase 3: thread t turns (P_t, G_t) into dL/dH_t by the implicit-function-theorem formula, the same
// backward_ift as birkhoff4_backward.  Neither P nor G ever goes through HBM.
template <bool XBF16>
__global__ void __launch_bounds__(kThreads, 512 / kThreads) backward_mix_kernel(
    const float* __restrict__ H, const typename MixVec<XBF16>::elem* __restrict__ X, const typename MixVec<XBF16>::elem* __restrict__ dY,
    typename MixVec<XBF16>::elem* __restrict__ dX, float* __restrict__ dH, float* __restrict__ P, int64_t B, int C, float tol_i,
    int max_iter, float lp_range) {
    pdl_wait_and_trigger();
    __shared__ float s_col[16 * kThreads];
    __shared__ float s_G[17 * kThreads];  // token t's entry q at [17 t + q]: conflict-free for the warp that writes it and for phase 3
    float* const sm = s_col + threadIdx.x;
    const int64_t tok0 = (int64_t)blockIdx.x * kMixTokens;
    const int64_t b = tok0 + threadIdx.x;
    const bool valid = b < B;
    const int64_t idx = valid ? b : B - 1;
    auto load = [&](float(&h)[16]) { load_matrix(H + 16 * idx, h); };
    auto commit = [&](const float(&out)[16]) {
        if (P) store_matrix(P + 16 * idx, out);
#pragma unroll
        for (int q = 0; q < 16; ++q) sm[q * kSmStride] = out[q];
    };
    auto record = [](int, bool) {};
    project_one<false>(load, valid, sm, tol_i, max_iter, lp_range, commit, record);
    __syncthreads();
    const int ntok = (int)((B - tok0 < kMixTokens) ? B - tok0 : kMixTokens);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int t = warp; t < ntok; t += kThreads / 32) {
        float G[16];
        const size_t off = (size_t)(tok0 + t) * 4 * C;
        mix_backward_token<XBF16>(s_col, t, X + off, dY + off, dX + off, C, G);
        const float total = mix_reduce16(G);
        if (!(lane & 1)) s_G[17 * t + mix_entry_of_lane(lane)] = total;
    }
    __syncthreads();
    if (valid) {
        float p[16], g[16], d[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            p[q] = sm[q * kSmStride];
            g[q] = s_G[17 * threadIdx.x + q];
        }
        backward_ift(p, g, d);
        store_matrix(dH + 16 * idx, d);
    }
}

// ---------------------------------------------------------------- backward kernel (HBM-bound: 192 B per matrix)
__global__ void __launch_bounds__(kThreadsBwd) backward_kernel(const float* __restrict__ P, const float* __restrict__ dP,
                                                            float* __restrict__ dH, int64_t B) {
    pdl_wait_and_trigger();
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    float p[16], g[16], d[16];
    load_matrix_nc(P + 16 * b, p);
    load_matrix(dP + 16 * b, g);  // dH may alias dP: coherent load
    backward_ift(p, g, d);
    store_matrix(dH + 16 * b, d);
}

// ---------------------------------------------------------------- Sinkhorn-Knopp baseline kernel
__global__ void __launch_bounds__(kThreadsBwd) sinkhorn_kernel(const float* __restrict__ H, float* __restrict__ P, int64_t B,
                                                            int n_iter) {
    pdl_wait_and_trigger();
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    float h[16], t[16];
    load_matrix(H + 16 * b, h);
    sinkhorn_knopp(h, n_iter, t);
    store_matrix(P + 16 * b, t);
}

// ---------------------------------------------------------------- host side
static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) != 0; }
static inline int cuda_rc(cudaError_t e) { return e == cudaSuccess ? BIRKHOFF4_OK : BIRKHOFF4_ECUDA_BASE + (int)e; }
static inline unsigned grid_for(int64_t B, int threads) { return (unsigned)((B + threads - 1) / threads); }

// The kernels test the column residual err = sum_m |g_m| computed in fp32 (rows sum to 1 by construction).  Err of
// PAPER.md:323, evaluated exactly on the stored fp32 P, adds to it the rounding of the stored entries (up to half an
// ulp of 1 in each of the 4 + 4 sums when P is close to a permutation) and the rounding of g itself: DESIGN.md S3/S9
// budgets these at 0.5 tol for tol = 1e-6, so the tested threshold is 0.5 tol, or tol - 7e-7 if that is larger.
static inline float internal_tol(float tol) {
    float f = 0.5f;
#ifdef BK4_EXPERIMENTS
    if (const char* e = getenv("BK4_TOLF")) f = (float)atof(e);
#endif
    return fmaxf(f * tol, tol - 7e-7f);
}

template <bool BF16, bool GUARDED_ONLY = false, bool FUSED_BWD = false>
static int launch_forward(const void* H, float* P, int64_t B, float tol, int max_iter, FwdDiag diag,
                          cudaStream_t stream, FusedBwd bwd = FusedBwd{nullptr, nullptr}) {
    if (B < 0 || !(tol >= 0.0f) || max_iter < 0) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!H || misaligned(H) || misaligned(P) || (!P && !FUSED_BWD)) return BIRKHOFF4_EINVAL;
    if (FUSED_BWD && (!bwd.dP || !bwd.dH || misaligned(bwd.dP) || misaligned(bwd.dH))) return BIRKHOFF4_EINVAL;
    const bool want_diag = diag.iters || diag.hist || diag.n_unconverged;
    const float tol_i = internal_tol(tol);
    cudaError_t rc;
#ifdef BK4_EXPERIMENTS
    const float lpr = lp_range_exp();
#else
    const float lpr = kLpRange;
#endif
    if (want_diag)
        rc = launch(forward_kernel<BF16, true, GUARDED_ONLY, FUSED_BWD>, grid_for(B, kThreads), kThreads, stream, H, P, B, tol_i,
                    max_iter, lpr, diag, bwd);
    else
        rc = launch(forward_kernel<BF16, false, GUARDED_ONLY, FUSED_BWD>, grid_for(B, kThreads), kThreads, stream, H, P, B, tol_i,
                    max_iter, lpr, diag, bwd);
    return cuda_rc(rc);
}

// ---- host-buffer path: a ring of device buffers and streams; chunked H2D -> kernels -> D2H
struct HostRing {
    static constexpr int kSlots = 3;
    static constexpr int64_t kChunk = 1 << 17;  // matrices per chunk (8 MiB per fp32 tensor; 2^16 / 2^17 / 2^18 measured: DESIGN.md)
    bool ready = false;
    int device = -1;
    cudaStream_t stream[kSlots] = {};
    float* buf[kSlots][4] = {};  // H, dP, P, dH
    std::mutex mu;

    void teardown() {
        for (int s = 0; s < kSlots; ++s) {
            if (stream[s]) cudaStreamSynchronize(stream[s]);
            for (int k = 0; k < 4; ++k) {
                if (buf[s][k]) cudaFree(buf[s][k]);
                buf[s][k] = nullptr;
            }
            if (stream[s]) cudaStreamDestroy(stream[s]);
            stream[s] = nullptr;
        }
        ready = false;
        device = -1;
    }
    // the ring lives on the device that is current at its first use; a call under another current device rebuilds it
    int init() {
        int dev = -1;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return cuda_rc(e);
        if (ready && dev == device) return BIRKHOFF4_OK;
        if (ready) teardown();
        for (int s = 0; s < kSlots && e == cudaSuccess; ++s) {
            e = cudaStreamCreateWithFlags(&stream[s], cudaStreamNonBlocking);
            for (int k = 0; k < 4 && e == cudaSuccess; ++k) e = cudaMalloc(&buf[s][k], kChunk * 64);
        }
        if (e != cudaSuccess) {
            teardown();  // nothing half-built is left behind
            return cuda_rc(e);
        }
        ready = true;
        device = dev;
        return BIRKHOFF4_OK;
    }
    void drain() {
        for (int s = 0; s < kSlots; ++s)
            if (stream[s]) cudaStreamSynchronize(stream[s]);
    }
};
static HostRing g_ring;

// mode bit 0: forward, bit 1: backward
static int run_host(const float* H_host, const float* P_in_host, const float* dP_host, float* P_host, float* dH_host,
                    int64_t B, float tol, int max_iter, int mode) {
    if (B < 0) return BIRKHOFF4_EINVAL;
    if ((mode & 1) && (!(tol >= 0.0f) || max_iter < 0)) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if ((mode & 1) && !H_host) return BIRKHOFF4_EINVAL;
    if ((mode & 2) && (!dP_host || !dH_host)) return BIRKHOFF4_EINVAL;
    if (mode == 1 && !P_host) return BIRKHOFF4_EINVAL;
    if (mode == 2 && !P_in_host) return BIRKHOFF4_EINVAL;
    std::lock_guard<std::mutex> lock(g_ring.mu);
    int rc = g_ring.init();
    if (rc) return rc;
    int slot = 0;
    for (int64_t off = 0; off < B && rc == BIRKHOFF4_OK; off += HostRing::kChunk, slot = (slot + 1) % HostRing::kSlots) {
        const int64_t n = (B - off < HostRing::kChunk) ? B - off : HostRing::kChunk;
        const size_t bytes = (size_t)n * 64;
        cudaStream_t st = g_ring.stream[slot];
        float *dHm = g_ring.buf[slot][0], *dG = g_ring.buf[slot][1], *dPm = g_ring.buf[slot][2],
              *dD = g_ring.buf[slot][3];
        if (mode == 3) {
            // forward + backward: both inputs up, the fused kernel (P stays in registers between the two halves), both results down
            rc = cuda_rc(cudaMemcpyAsync(dHm, H_host + 16 * off, bytes, cudaMemcpyHostToDevice, st));
            if (!rc) rc = cuda_rc(cudaMemcpyAsync(dG, dP_host + 16 * off, bytes, cudaMemcpyHostToDevice, st));
            if (!rc)
                rc = launch_forward<false, false, true>(dHm, P_host ? dPm : nullptr, n, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, st,
                                                        FusedBwd{dG, dD});
            if (!rc && P_host) rc = cuda_rc(cudaMemcpyAsync(P_host + 16 * off, dPm, bytes, cudaMemcpyDeviceToHost, st));
            if (!rc) rc = cuda_rc(cudaMemcpyAsync(dH_host + 16 * off, dD, bytes, cudaMemcpyDeviceToHost, st));
            continue;
        }
        if (mode & 1) {
            rc = cuda_rc(cudaMemcpyAsync(dHm, H_host + 16 * off, bytes, cudaMemcpyHostToDevice, st));
            if (!rc) rc = launch_forward<false>(dHm, dPm, n, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, st);
            if (!rc && P_host) rc = cuda_rc(cudaMemcpyAsync(P_host + 16 * off, dPm, bytes, cudaMemcpyDeviceToHost, st));
        } else {
            rc = cuda_rc(cudaMemcpyAsync(dPm, P_in_host + 16 * off, bytes, cudaMemcpyHostToDevice, st));
            if (!rc) rc = cuda_rc(cudaMemcpyAsync(dG, dP_host + 16 * off, bytes, cudaMemcpyHostToDevice, st));
            if (!rc) rc = birkhoff4_backward(dPm, dG, dD, n, st);
            if (!rc) rc = cuda_rc(cudaMemcpyAsync(dH_host + 16 * off, dD, bytes, cudaMemcpyDeviceToHost, st));
        }
    }
    // also on an error: no copy into the caller's buffers is in flight when the call returns
    for (int s = 0; s < HostRing::kSlots; ++s) {
        const cudaError_t e = cudaStreamSynchronize(g_ring.stream[s]);
        if (e != cudaSuccess && rc == BIRKHOFF4_OK) rc = cuda_rc(e);
    }
    return rc;
}

template <bool XBF16>
static int launch_mix(const float* H, const void* X, void* Y, float* P, int64_t B, int C, float tol, int max_iter,
                      cudaStream_t stream) {
    using E = typename MixVec<XBF16>::elem;
    if (B < 0 || !(tol >= 0.0f) || max_iter < 0 || C < 1 || C % MixVec<XBF16>::kElems) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!H || !X || !Y || misaligned(H) || misaligned(P) || (reinterpret_cast<uintptr_t>(X) & 15u) ||
        (reinterpret_cast<uintptr_t>(Y) & 15u))
        return BIRKHOFF4_EINVAL;
    return cuda_rc(launch(forward_mix_kernel<XBF16>, grid_for(B, kMixTokens), kThreads, stream, H, (const E*)X, (E*)Y, P, B, C,
                          internal_tol(tol), max_iter, kLpRange));
}

// ---- host-buffer forward that allocates nothing (birkhoff4_forward_host_static)
// The device copy of the batch lives in this array instead of in buffers from cudaMalloc: 4 MiB that every GPU
// which loads the library holds until the process exits.  The logits are copied in, projected IN PLACE (P == H is
// an allowed alias of the forward kernel) and copied out, so one region serves as input and output.
// Nothing here has to start at zero: a call overwrites the first B matrices before the kernel reads them and the
// kernel touches no others, so what an earlier call left behind is never read.
static __device__ __align__(256) float g_static_stage[BIRKHOFF4_STATIC_MAX * 16];

// In host code `g_static_stage` is only a handle for the runtime, not an address a kernel can use.  The device
// address differs from GPU to GPU, so it is asked for once per device, with that device current, and kept.
struct StaticStage {
    static constexpr int kMaxDevices = 64;
    std::mutex mu;
    float* addr[kMaxDevices] = {};
};
static StaticStage g_static;

static int static_stage_address(float** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_rc(e);
    if (dev < 0 || dev >= StaticStage::kMaxDevices) return BIRKHOFF4_EINVAL;
    std::lock_guard<std::mutex> lock(g_static.mu);
    if (!g_static.addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_stage);  // first use on this device: may load the module (do it before any capture)
        if (e != cudaSuccess) return cuda_rc(e);
        if (!p || misaligned(p)) return BIRKHOFF4_EINVAL;
        g_static.addr[dev] = static_cast<float*>(p);
    }
    *out = g_static.addr[dev];
    return BIRKHOFF4_OK;
}

static int run_host_static(const float* H_host, float* P_host, int64_t B, float tol, int max_iter, cudaStream_t stream) {
    if (B < 0 || !(tol >= 0.0f) || max_iter < 0) return BIRKHOFF4_EINVAL;
    if (B > BIRKHOFF4_STATIC_MAX) return BIRKHOFF4_ETOOBIG;  // before anything touches the device
    if (B == 0) return BIRKHOFF4_OK;
    if (!H_host || !P_host) return BIRKHOFF4_EINVAL;
    float* stage = nullptr;
    int rc = static_stage_address(&stage);
    if (rc) return rc;
    const size_t bytes = (size_t)B * 64;
    rc = cuda_rc(cudaMemcpyAsync(stage, H_host, bytes, cudaMemcpyHostToDevice, stream));
    if (!rc) rc = launch_forward<false>(stage, stage, B, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, stream);
    if (!rc) rc = cuda_rc(cudaMemcpyAsync(P_host, stage, bytes, cudaMemcpyDeviceToHost, stream));
    // also on an error: nothing is still reading or writing the caller's buffers when the call returns
    const cudaError_t e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess && rc == BIRKHOFF4_OK) rc = cuda_rc(e);
    return rc;
}

template <bool XBF16>
static int launch_mix_backward(const float* H, const void* X, const void* dY, void* dX, float* dH, float* P, int64_t B, int C,
                               float tol, int max_iter, cudaStream_t stream) {
    using E = typename MixVec<XBF16>::elem;
    if (B < 0 || !(tol >= 0.0f) || max_iter < 0 || C < 1 || C % MixVec<XBF16>::kElems) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!H || !X || !dY || !dX || !dH || misaligned(H) || misaligned(dH) || misaligned(P) || (reinterpret_cast<uintptr_t>(X) & 15u) ||
        (reinterpret_cast<uintptr_t>(dY) & 15u) || (reinterpret_cast<uintptr_t>(dX) & 15u))
        return BIRKHOFF4_EINVAL;
    return cuda_rc(launch(backward_mix_kernel<XBF16>, grid_for(B, kMixTokens), kThreads, stream, H, (const E*)X, (const E*)dY, (E*)dX,
                          dH, P, B, C, internal_tol(tol), max_iter, kLpRange));
}

}  // namespace bk4

// =================================================================== C ABI
using namespace bk4;

extern "C" {

int birkhoff4_forward(const float* H, float* P, int64_t B, float tol, int max_iter, birkhoff4_stream_t stream) {
    return launch_forward<false>(H, P, B, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, (cudaStream_t)stream);
}

int birkhoff4_forward_ex(const float* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                         unsigned long long* hist, unsigned long long* n_unconverged, birkhoff4_stream_t stream) {
    return launch_forward<false>(H, P, B, tol, max_iter, FwdDiag{iters, hist, n_unconverged}, (cudaStream_t)stream);
}

int birkhoff4_forward_bf16(const uint16_t* H, float* P, int64_t B, float tol, int max_iter,
                           birkhoff4_stream_t stream) {
    return launch_forward<true>(H, P, B, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, (cudaStream_t)stream);
}

int birkhoff4_forward_bf16_ex(const uint16_t* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                              unsigned long long* hist, unsigned long long* n_unconverged, birkhoff4_stream_t stream) {
    return launch_forward<true>(H, P, B, tol, max_iter, FwdDiag{iters, hist, n_unconverged}, (cudaStream_t)stream);
}

int birkhoff4_forward_guarded(const float* H, float* P, int64_t B, float tol, int max_iter, int32_t* iters,
                              unsigned long long* hist, unsigned long long* n_unconverged, birkhoff4_stream_t stream) {
    return launch_forward<false, true>(H, P, B, tol, max_iter, FwdDiag{iters, hist, n_unconverged}, (cudaStream_t)stream);
}

int birkhoff4_forward_backward(const float* H, const float* dP, float* P, float* dH, int64_t B, float tol, int max_iter,
                               birkhoff4_stream_t stream) {
    return launch_forward<false, false, true>(H, P, B, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, (cudaStream_t)stream,
                                              FusedBwd{dP, dH});
}

int birkhoff4_forward_mix(const float* H, const float* X, float* Y, float* P, int64_t B, int C, float tol, int max_iter,
                          birkhoff4_stream_t stream) {
    return launch_mix<false>(H, X, Y, P, B, C, tol, max_iter, (cudaStream_t)stream);
}

int birkhoff4_forward_mix_bf16(const float* H, const uint16_t* X, uint16_t* Y, float* P, int64_t B, int C, float tol,
                               int max_iter, birkhoff4_stream_t stream) {
    return launch_mix<true>(H, X, Y, P, B, C, tol, max_iter, (cudaStream_t)stream);
}

int birkhoff4_backward_mix(const float* H, const float* X, const float* dY, float* dX, float* dH, float* P, int64_t B, int C,
                           float tol, int max_iter, birkhoff4_stream_t stream) {
    return launch_mix_backward<false>(H, X, dY, dX, dH, P, B, C, tol, max_iter, (cudaStream_t)stream);
}

int birkhoff4_backward_mix_bf16(const float* H, const uint16_t* X, const uint16_t* dY, uint16_t* dX, float* dH, float* P,
                                int64_t B, int C, float tol, int max_iter, birkhoff4_stream_t stream) {
    return launch_mix_backward<true>(H, X, dY, dX, dH, P, B, C, tol, max_iter, (cudaStream_t)stream);
}

int birkhoff4_backward(const float* P, const float* dP, float* dH, int64_t B, birkhoff4_stream_t stream) {
    if (B < 0) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!P || !dP || !dH || misaligned(P) || misaligned(dP) || misaligned(dH)) return BIRKHOFF4_EINVAL;
    return cuda_rc(launch(backward_kernel, grid_for(B, kThreadsBwd), kThreadsBwd, (cudaStream_t)stream, P, dP, dH, B));
}

int birkhoff4_sinkhorn(const float* H, float* P, int64_t B, int n_iter, birkhoff4_stream_t stream) {
    if (B < 0 || n_iter < 0) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!H || !P || misaligned(H) || misaligned(P)) return BIRKHOFF4_EINVAL;
    return cuda_rc(launch(sinkhorn_kernel, grid_for(B, kThreadsBwd), kThreadsBwd, (cudaStream_t)stream, H, P, B, n_iter));
}

int birkhoff4_forward_host(const float* H_host, float* P_host, int64_t B, float tol, int max_iter) {
    return run_host(H_host, nullptr, nullptr, P_host, nullptr, B, tol, max_iter, 1);
}

int birkhoff4_backward_host(const float* P_host, const float* dP_host, float* dH_host, int64_t B) {
    return run_host(nullptr, P_host, dP_host, nullptr, dH_host, B, 0.0f, 0, 2);
}

int birkhoff4_forward_backward_host(const float* H_host, const float* dP_host, float* P_host, float* dH_host,
                                    int64_t B, float tol, int max_iter) {
    return run_host(H_host, nullptr, dP_host, P_host, dH_host, B, tol, max_iter, 3);
}

int birkhoff4_forward_host_static(const float* H_host, float* P_host, int64_t B, float tol, int max_iter,
                                  birkhoff4_stream_t stream) {
    return run_host_static(H_host, P_host, B, tol, max_iter, (cudaStream_t)stream);
}

void birkhoff4_host_release(void) {
    std::lock_guard<std::mutex> lock(g_ring.mu);
    g_ring.teardown();
}

const char* birkhoff4_strerror(int code) {
    if (code == BIRKHOFF4_OK) return "success";
    if (code == BIRKHOFF4_EINVAL) return "invalid argument (null or misaligned pointer, negative size, bad tol/max_iter)";
    if (code == BIRKHOFF4_ETOOBIG)
        return "batch too large for birkhoff4_forward_host_static: at most BIRKHOFF4_STATIC_MAX (65536) matrices per call; "
               "split the batch or use birkhoff4_forward_host";
    if (code >= BIRKHOFF4_ECUDA_BASE) return cudaGetErrorString((cudaError_t)(code - BIRKHOFF4_ECUDA_BASE));
    return "unknown error";
}

int birkhoff4_version(void) { return 200; }

}  // extern "C"
