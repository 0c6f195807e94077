// birkhoff4.cu -- kernels and C ABI of libbirkhoff4.so (include/birkhoff4.h).  sm_100a only.
//
// Mapping: one thread owns one matrix (two adjacent matrices in variant 2, where every FP32 instruction is a
// packed FFMA2/FADD2/FMUL2).  A 64-byte matrix is two 32-byte DRAM sectors, so each thread moves its matrix with
// 256-bit LDG/STG (ld.global.v8.f32, new on sm_100): every request touches whole sectors and nothing is fetched
// twice.  All intermediates live in registers.  Variants: include/birkhoff4.h.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include <mutex>

#include "../../include/birkhoff4.h"
#include "bk4_core.cuh"

namespace bk4 {

// ---------------------------------------------------------------- 256-bit global access
BK4_DEV void ldg256(const float* p, float (&a)[8]) {
    asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]), "=f"(a[4]), "=f"(a[5]), "=f"(a[6]), "=f"(a[7])
                 : "l"(p));
}
// plain (coherent) version: used when the output may alias the input (P == H) and for re-reads
BK4_DEV void ld256(const float* p, float (&a)[8]) {
    asm volatile("ld.global.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]), "=f"(a[4]), "=f"(a[5]), "=f"(a[6]), "=f"(a[7])
                 : "l"(p)
                 : "memory");
}
BK4_DEV void stg256(float* p, const float (&a)[8]) {
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(a[0]), "f"(a[1]), "f"(a[2]),
                 "f"(a[3]), "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7])
                 : "memory");
}
BK4_DEV void load_matrix(const float* p, float (&m)[16]) {
    float lo[8], hi[8];
    ld256(p, lo);
    ld256(p + 8, hi);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        m[k] = lo[k];
        m[8 + k] = hi[k];
    }
}
BK4_DEV void load_matrix_nc(const float* p, float (&m)[16]) {
    float lo[8], hi[8];
    ldg256(p, lo);
    ldg256(p + 8, hi);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        m[k] = lo[k];
        m[8 + k] = hi[k];
    }
}
// bf16 bit patterns, 32 B per matrix: widening is a 16-bit shift (exact)
BK4_DEV void load_matrix_bf16(const uint16_t* p, float (&m)[16]) {
    uint32_t w[8];
    asm volatile("ld.global.nc.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7])
                 : "l"(p));
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        m[2 * k] = __uint_as_float(w[k] << 16);
        m[2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
    }
}
BK4_DEV void store_matrix(float* p, const float (&m)[16]) {
    float lo[8], hi[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        lo[k] = m[k];
        hi[k] = m[8 + k];
    }
    stg256(p, lo);
    stg256(p + 8, hi);
}

template <bool BF16>
BK4_DEV void load_logits(const void* H, int64_t b, float (&m)[16]) {
    if constexpr (BF16) load_matrix_bf16(reinterpret_cast<const uint16_t*>(H) + 16 * b, m);
    else load_matrix(reinterpret_cast<const float*>(H) + 16 * b, m);
}

// logit range (max - min over the 16 entries) above which a matrix takes the LP dual start (S1):
// N(0,1) logits stay below it, N(0,2^2) and larger mostly exceed it.
constexpr float kHardRange = 8.0f;
// largest in-row logit range up to which lean_start starts from beta = 0 (above: LP dual start); chosen by
// measurement, DESIGN.md
constexpr float kEasyRange = 12.0f;

struct FwdDiag {
    int32_t* iters;
    unsigned long long* hist;
    unsigned long long* n_unconverged;
};

// ---------------------------------------------------------------- launch with programmatic dependent launch
// Every kernel of the library starts with pdl_wait() (griddepcontrol.wait: returns once the kernel before it in
// the stream has completed and its writes are visible) and then lets the kernel after it begin launching
// (griddepcontrol.launch_dependents).  Launched with programmatic stream serialization, the next kernel's launch
// latency and block ramp-up overlap this kernel's tail; stream-order semantics are unchanged because nothing is
// read or written before the wait.  BIRKHOFF4_NO_PDL=1 in the environment turns the attribute off (measurement).
BK4_DEV void pdl_wait_and_trigger() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

static bool use_pdl() {
    static int v = -1;
    if (v < 0) {
        const char* e = getenv("BIRKHOFF4_NO_PDL");
        v = (e && e[0] == '1') ? 0 : 1;
    }
    return v != 0;
}

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
    cfg.numAttrs = use_pdl() ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---------------------------------------------------------------- forward kernel
// NL = matrices per thread (1: scalar FP32, 2: packed FP32x2).
template <int NL, bool BF16, bool DIAG>
__global__ void __launch_bounds__(256) forward_kernel(const void* __restrict__ H, float* __restrict__ P, int64_t B,
                                                      float tol_i, int max_iter, FwdDiag diag) {
    using V = typename std::conditional<NL == 1, float, float2>::type;
    pdl_wait_and_trigger();
    __shared__ unsigned int s_hist[DIAG ? BIRKHOFF4_HIST_BINS : 1];
    __shared__ unsigned int s_unc;
    if constexpr (DIAG) {
        if (threadIdx.x < BIRKHOFF4_HIST_BINS) s_hist[threadIdx.x] = 0;
        if (threadIdx.x == 0) s_unc = 0;
        __syncthreads();
    }
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t b0 = t * NL;
    if (b0 < B) {
        int64_t idx[NL];
        bool valid[NL], bad[NL], hard[NL];
        float h[NL][16];
#pragma unroll
        for (int k = 0; k < NL; ++k) {
            valid[k] = b0 + k < B;
            idx[k] = valid[k] ? b0 + k : b0;  // an odd tail duplicates the last matrix in the idle half
            load_logits<BF16>(H, idx[k], h[k]);
            float hmax = h[k][0], hmin = h[k][0], poison = 0.0f;
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                hmax = fmaxf(hmax, h[k][q]);
                hmin = fminf(hmin, h[k][q]);
                poison = __fmaf_rn(h[k][q], 0.0f, poison);  // NaN iff some logit is NaN or +-Inf (fmaxf skips NaN)
            }
            bad[k] = !(poison == 0.0f);
            hard[k] = hmax - hmin > kHardRange;
        }
        // the LP dual start is compiled into a branch that a warp takes only if one of its matrices needs it
        bool any_hard = hard[0];
        if constexpr (NL == 2) any_hard = any_hard || hard[1];
        any_hard = __any_sync(__activemask(), any_hard);
        typename vtraits<V>::mask hardm;
        if constexpr (NL == 1) hardm = bool1(hard[0]);
        else hardm = bool2(hard[0], hard[1]);
        V Hv[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            if constexpr (NL == 1) Hv[q] = h[0][q];
            else Hv[q] = make_float2(h[0][q], h[1][q]);
        }
        auto reload = [&](V(&Hr)[16]) {
            float r[NL][16];
#pragma unroll
            for (int k = 0; k < NL; ++k) load_logits<BF16>(H, idx[k], r[k]);
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                if constexpr (NL == 1) Hr[q] = r[0][q];
                else Hr[q] = make_float2(r[0][q], r[1][q]);
            }
        };
        auto emit = [&](int k, const V(&T)[16], int iters, bool converged) {
            if (!valid[k]) return;
            float out[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) out[q] = bad[k] ? kNaN : vget(T[q], k);
            store_matrix(P + 16 * idx[k], out);
            if constexpr (DIAG) {
                if (diag.iters) diag.iters[idx[k]] = iters;
                atomicAdd(&s_hist[min(iters, BIRKHOFF4_HIST_BINS - 1)], 1u);
                if (!converged) atomicAdd(&s_unc, 1u);
            }
        };
        newton_forward<V>(Hv, hardm, any_hard, msplat(V{}, false), tol_i, max_iter, reload, emit);
    }
    if constexpr (DIAG) {
        __syncthreads();
        if (diag.hist && threadIdx.x < BIRKHOFF4_HIST_BINS && s_hist[threadIdx.x])
            atomicAdd(&diag.hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
        if (diag.n_unconverged && threadIdx.x == 0 && s_unc) atomicAdd(diag.n_unconverged, (unsigned long long)s_unc);
    }
}

// ---------------------------------------------------------------- forward kernel, variants 3 and 4 (default)
// One matrix per thread.  Every matrix first runs the lean iteration in warp lockstep (lean_start, lean_iterate:
// LP dual start when its largest in-row logit range exceeds lp_range) and the results are stored together.  What
// that leaves (NaN/Inf, a residual that stopped falling: none in a million N(0,1) matrices, about one in a thousand
// at N(0,30^2)) runs the guarded newton_forward afterwards, in a branch a warp skips when it has none.
// A matrix's result depends on that matrix alone, not on which matrices share its warp.
template <bool BF16, bool DIAG, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) forward_lean_kernel(const void* __restrict__ H, float* __restrict__ P,
                                                           int64_t B, float tol_i, int max_iter, float lp_range,
                                                           FwdDiag diag) {
    pdl_wait_and_trigger();
    __shared__ unsigned int s_hist[DIAG ? BIRKHOFF4_HIST_BINS : 1];
    __shared__ unsigned int s_unc;
    if constexpr (DIAG) {
        if (threadIdx.x < BIRKHOFF4_HIST_BINS) s_hist[threadIdx.x] = 0;
        if (threadIdx.x == 0) s_unc = 0;
        __syncthreads();
    }
    const int64_t b = (int64_t)blockIdx.x * THREADS + threadIdx.x;
    const bool valid = b < B;
    const int64_t idx = valid ? b : B - 1;  // padding lanes shadow the last matrix and store nothing
    auto finish = [&](const float(&T)[16], int iters, bool converged) {
        store_matrix(P + 16 * idx, T);
        if constexpr (DIAG) {
            if (diag.iters) diag.iters[idx] = iters;
            atomicAdd(&s_hist[min(iters, BIRKHOFF4_HIST_BINS - 1)], 1u);
            if (!converged) atomicAdd(&s_unc, 1u);
        }
    };
    bool left = valid;  // this thread's matrix still has to be solved
    {
        float h[16], T[16];
        load_logits<BF16>(H, idx, h);
        LeanState st;
        if (lean_start(h, valid, lp_range, max_iter, st)) lean_iterate(st, tol_i, max_iter, T);
        if (valid && st.status != kLeanFailed) {
            left = false;
            finish(T, st.it, st.status == kLeanConverged);
        }
    }
    if (__any_sync(0xffffffffu, left)) {
        float h[16];
        load_logits<BF16>(H, idx, h);  // the lean part has stored only matrices this branch does not touch
        float hmax = h[0], hmin = h[0], poison = 0.0f;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            hmax = fmaxf(hmax, h[q]);
            hmin = fminf(hmin, h[q]);
            poison = __fmaf_rn(h[q], 0.0f, poison);  // NaN iff some logit is NaN or +-Inf (fmaxf skips NaN)
        }
        const bool bad = !(poison == 0.0f);
        const bool hard = hmax - hmin > kHardRange;
        const bool any_hard = __any_sync(0xffffffffu, left && hard);
        auto reload = [&](float(&Hr)[16]) { load_logits<BF16>(H, idx, Hr); };
        auto emit = [&](int, const float(&T)[16], int iters, bool converged) {
            float out[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) out[q] = bad ? kNaN : T[q];
            finish(out, iters, converged);
        };
        newton_forward<float, true>(h, bool1(hard), any_hard, bool1(!left), tol_i, max_iter, reload, emit);
    }
    if constexpr (DIAG) {
        __syncthreads();
        if (diag.hist && threadIdx.x < BIRKHOFF4_HIST_BINS && s_hist[threadIdx.x])
            atomicAdd(&diag.hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
        if (diag.n_unconverged && threadIdx.x == 0 && s_unc) atomicAdd(diag.n_unconverged, (unsigned long long)s_unc);
    }
}

// ---------------------------------------------------------------- backward kernel (HBM-bound: 192 B per matrix)
__global__ void __launch_bounds__(256) backward_kernel(const float* __restrict__ P, const float* __restrict__ dP,
                                                       float* __restrict__ dH, int64_t B) {
    pdl_wait_and_trigger();
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    float p[16], g[16], d[16];
    load_matrix_nc(P + 16 * b, p);
    load_matrix(dP + 16 * b, g);  // dH may alias dP: coherent load
    backward_ift<float>(p, g, d);
    store_matrix(dH + 16 * b, d);
}

// ---------------------------------------------------------------- Sinkhorn-Knopp baseline kernel
__global__ void __launch_bounds__(256) sinkhorn_kernel(const float* __restrict__ H, float* __restrict__ P, int64_t B,
                                                       int n_iter) {
    pdl_wait_and_trigger();
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    float h[16], t[16];
    load_matrix(H + 16 * b, h);
    sinkhorn_knopp<float>(h, n_iter, t);
    store_matrix(P + 16 * b, t);
}

// ---------------------------------------------------------------- host side
static int g_variant = 0;
constexpr int kDefaultVariant = 4;
static float g_easy_range = -1.0f;  // < 0: kEasyRange, or BIRKHOFF4_EASY_RANGE from the environment (tuning only)

static float easy_range() {
    if (g_easy_range < 0.0f) {
        const char* e = getenv("BIRKHOFF4_EASY_RANGE");
        g_easy_range = e ? (float)atof(e) : kEasyRange;
    }
    return g_easy_range;
}
constexpr int kThreads = 256;

static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) != 0; }
static inline int cuda_rc(cudaError_t e) { return e == cudaSuccess ? BIRKHOFF4_OK : BIRKHOFF4_ECUDA_BASE + (int)e; }

static inline float internal_tol(float tol) {
    // Err(T) = column part (tested) + row part (fp32 rounding of four normalised rows, <~ 5e-7): DESIGN.md S3/S9
    const float t = fmaxf(0.5f * tol, tol - 5e-7f);
    return fminf(tol, t);
}

template <bool BF16>
static int launch_forward(const void* H, float* P, int64_t B, float tol, int max_iter, FwdDiag diag,
                          cudaStream_t stream) {
    if (B < 0 || !(tol >= 0.0f) || max_iter < 0) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!H || !P || misaligned(H) || misaligned(P)) return BIRKHOFF4_EINVAL;
    const bool want_diag = diag.iters || diag.hist || diag.n_unconverged;
    const int variant = g_variant ? g_variant : kDefaultVariant;
    const int nl = variant == 2 ? 2 : 1;
    const int64_t threads = (B + nl - 1) / nl;
    const unsigned grid = (unsigned)((threads + kThreads - 1) / kThreads);
    const float tol_i = internal_tol(tol);
    cudaError_t rc = cudaSuccess;
    if (variant >= 3) {
        const float em = easy_range();
#define BK4_LAUNCH_LEAN(T, M)                                                                                     \
    do {                                                                                                          \
        const unsigned g = (unsigned)((B + (T)-1) / (T));                                                         \
        if (want_diag) rc = launch(forward_lean_kernel<BF16, true, T, M>, g, T, stream, H, P, B, tol_i, max_iter, em, diag); \
        else rc = launch(forward_lean_kernel<BF16, false, T, M>, g, T, stream, H, P, B, tol_i, max_iter, em, diag);     \
    } while (0)
        if (variant == 3) BK4_LAUNCH_LEAN(256, 3);
        else BK4_LAUNCH_LEAN(256, 4);
#undef BK4_LAUNCH_LEAN
    } else if (nl == 1) {
        if (want_diag) rc = launch(forward_kernel<1, BF16, true>, grid, kThreads, stream, H, P, B, tol_i, max_iter, diag);
        else rc = launch(forward_kernel<1, BF16, false>, grid, kThreads, stream, H, P, B, tol_i, max_iter, diag);
    } else {
        if (want_diag) rc = launch(forward_kernel<2, BF16, true>, grid, kThreads, stream, H, P, B, tol_i, max_iter, diag);
        else rc = launch(forward_kernel<2, BF16, false>, grid, kThreads, stream, H, P, B, tol_i, max_iter, diag);
    }
    return cuda_rc(rc);
}

// ---- host-buffer path: a ring of device buffers and streams; chunked H2D -> kernels -> D2H
struct HostRing {
    static constexpr int kSlots = 3;
    static constexpr int64_t kChunk = 1 << 18;  // matrices per chunk (16 MiB per fp32 tensor)
    bool ready = false;
    cudaStream_t stream[kSlots];
    float* buf[kSlots][4];  // H, dP, P, dH
    std::mutex mu;

    int init() {
        if (ready) return BIRKHOFF4_OK;
        for (int s = 0; s < kSlots; ++s) {
            cudaError_t e = cudaStreamCreateWithFlags(&stream[s], cudaStreamNonBlocking);
            if (e != cudaSuccess) return cuda_rc(e);
            for (int k = 0; k < 4; ++k) {
                e = cudaMalloc(&buf[s][k], kChunk * 64);
                if (e != cudaSuccess) return cuda_rc(e);
            }
        }
        ready = true;
        return BIRKHOFF4_OK;
    }
    void release() {
        if (!ready) return;
        for (int s = 0; s < kSlots; ++s) {
            cudaStreamSynchronize(stream[s]);
            for (int k = 0; k < 4; ++k) cudaFree(buf[s][k]);
            cudaStreamDestroy(stream[s]);
        }
        ready = false;
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
    for (int64_t off = 0; off < B; off += HostRing::kChunk, slot = (slot + 1) % HostRing::kSlots) {
        const int64_t n = (B - off < HostRing::kChunk) ? B - off : HostRing::kChunk;
        const size_t bytes = (size_t)n * 64;
        cudaStream_t st = g_ring.stream[slot];
        float *dHm = g_ring.buf[slot][0], *dG = g_ring.buf[slot][1], *dPm = g_ring.buf[slot][2],
              *dD = g_ring.buf[slot][3];
        cudaError_t e;
        if (mode & 1) {
            if ((e = cudaMemcpyAsync(dHm, H_host + 16 * off, bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess)
                return cuda_rc(e);
            if ((rc = launch_forward<false>(dHm, dPm, n, tol, max_iter, FwdDiag{nullptr, nullptr, nullptr}, st))) return rc;
            if (P_host && (e = cudaMemcpyAsync(P_host + 16 * off, dPm, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
                return cuda_rc(e);
        } else {
            if ((e = cudaMemcpyAsync(dPm, P_in_host + 16 * off, bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess)
                return cuda_rc(e);
        }
        if (mode & 2) {
            if ((e = cudaMemcpyAsync(dG, dP_host + 16 * off, bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess)
                return cuda_rc(e);
            if ((rc = birkhoff4_backward(dPm, dG, dD, n, st))) return rc;
            if ((e = cudaMemcpyAsync(dH_host + 16 * off, dD, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
                return cuda_rc(e);
        }
    }
    for (int s = 0; s < HostRing::kSlots; ++s) {
        cudaError_t e = cudaStreamSynchronize(g_ring.stream[s]);
        if (e != cudaSuccess) return cuda_rc(e);
    }
    return BIRKHOFF4_OK;
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

int birkhoff4_backward(const float* P, const float* dP, float* dH, int64_t B, birkhoff4_stream_t stream) {
    if (B < 0) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!P || !dP || !dH || misaligned(P) || misaligned(dP) || misaligned(dH)) return BIRKHOFF4_EINVAL;
    const unsigned grid = (unsigned)((B + kThreads - 1) / kThreads);
    return cuda_rc(launch(backward_kernel, grid, kThreads, (cudaStream_t)stream, P, dP, dH, B));
}

int birkhoff4_sinkhorn(const float* H, float* P, int64_t B, int n_iter, birkhoff4_stream_t stream) {
    if (B < 0 || n_iter < 0) return BIRKHOFF4_EINVAL;
    if (B == 0) return BIRKHOFF4_OK;
    if (!H || !P || misaligned(H) || misaligned(P)) return BIRKHOFF4_EINVAL;
    const unsigned grid = (unsigned)((B + kThreads - 1) / kThreads);
    return cuda_rc(launch(sinkhorn_kernel, grid, kThreads, (cudaStream_t)stream, H, P, B, n_iter));
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

void birkhoff4_host_release(void) {
    std::lock_guard<std::mutex> lock(g_ring.mu);
    g_ring.release();
}

int birkhoff4_set_variant(int variant) {
    const int old = g_variant;
    if (variant >= 0 && variant <= 4) g_variant = variant;
    return old;
}

const char* birkhoff4_strerror(int code) {
    if (code == BIRKHOFF4_OK) return "success";
    if (code == BIRKHOFF4_EINVAL) return "invalid argument (null or misaligned pointer, negative size, bad tol/max_iter)";
    if (code >= BIRKHOFF4_ECUDA_BASE) return cudaGetErrorString((cudaError_t)(code - BIRKHOFF4_ECUDA_BASE));
    return "unknown error";
}

int birkhoff4_version(void) { return 100; }

}  // extern "C"
