// bk4_mix.cuh -- the fused consumer of the projection: the residual-stream mix
// x_{l+1} = H^res x_l of PAPER.md:46-50 with H^res = proj(exp(H)) computed in the same kernel, so that the
// doubly-stochastic matrix never makes the round trip through HBM that the separate calls pay (64 B written + 64 B
// re-read per token; the mix itself is bound by the 4 C elements of x_l in and out).
//
// One block = kMixTokens tokens.  Phase 1: thread t projects token t's matrix (project_one: the same code as
// birkhoff4_forward) and leaves P_t in its shared-memory column.  Phase 2: the block streams the tokens' 4 x C
// activations, kMixGroup tokens at a time: every thread reads P_t (a broadcast) and mixes a 16-byte slice of each of the
// four streams, with the loads of the whole group in flight together.
#pragma once
#include <cuda_bf16.h>

#include "bk4_project.cuh"

namespace bk4 {

constexpr int kMixTokens = BK4_THREADS;  // tokens per block = threads per block (one matrix per thread in phase 1)

template <bool XBF16>
struct MixVec;
template <>
struct MixVec<false> {  // fp32 activations: 4 elements per 16-byte access
    static constexpr int kElems = 4;
    using elem = float;
    using raw = float4;
    BK4_DEV static raw load_raw(const float* p) { return __ldcs(reinterpret_cast<const float4*>(p)); }
    BK4_DEV static void widen(const raw& t, float (&x)[4]) { x[0] = t.x, x[1] = t.y, x[2] = t.z, x[3] = t.w; }
    BK4_DEV static void load(const float* p, float (&x)[4]) {
        const float4 t = __ldcs(reinterpret_cast<const float4*>(p));
        x[0] = t.x, x[1] = t.y, x[2] = t.z, x[3] = t.w;
    }
    BK4_DEV static void store(float* p, const float (&y)[4]) {
        __stcs(reinterpret_cast<float4*>(p), make_float4(y[0], y[1], y[2], y[3]));
    }
};
template <>
struct MixVec<true> {  // bf16 activations (bit patterns): 8 elements per 16-byte access, fp32 accumulation
    static constexpr int kElems = 8;
    using elem = uint16_t;
    using raw = uint4;
    BK4_DEV static raw load_raw(const uint16_t* p) { return __ldcs(reinterpret_cast<const uint4*>(p)); }
    BK4_DEV static void widen(const raw& t, float (&x)[8]) {
        const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            x[2 * k] = __uint_as_float(w[k] << 16);
            x[2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
        }
    }
    BK4_DEV static void load(const uint16_t* p, float (&x)[8]) {
        const uint4 t = __ldcs(reinterpret_cast<const uint4*>(p));
        const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            x[2 * k] = __uint_as_float(w[k] << 16);
            x[2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
        }
    }
    BK4_DEV static void store(uint16_t* p, const float (&y)[8]) {
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(y[2 * k], y[2 * k + 1]);  // round to nearest even
            w[k] = *reinterpret_cast<const uint32_t*>(&h);
        }
        __stcs(reinterpret_cast<uint4*>(p), make_uint4(w[0], w[1], w[2], w[3]));
    }
};

// phase 2 for kMixGroup consecutive tokens (`n` of them exist): y_i = sum_j P_ij x_j over this thread's slices of the C
// columns.  All the group's loads (kMixGroup x 4 streams x 16 bytes per thread) are issued before the first is used:
// with four blocks of 128 threads per SM that is what keeps enough bytes in flight to fill HBM (one token at a time
// left 64 bytes per thread in flight and the kernel at 0.77 of the copy bandwidth; two: 0.92).  sP: the block's results, entry q
// of token t at [q * kSmStride + t] (read as a broadcast).
constexpr int kMixGroup = 2;  // measured: 1 / 2 / 3 / 4 tokens per group: 214 / 179 / 191 / 192 us (B = 2^16, C = 1024 bf16)
template <bool XBF16>
BK4_DEV void mix_tokens(const float* sP, int t0, int n, const typename MixVec<XBF16>::elem* x, typename MixVec<XBF16>::elem* y, int C) {
    using MV = MixVec<XBF16>;
    constexpr int V = MV::kElems;
    for (int c = threadIdx.x * V; c < C; c += kMixTokens * V) {
        typename MV::raw in[kMixGroup][4];
#pragma unroll
        for (int g = 0; g < kMixGroup; ++g)
            if (g < n) {
#pragma unroll
                for (int j = 0; j < 4; ++j) in[g][j] = MV::load_raw(x + ((size_t)g * 4 + j) * C + c);
            }
#pragma unroll
        for (int g = 0; g < kMixGroup; ++g)
            if (g < n) {
                float p[16], xin[4][V], yout[V];
#pragma unroll
                for (int q = 0; q < 16; ++q) p[q] = sP[q * kSmStride + t0 + g];
#pragma unroll
                for (int j = 0; j < 4; ++j) MV::widen(in[g][j], xin[j]);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
#pragma unroll
                    for (int e = 0; e < V; ++e)
                        yout[e] = fmaf(p[4 * i + 3], xin[3][e],
                                       fmaf(p[4 * i + 2], xin[2][e], fmaf(p[4 * i + 1], xin[1][e], p[4 * i] * xin[0][e])));
                    MV::store(y + ((size_t)g * 4 + i) * C + c, yout);
                }
            }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Backward of the mix for ONE token, by one warp (birkhoff4_backward_mix): with y_i = sum_j P_ij x_j,
//     dx_j = sum_i P_ij dy_i          (written as it is formed),
//     G_ij = dL/dP_ij = sum_c dy_i[c] x_j[c]   (returned as this lane's partial sums: mix_reduce16 adds them over the warp).
// Lane l takes the 16-byte slices l, l + 32, ... of each of the eight streams (4 of x, 4 of dy).  sP: as in mix_tokens.
template <bool XBF16>
BK4_DEV void mix_backward_token(const float* sP, int t, const typename MixVec<XBF16>::elem* __restrict__ x,
                                const typename MixVec<XBF16>::elem* __restrict__ dy, typename MixVec<XBF16>::elem* __restrict__ dx,
                                int C, float (&G)[16]) {
    using MV = MixVec<XBF16>;
    constexpr int V = MV::kElems;
    const int lane = threadIdx.x & 31;
    float p[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        p[q] = sP[q * kSmStride + t];
        G[q] = 0.0f;
    }
    for (int c = lane * V; c < C; c += 32 * V) {
        typename MV::raw rx[4], rg[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) rx[j] = MV::load_raw(x + (size_t)j * C + c);
#pragma unroll
        for (int i = 0; i < 4; ++i) rg[i] = MV::load_raw(dy + (size_t)i * C + c);
        float xin[4][V], gin[4][V];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            MV::widen(rx[j], xin[j]);
            MV::widen(rg[j], gin[j]);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int e = 0; e < V; ++e) G[4 * i + j] = fmaf(gin[i][e], xin[j][e], G[4 * i + j]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float out[V];
#pragma unroll
            for (int e = 0; e < V; ++e)
                out[e] = fmaf(p[12 + j], gin[3][e], fmaf(p[8 + j], gin[2][e], fmaf(p[4 + j], gin[1][e], p[j] * gin[0][e])));
            MV::store(dx + (size_t)j * C + c, out);
        }
    }
}

// Sum of the 16 partial sums G[.] over the 32 lanes of the warp by a transposing butterfly: at each of the steps
// xor 16, 8, 4, 2 a lane keeps one half of its values and hands the other half to its partner (8 + 4 + 2 + 1 shuffles),
// a last step xor 1 completes the sum: 16 shuffles instead of the 80 of sixteen plain butterflies.  Afterwards lane l
// holds the total of entry mix_entry_of_lane(l) (lanes l and l ^ 1 hold the same one).
BK4_DEV int mix_entry_of_lane(int lane) { return lane >> 1; }
BK4_DEV float mix_reduce16(const float (&G)[16]) {
    const int lane = threadIdx.x & 31;
    const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4, h2 = lane & 2;
    float a[8], b[4], c[2];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = (h16 ? G[k + 8] : G[k]) + __shfl_xor_sync(0xffffffffu, h16 ? G[k] : G[k + 8], 16);
#pragma unroll
    for (int k = 0; k < 4; ++k) b[k] = (h8 ? a[k + 4] : a[k]) + __shfl_xor_sync(0xffffffffu, h8 ? a[k] : a[k + 4], 8);
#pragma unroll
    for (int k = 0; k < 2; ++k) c[k] = (h4 ? b[k + 2] : b[k]) + __shfl_xor_sync(0xffffffffu, h4 ? b[k] : b[k + 2], 4);
    float d = (h2 ? c[1] : c[0]) + __shfl_xor_sync(0xffffffffu, h2 ? c[0] : c[1], 2);
    d += __shfl_xor_sync(0xffffffffu, d, 1);
    return d;  // entry 8 [lane & 16] + 4 [lane & 8] + 2 [lane & 4] + [lane & 2] = lane >> 1
}

}  // namespace bk4
