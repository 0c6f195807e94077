// bk4_vec.cuh -- value types for the per-matrix solvers: `float` (one matrix per thread) and `float2`
// (two matrices per thread, one in each half, so that every FP32 instruction is a packed sm_100
// FFMA2/FADD2/FMUL2).  The solvers in bk4_core.cuh are written once against these overloads.
//
// sm_100a only.  MUFU ops (ex2/rcp/lg2) are scalar in hardware; the packed versions issue one per half.
#pragma once
#include <cuda_runtime.h>

namespace bk4 {

#define BK4_DEV __device__ __forceinline__

// ---------------------------------------------------------------- SFU primitives (MUFU.EX2 / RCP / LG2)
BK4_DEV float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
BK4_DEV float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
BK4_DEV float sqrt_approx(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
BK4_DEV float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---------------------------------------------------------------- masks
// Masks are 32-bit 0/1 words combined with bitwise ops, never `bool`: for the Blackwell targets (compute_100*,
// compute_120) nvcc 12.9 miscompiles the solver's loop-carried `bool` logic -- with `bool` (and with a struct of
// two `bool`s) the PTX of newton_forward lost the `rejected` path and the `accepted` guard of the re-basing,
// while the same source is compiled correctly for compute_90.  tests/test_gpu_parity.py
// (test_two_variants_agree_and_deterministic, test_config5_full_size) are the regression tests.
struct bool1 {
    unsigned x;
    BK4_DEV bool1() : x(0u) {}
    BK4_DEV explicit bool1(bool a) : x(a ? 1u : 0u) {}
};
struct bool2 {
    unsigned x, y;
    BK4_DEV bool2() : x(0u), y(0u) {}
    BK4_DEV bool2(bool a, bool b) : x(a ? 1u : 0u), y(b ? 1u : 0u) {}
};

template <class V>
struct vtraits;
template <>
struct vtraits<float> {
    using mask = bool1;
    static constexpr int lanes = 1;
};
template <>
struct vtraits<float2> {
    using mask = bool2;
    static constexpr int lanes = 2;
};

// ---------------------------------------------------------------- float
BK4_DEV float vsplat(float, float a) { return a; }
// explicit _rn intrinsics: never contracted into FMAs by the compiler, so that the scalar and the packed
// instantiation of a solver perform the same roundings and give the same bits
BK4_DEV float vadd(float a, float b) { return __fadd_rn(a, b); }
BK4_DEV float vsub(float a, float b) { return __fmaf_rn(b, -1.0f, a); }
BK4_DEV float vmul(float a, float b) { return __fmul_rn(a, b); }
BK4_DEV float vfma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
BK4_DEV float vneg(float a) { return -a; }
BK4_DEV float vabs(float a) { return fabsf(a); }
BK4_DEV float vmax(float a, float b) { return fmaxf(a, b); }
BK4_DEV float vmin(float a, float b) { return fminf(a, b); }
BK4_DEV float vrcp(float a) { return rcp_approx(a); }
BK4_DEV float vex2(float a) { return ex2_approx(a); }
BK4_DEV float vlg2(float a) { return lg2_approx(a); }
BK4_DEV bool1 vgt(float a, float b) { return bool1(a > b); }
BK4_DEV bool1 vlt(float a, float b) { return bool1(a < b); }
BK4_DEV bool1 veq(float a, float b) { return bool1(a == b); }
BK4_DEV float vsel(bool1 m, float a, float b) { return m.x != 0u ? a : b; }
BK4_DEV bool1 mand(bool1 a, bool1 b) { bool1 r; r.x = a.x & b.x; return r; }
BK4_DEV bool1 mor(bool1 a, bool1 b) { bool1 r; r.x = a.x | b.x; return r; }
BK4_DEV bool1 mnot(bool1 a) { bool1 r; r.x = a.x ^ 1u; return r; }
BK4_DEV bool many(bool1 a) { return a.x != 0u; }
BK4_DEV bool mall(bool1 a) { return a.x != 0u; }
BK4_DEV bool1 msplat(float, bool a) { return bool1(a); }
BK4_DEV int isel(bool1 m, int a, int b) { return m.x != 0u ? a : b; }

// ---------------------------------------------------------------- float2 (packed: FFMA2 / FADD2 / FMUL2)
BK4_DEV float2 vsplat(float2, float a) { return make_float2(a, a); }
BK4_DEV float2 vadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
BK4_DEV float2 vmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
BK4_DEV float2 vfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
BK4_DEV float2 vsub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.0f, -1.0f), a); }
BK4_DEV float2 vneg(float2 a) { return make_float2(-a.x, -a.y); }
BK4_DEV float2 vabs(float2 a) { return make_float2(fabsf(a.x), fabsf(a.y)); }
BK4_DEV float2 vmax(float2 a, float2 b) { return make_float2(fmaxf(a.x, b.x), fmaxf(a.y, b.y)); }
BK4_DEV float2 vmin(float2 a, float2 b) { return make_float2(fminf(a.x, b.x), fminf(a.y, b.y)); }
BK4_DEV float2 vrcp(float2 a) { return make_float2(rcp_approx(a.x), rcp_approx(a.y)); }
BK4_DEV float2 vex2(float2 a) { return make_float2(ex2_approx(a.x), ex2_approx(a.y)); }
BK4_DEV float2 vlg2(float2 a) { return make_float2(lg2_approx(a.x), lg2_approx(a.y)); }
BK4_DEV bool2 vgt(float2 a, float2 b) { return bool2(a.x > b.x, a.y > b.y); }
BK4_DEV bool2 vlt(float2 a, float2 b) { return bool2(a.x < b.x, a.y < b.y); }
BK4_DEV bool2 veq(float2 a, float2 b) { return bool2(a.x == b.x, a.y == b.y); }
BK4_DEV float2 vsel(bool2 m, float2 a, float2 b) { return make_float2(m.x != 0u ? a.x : b.x, m.y != 0u ? a.y : b.y); }
BK4_DEV bool2 mand(bool2 a, bool2 b) { bool2 r; r.x = a.x & b.x; r.y = a.y & b.y; return r; }
BK4_DEV bool2 mor(bool2 a, bool2 b) { bool2 r; r.x = a.x | b.x; r.y = a.y | b.y; return r; }
BK4_DEV bool2 mnot(bool2 a) { bool2 r; r.x = a.x ^ 1u; r.y = a.y ^ 1u; return r; }
BK4_DEV bool many(bool2 a) { return (a.x | a.y) != 0u; }
BK4_DEV bool mall(bool2 a) { return (a.x & a.y) != 0u; }
BK4_DEV bool2 msplat(float2, bool a) { return bool2(a, a); }
BK4_DEV int2 isel(bool2 m, int2 a, int2 b) { return make_int2(m.x != 0u ? a.x : b.x, m.y != 0u ? a.y : b.y); }

// half access (lane k of a value): used only for I/O and diagnostics
BK4_DEV float vget(float a, int) { return a; }
BK4_DEV float vget(float2 a, int k) { return k ? a.y : a.x; }
BK4_DEV bool mget(bool1 a, int) { return a.x != 0u; }
BK4_DEV bool mget(bool2 a, int k) { return (k ? a.y : a.x) != 0u; }

}  // namespace bk4
