// bk4_math.cuh -- SFU primitives, constants and 256-bit global memory access for the batched 4x4 Birkhoff
// projection kernels.  sm_100a only.
//
// Cost model the kernels are written against (measured on B200, profiles/r2_pipe_microbench.md): per SM
// sub-partition one warp instruction issues per clock; FADD/FMUL/FFMA are full rate, every ALU-pipe instruction
// (FMNMX, FSEL, FSETP, ISETP, LOP3, ...) and every packed FFMA2/FADD2/FMUL2 holds the issue port for two clocks,
// MUFU (ex2/rcp/sqrt) runs at a quarter rate on its own queue.  So the code prefers FMA-pipe arithmetic over
// selects and min/max, keeps control flow warp-uniform, and moves data-dependent indexing to shared memory.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bk4 {

#define BK4_DEV __device__ __forceinline__

constexpr float kLog2e = 1.4426950408889634f;
#define kInf __int_as_float(0x7f800000)
#define kNaN __int_as_float(0x7fc00000)

// ---------------------------------------------------------------- SFU primitives (MUFU.EX2 / RCP / SQRT / LG2)
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

// ---------------------------------------------------------------- 256-bit global access
// A 64-byte matrix is two 32-byte DRAM sectors; each thread moves its matrix with two 256-bit LDG/STG
// (ld.global.v8.f32, new on sm_100): every request touches whole sectors and nothing is fetched twice.
BK4_DEV void ldg256(const float* p, float (&a)[8]) {  // read-only path, no L1 allocation
    asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]), "=f"(a[4]), "=f"(a[5]), "=f"(a[6]), "=f"(a[7])
                 : "l"(p));
}
// plain (coherent) version: used when the output may alias the input (P == H, dH == dP) and for re-reads
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

// ---------------------------------------------------------------- programmatic dependent launch
// Every kernel of the library starts with this: griddepcontrol.wait returns once the kernel before it in the
// stream has completed and its writes are visible; launch_dependents then lets the kernel after it begin
// launching.  Launched with programmatic stream serialization, the next kernel's launch latency and block ramp-up
// overlap this kernel's tail; stream-order semantics are unchanged because nothing is read or written before the
// wait.
BK4_DEV void pdl_wait_and_trigger() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

}  // namespace bk4
