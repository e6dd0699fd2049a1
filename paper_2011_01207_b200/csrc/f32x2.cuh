// f32x2.cuh -- packed FP32 arithmetic of sm_100 (add/sub/mul/fma.rn.f32x2 -> FADD2/FMUL2/FFMA2).
//
// A packed instruction does two IEEE FP32 operations (same rounding as the scalar forms) on an
// aligned 64-bit register pair and takes ONE issue slot; the FMA pipe is busy two cycles for it,
// so the FP32 peak is unchanged (measured on B200: 8 FFMA2 = 16 FFMA = 16.3 cycles per warp and
// SMSP) but the issue port is free every other cycle for MUFU, LDS and integer instructions.  The
// pair kernels are issue bound in scalar form (61 instructions per pair, 46 of them FP32), which is
// why they are written with these.
//
// ptxas folds a per-half negation into the operand modifier (-R.F32x2) and a pack of the same
// scalar twice into a broadcast operand (R.F32 / UR.F32); a pack of two unrelated registers
// costs MOVs, so values are kept in the pairs they are produced in.
#pragma once

#include <cuda_runtime.h>

namespace tkhp {

typedef unsigned long long f2;      // two packed floats: lo = bits 0..31, hi = bits 32..63

__device__ __forceinline__ f2 pk(float lo, float hi) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 bc(float s) { return pk(s, s); }
__device__ __forceinline__ float lo(f2 v) {
    float a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
    return a;
}
__device__ __forceinline__ float hi(f2 v) {
    float a, b;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
    return b;
}
__device__ __forceinline__ f2 neg2(f2 v) { return pk(-lo(v), -hi(v)); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b) {
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b) {
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f2 sub2(f2 a, f2 b) {
    f2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

}  // namespace tkhp
