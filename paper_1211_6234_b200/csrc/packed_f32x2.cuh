// packed_f32x2.cuh -- two fp32 values in one 64-bit register pair and the sm_100a instructions that work
// on both at once (FFMA2 / FMUL2 / FADD2).  Used for replica pairs in the Metropolis kernel and for
// complex numbers (re, im) in the FFT field.
#pragma once
#include <cuda_runtime.h>

// One instruction works on both halves.  A scalar operand written f2_bc(x) is folded by ptxas into the
// instruction's broadcast / immediate operand form, so constants cost nothing.
typedef unsigned long long f2;
__device__ __forceinline__ f2 f2_make(float lo, float hi) {
    f2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ f2 f2_bc(float a) { return f2_make(a, a); }
__device__ __forceinline__ void f2_split(f2 v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f2 f2_fma(f2 a, f2 b, f2 c) {
    f2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f2 f2_mul(f2 a, f2 b) {
    f2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 f2_add(f2 a, f2 b) {
    f2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f2 f2_sub(f2 a, f2 b) { return f2_fma(b, f2_bc(-1.0f), a); }  // a - b, exact like FADD
