// Value types of the per-cell arithmetic.  The cell update is written once, generic in the
// value type V:
//   V = float / double : one cell per thread, scalar instructions;
//   V = F2             : TWO fp32 cells per thread, one packed instruction (Blackwell FADD2 / FMUL2 / FFMA2, PTX
//                        add / mul / fma .rn.f32x2) per operation of the expression tree.
// Every operation of the tree is exactly one call here: vfma is ONE fused multiply-add (one rounding), + - * are one
// IEEE operation each (the translation units are built with --fmad=false, so nvcc contracts nothing).  ptxas 12.9
// contracts a packed mul whose only consumer is a packed add into FFMA2 regardless of --fmad; the specification has
// no product that feeds a sum un-fused except the velocity u_a = (...) * (1/rho), which has several consumers and
// stays an FMUL2 (checked in the SASS and, bit for bit, by the GPU parity tests).
#pragma once
#include <cuda_runtime.h>

namespace lbm {

struct F2 {
    unsigned long long v;    // lo 32 bits: cell x, hi 32 bits: cell x + 1
};

template <class V> struct ScalarOfV { using type = V; };
template <> struct ScalarOfV<F2> { using type = float; };

__device__ __forceinline__ F2 pack2(float lo, float hi) {
    F2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(F2 a, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }

__device__ __forceinline__ F2 operator+(F2 a, F2 b) { F2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ F2 operator-(F2 a, F2 b) { F2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ F2 operator*(F2 a, F2 b) { F2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ F2 operator-(F2 a) { F2 d; d.v = a.v ^ 0x8000000080000000ULL; return d; }
__device__ __forceinline__ F2 vfma(F2 a, F2 b, F2 c) {
    F2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return d;
}
__device__ __forceinline__ float vfma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double vfma(double a, double b, double c) { return __fma_rn(a, b, c); }

// a constant / a run-time scalar in every lane
template <class V> __device__ __forceinline__ V vconst(double c) { return (V)c; }
template <> __device__ __forceinline__ F2 vconst<F2>(double c) { return pack2((float)c, (float)c); }
template <class V, class T> __device__ __forceinline__ V vbcast(T c) { return (V)c; }
template <> __device__ __forceinline__ F2 vbcast<F2, float>(float c) { return pack2(c, c); }

// 1 / x, IEEE division per lane
__device__ __forceinline__ float vrecip(float x) { return 1.0f / x; }
__device__ __forceinline__ double vrecip(double x) { return 1.0 / x; }
__device__ __forceinline__ F2 vrecip(F2 x) {
    float a, b;
    unpack2(x, a, b);
    return pack2(1.0f / a, 1.0f / b);
}

// Eq. 10 / 24: psi = rho0 (1 - exp(-(rho / rho0))), or psi = rho (R3)
template <class T>
__device__ __forceinline__ T psi_of(T rho, int kind, T rho0) {
    if (kind == 1) return rho;
    return rho0 * ((T)1 - exp(-(rho / rho0)));
}
__device__ __forceinline__ F2 psi_of(F2 rho, int kind, float rho0) {
    if (kind == 1) return rho;
    float a, b;
    unpack2(rho, a, b);
    return pack2(psi_of(a, 0, rho0), psi_of(b, 0, rho0));
}

}  // namespace lbm
