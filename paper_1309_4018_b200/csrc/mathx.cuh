// mathx.cuh -- precision traits of the P2P / M2P arithmetic.
//   double: plain fp64 (rsqrt, exp from libdevice).
//   float : fp32 with the special-function unit: MUFU.RSQ (rsqrt.approx) and MUFU.EX2 (ex2.approx) --
//           "rsqrt/exp on the SFU" of the north star; ~2 ulp each, far below the 1e-4 parity bar.
#pragma once
#include <cuda_runtime.h>

template <typename T> struct Real;

template <> struct Real<double> {
    typedef double4 vec4;
    static __device__ __forceinline__ double rsqrt_(double x) { return rsqrt(x); }
    // exp(-kappa r); ks = kappa
    static __device__ __forceinline__ double exp_neg(double ks, double r) { return exp(-ks * r); }
    static __host__ __device__ double kscale(double kappa) { return kappa; }
};

template <> struct Real<float> {
    typedef float4 vec4;
    static __device__ __forceinline__ float rsqrt_(float x)
    {
        float y;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
        return y;
    }
    // exp(-kappa r) = 2^(-kappa log2(e) r); ks = kappa * log2(e)
    static __device__ __forceinline__ float exp_neg(float ks, float r)
    {
        float y;
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(-ks * r));
        return y;
    }
    static __host__ __device__ double kscale(double kappa) { return kappa * 1.4426950408889634; }
};

// Packed fp32 pairs (sm_100: add / sub / mul / fma .f32x2 = FADD2 / FMUL2 / FFMA2, one issue slot for two
// lanes; ptxas folds f2_pack(a, a) into a scalar broadcast operand).  Used by the mixed-precision P2P and M2P.
typedef unsigned long long f2_t;                                      // two packed floats
__device__ __forceinline__ f2_t f2_pack(float lo, float hi) { f2_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void f2_unpack(f2_t v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f2_t f2_add(f2_t a, f2_t b) { f2_t r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2_t f2_sub(f2_t a, f2_t b) { f2_t r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2_t f2_mul(f2_t a, f2_t b) { f2_t r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f2_t f2_fma(f2_t a, f2_t b, f2_t c) { f2_t r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

