// mathx.cuh -- precision traits of the P2P / M2P arithmetic.
//   double: plain fp64 (rsqrt, exp from libdevice).
//   float : fp32 with the special-function unit: MUFU.RSQ (rsqrt.approx) and MUFU.EX2 (ex2.approx) --
//           "rsqrt/exp on the SFU" of the north star; ~2 ulp each, far below the 1e-4 parity bar.
#pragma once
#include <cuda_runtime.h>

template <typename T> struct Real;

// fp64 has no special-function unit; libdevice's rsqrt / exp cost ~12 and ~25 fp64-pipe instructions with
// their range checks.  The P2P arguments are tame (r^2 > 0 finite, 0 <= kappa r < 700), so:
//   rsqrt: MUFU.RSQ64H seed (rsqrt.approx.ftz.f64, ~2^-22 relative) + one third-order step
//          y (1 + e/2 + 3 e^2/8), e = 1 - x y^2   -> ~2^-60, 5 fp64 instructions;
//   exp  : n = rint(t log2 e) by the 1.5 * 2^52 shift, Cody-Waite reduction with a two-part ln 2, Taylor
//          polynomial of degree 12 on |r| <= ln(2)/2 (remainder 2e-16), 2^n added into the exponent field;
//          t < -700 returns 0 (the result would be below 1e-304).
// Both are checked through the direct-mode parity tests against the oracle's libm (1e-11 bar, observed 1e-15).
template <> struct Real<double> {
    typedef double4 vec4;
    static __device__ __forceinline__ double rsqrt_(double x)
    {
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        const double h = x * y;
        const double e = fma(-h, y, 1.0);
        const double p = fma(0.375, e, 0.5);
        return fma(y, e * p, y);
    }
    // exp(-kappa r); ks = kappa
    static __device__ __forceinline__ double exp_neg(double ks, double r)
    {
        const double t = -ks * r;
        const double z = fma(t, 1.4426950408889634, 6755399441055744.0);
        const double n = z - 6755399441055744.0;
        double f = fma(n, -6.93147180369123816490e-01, t);
        f = fma(n, -1.90821492927058770002e-10, f);
        double p = 2.08767569878680989792e-09;                       // 1/12!
        p = fma(p, f, 2.50521083854417187751e-08);
        p = fma(p, f, 2.75573192239858906526e-07);
        p = fma(p, f, 2.75573192239858906526e-06);
        p = fma(p, f, 2.48015873015873015873e-05);
        p = fma(p, f, 1.98412698412698412698e-04);
        p = fma(p, f, 1.38888888888888888889e-03);
        p = fma(p, f, 8.33333333333333333333e-03);
        p = fma(p, f, 4.16666666666666666667e-02);
        p = fma(p, f, 1.66666666666666666667e-01);
        p = fma(p, f, 0.5);
        p = fma(p, f, 1.0);
        p = fma(p, f, 1.0);
        const int hi = __double2hiint(p) + (__double2loint(z) << 20);
        return t < -700.0 ? 0.0 : __hiloint2double(hi, __double2loint(p));
    }
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

