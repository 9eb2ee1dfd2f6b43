// m2p.cuh -- M2P (a6) of the Cartesian Taylor treecode, eq. (13)-(14).
// Compiled once per expansion order P (m2p_inst.cu with -DM2P_P=<P>) so that the orders build in parallel.
#pragma once
#include <cuda_runtime.h>
#include "mathx.cuh"
#define PYGBE_TG_M2P 128

struct M2PArgs {
    const int *skip; const int4 *items; const int *m2p_cell; int n_items; int np;
    const double4 *tpos; const double4 *cgeo; const double *mom;   // mom[cell][2][Nc]: MV, MK (farfield.cuh)
    double ca, cb;             // the region's multipole is ca * MV + cb * MK
    double kappa; double *out;
    int yukawa; int fp32; cudaStream_t stream;
};

// Taylor coefficients by recurrence ("recursive relations for the Green's function of
// the Poisson equation [20] and linearized Poisson-Boltzmann equation [21]"; reading A13), d = x - y_c,
// R^2 = |d|^2, n = |k|, terms with a negative index dropped:
//   Laplace:  a^0 = 1/R;       n R^2 a^k = (2n-1) sum_i d_i a^(k-e_i) - (n-1) sum_i a^(k-2e_i)
//   Yukawa :  b^0 = exp(-kappa R), a^0 = b^0/R;
//             n b^k     = kappa [ sum_i d_i a^(k-e_i) - sum_i a^(k-2e_i) ]
//             n R^2 a^k = (2n-1) sum_i d_i a^(k-e_i) - (n-1) sum_i a^(k-2e_i)
//                         + kappa [ sum_i d_i b^(k-e_i) - sum_i b^(k-2e_i) ]
// The loops are fully unrolled for the compile-time order P: the coefficient arrays live in registers
// and only two order-shells are alive at a time.  Returns sum_k a^k M^k (M in shared memory).
// T = double: fp64 throughout.  T = float: fp32 recurrence with MUFU rsqrt / ex2 (mathx.cuh); SURVEY A8b:
// fp32 coefficient error 1.4e-7 (order 0) .. 1.8e-6 (order 8), far below the truncation error.
template <int P, bool YUKAWA, typename T>
__device__ __forceinline__ T m2p_eval(T dx, T dy, T dz, T kappa, T kscaled, const T *__restrict__ M)
{
    T a[P + 1][P + 1][P + 1];
    T b[YUKAWA ? P + 1 : 1][YUKAWA ? P + 1 : 1][YUKAWA ? P + 1 : 1];
    const T R2 = dx * dx + dy * dy + dz * dz;
    const T invR = Real<T>::rsqrt_(R2);
    const T invR2 = invR * invR;
    if constexpr (YUKAWA) {
        b[0][0][0] = Real<T>::exp_neg(kscaled, R2 * invR);
        a[0][0][0] = b[0][0][0] * invR;
    } else {
        a[0][0][0] = invR;
    }
    T acc = a[0][0][0] * M[0];
    int idx = 1;
#pragma unroll
    for (int n = 1; n <= P; n++) {
        const T c1 = T(2 * n - 1) / T(n) * invR2, c2 = T(n - 1) / T(n) * invR2;
        const T c3 = kappa / T(n), c4 = c3 * invR2;
#pragma unroll
        for (int kx = n; kx >= 0; kx--) {
#pragma unroll
            for (int ky = n - kx; ky >= 0; ky--) {
                const int kz = n - kx - ky;
                T s1 = T(0), s2 = T(0);
                if (kx > 0) s1 += dx * a[kx > 0 ? kx - 1 : 0][ky][kz];
                if (ky > 0) s1 += dy * a[kx][ky > 0 ? ky - 1 : 0][kz];
                if (kz > 0) s1 += dz * a[kx][ky][kz > 0 ? kz - 1 : 0];
                if (kx > 1) s2 += a[kx > 1 ? kx - 2 : 0][ky][kz];
                if (ky > 1) s2 += a[kx][ky > 1 ? ky - 2 : 0][kz];
                if (kz > 1) s2 += a[kx][ky][kz > 1 ? kz - 2 : 0];
                T v = c1 * s1 - c2 * s2;
                if constexpr (YUKAWA) {
                    T t1 = T(0), t2 = T(0);
                    if (kx > 0) t1 += dx * b[kx > 0 ? kx - 1 : 0][ky][kz];
                    if (ky > 0) t1 += dy * b[kx][ky > 0 ? ky - 1 : 0][kz];
                    if (kz > 0) t1 += dz * b[kx][ky][kz > 0 ? kz - 1 : 0];
                    if (kx > 1) t2 += b[kx > 1 ? kx - 2 : 0][ky][kz];
                    if (ky > 1) t2 += b[kx][ky > 1 ? ky - 2 : 0][kz];
                    if (kz > 1) t2 += b[kx][ky][kz > 1 ? kz - 2 : 0];
                    b[kx][ky][kz] = c3 * (s1 - s2);
                    v += c4 * (t1 - t2);
                }
                a[kx][ky][kz] = v;
                acc += v * M[idx];
                idx++;
            }
        }
    }
    return acc;
}

// Work item = (target group, a run of its M2P list).  One thread per target; the moments of M2P_CB cells
// at a time are staged in shared memory (combined ca MV + cb MK, converted to T) and read by all threads
// as broadcasts.  The target offset d = x - y_c is always formed in fp64 and then rounded to T, so the
// fp32 path never subtracts large absolute coordinates; accumulation over cells is fp64.
#define M2P_CB 4
template <int P, bool YUKAWA, typename T>
__global__ void __launch_bounds__(PYGBE_TG_M2P)
k_m2p(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
      const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const double *__restrict__ mom,
      double ca, double cb, double kappa, double kscaled, double *__restrict__ out)
{
    constexpr int Nc = (P + 1) * (P + 2) * (P + 3) / 6;
    __shared__ T s_M[M2P_CB][Nc];
    __shared__ double4 s_c[M2P_CB];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t = it.x * PYGBE_TG_M2P + threadIdx.x;
    const bool ok = t < np;
    double4 X = ok ? tpos[t] : make_double4(1e30, 1e30, 1e30, 0);
    double acc = 0.0;
    for (int s0 = it.y; s0 < it.z; s0 += M2P_CB) {
        int nb = min(M2P_CB, it.z - s0);
        __syncthreads();
        for (int i = threadIdx.x; i < nb * Nc; i += PYGBE_TG_M2P) {
            int cb_ = i / Nc, k = i - cb_ * Nc;
            const double *m = mom + (long)m2p_cell[s0 + cb_] * 2 * Nc;
            s_M[cb_][k] = (T)(ca * m[k] + cb * m[Nc + k]);
        }
        if (threadIdx.x < nb) s_c[threadIdx.x] = cgeo[m2p_cell[s0 + threadIdx.x]];
        __syncthreads();
        for (int c_ = 0; c_ < nb; c_++) {
            double4 c = s_c[c_];
            acc += (double)m2p_eval<P, YUKAWA, T>((T)(X.x - c.x), (T)(X.y - c.y), (T)(X.z - c.z), (T)kappa,
                                                  (T)kscaled, s_M[c_]);
        }
    }
    if (ok) atomicAdd(out + t, acc);
}
