// m2p.cuh -- M2P (a6) of the Cartesian Taylor treecode, eq. (13)-(14).
// Compiled once per expansion order P (m2p_inst.cu with -DM2P_P=<P>) so that the orders build in parallel.
#pragma once
#include <cuda_runtime.h>
#include "mathx.cuh"
#ifndef PYGBE_TG
#define PYGBE_TG 64
#endif
#define PYGBE_TG_M2P PYGBE_TG

// Row stride of the combined moments momc[cell][stride] (elements of T): Nc padded to a multiple of 4 so
// that every row starts on a 16-byte boundary and can be moved with 16-byte cp.async.
static inline __host__ __device__ int m2p_stride(int Nc) { return (Nc + 3) / 4 * 4; }

struct M2PArgs {
    const int *skip; const int4 *items; const int *m2p_cell; int n_items; int np;
    const double4 *tpos; const double4 *cgeo;
    const void *momc;          // the region's multipoles ca * MV + cb * MK, already in T (written by P2M / M2M, farfield.cuh)
    double kappa; double *out;
    int yukawa; int fp32; cudaStream_t stream;
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

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
// The batches are double-buffered with cp.async (LDGSTS): while the threads evaluate the recurrences of one
// batch, the moments and centres of the next one stream from L2 into the other buffer (capture r1b showed
// 7-9 % barrier + 5-9 % long-scoreboard stalls with synchronous staging at 2 warps per CTA).
#ifndef M2P_CB
#define M2P_CB 4
#endif
#ifndef M2P_MINB
#define M2P_MINB 1       // min CTAs per SM asked of ptxas (register cap); tuning knob
#endif
template <int P, bool YUKAWA, typename T>
__global__ void __launch_bounds__(PYGBE_TG_M2P, M2P_MINB)
k_m2p(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
      const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const T *__restrict__ momc,
      double kappa, double kscaled, double *__restrict__ out)
{
    constexpr int Nc = (P + 1) * (P + 2) * (P + 3) / 6;
    constexpr int NCS = (Nc + 3) / 4 * 4;                    // = m2p_stride(Nc)
    constexpr int EPC = 16 / (int)sizeof(T);                 // elements per 16-byte chunk
    constexpr int CH = NCS / EPC;                            // chunks per cell
    __shared__ __align__(16) T s_M[2][M2P_CB][NCS];
    __shared__ __align__(16) double4 s_c[2][M2P_CB];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t = it.x * PYGBE_TG_M2P + threadIdx.x;
    const bool ok = t < np;
    const double4 X = ok ? tpos[t] : make_double4(1e30, 1e30, 1e30, 0);
    double acc = 0.0;
    auto stage = [&](int buf, int s0) {
        const int nb = min(M2P_CB, it.z - s0);
        for (int i = threadIdx.x; i < nb * CH; i += PYGBE_TG_M2P) {
            const int c_ = i / CH, j = i - c_ * CH;
            cp_async16(&s_M[buf][c_][j * EPC], momc + (long)m2p_cell[s0 + c_] * NCS + j * EPC);
        }
        if (threadIdx.x < nb * 2) {
            const int c_ = threadIdx.x >> 1, hf = threadIdx.x & 1;
            cp_async16((char *)&s_c[buf][c_] + 16 * hf, (const char *)(cgeo + m2p_cell[s0 + c_]) + 16 * hf);
        }
        cp_async_commit();
    };
    stage(0, it.y);
    int buf = 0;
    for (int s0 = it.y; s0 < it.z; s0 += M2P_CB, buf ^= 1) {
        const int nb = min(M2P_CB, it.z - s0);
        const bool more = s0 + M2P_CB < it.z;
        if (more) { stage(buf ^ 1, s0 + M2P_CB); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
        for (int c_ = 0; c_ < nb; c_++) {
            const double4 c = s_c[buf][c_];
            acc += (double)m2p_eval<P, YUKAWA, T>((T)(X.x - c.x), (T)(X.y - c.y), (T)(X.z - c.z), (T)kappa,
                                                  (T)kscaled, s_M[buf][c_]);
        }
        __syncthreads();                                     // buf is refilled two iterations from now
    }
    if (ok) atomicAdd(out + t, acc);
}

