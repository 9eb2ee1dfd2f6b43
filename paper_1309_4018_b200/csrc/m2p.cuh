// m2p.cuh -- M2P (a6) of the Cartesian Taylor treecode, eq. (13)-(14).
// Compiled once per expansion order P (m2p_inst.cu with -DM2P_P=<P>) so that the orders build in parallel.
//
// What is evaluated is eq. (14)'s truncated series  sum_{|k| <= P} a^k(x, y_c) M^k,  a^k = (1/k!) D_y^k G.
// The paper obtains a^k by recurrences (reading A13).  Both kernels are radial,
// G = F(s), s = |d|^2 / 2, d = x - y_c, and for such a function
//     D_d^k F(s) = sum_j  prod_axes [ k_a! / (2^j_a j_a! (k_a - 2 j_a)!) d_a^(k_a - 2 j_a) ]  F^(|k| - |j|)(s)
// (derivatives of a function of a quadratic; j_a <= k_a / 2).  Collecting the series by the order m of the
// radial derivative and by the monomial d^e, e = k - 2j, gives the same sum in the form
//     sum_k a^k M^k = sum_{m=0..P} F^(m)(s) Q_m,     Q_m = sum_{e : |e| <= m, 2m - |e| <= P} W_{m,e} d^e,
//     W_{m,e} = (-1)^|e| / e!  sum_{|j| = m - |e|}  M^(e + 2j) / (2^|j| j!)
// where the W depend on the cell only: they are formed when the cell's multipoles are (P2M / M2M epilogue,
// farfield.cuh, from a table built at create) and replace the multipoles as the M2P's input.  The M here are the
// HARMONICALLY REDUCED moments of tables.cuh ((laplace - kappa^2) G = 0 folds every moment with kz >= 2 into lower
// ones, exactly), so only e with ez <= 1 occur.  Per (target, cell) the work is then (P+1)^2 - 1 multiplies for the
// monomials and one FMA per W -- 84 per moment set at P = 6, 165 at P = 8 (unreduced: Nc - 1 and 130 / 295) -- instead
// of a recurrence of 6 (Laplace) to 12 (Yukawa) instructions per coefficient, and its form is
// independent of the kernel: Laplace and Yukawa differ only in the table and in the P + 1 numbers F^(m)(s),
//     F^(0) = exp(-kappa r) / r,   F^(1) = -exp(-kappa r) (kappa r + 1) / r^3,
//     F^(m+1) = -[ (2m + 1) F^(m) - kappa^2 F^(m-1) ] / r^2        (kappa = 0: Laplace),
// so the two regions on either side of a surface set ("twins") are evaluated in one pass.
// fp32 check (numpy emulation, P = 6 and 8, cells of 2..16 A at 1..4 times the MAC distance): relative error
// <= 5.5e-7 against the fp64 evaluation of the same series.
#pragma once
#include <cuda_runtime.h>
#include "mathx.cuh"
#ifndef PYGBE_TG
#define PYGBE_TG 64
#endif
#define PYGBE_TG_M2P PYGBE_TG

// number of W_{m,e} per moment set, in the order the kernel consumes them (ex, ey, ez ascending, then J)
// (harmonically reduced moments, tables.cuh: ez <= 1, i.e. 2 t + 1 monomials of degree t)
static inline __host__ __device__ constexpr int m2p_nw(int P)
{
    int n = 0;
    for (int t = 0; t <= P; t++) n += (2 * t + 1) * ((P - t) / 2 + 1);
    return n;
}
#define M2P_EZ(P, ex, ey) ((P) - (ex) - (ey) < 1 ? (P) - (ex) - (ey) : 1)      // last ez of the reduced index set
// Row stride of wc[cell][stride] (elements of T): the W of the tree owner and, interleaved, of its twin,
// padded to a multiple of 4 so that every row starts on a 16-byte boundary and moves with 16-byte cp.async.
static inline __host__ __device__ constexpr int m2p_stride(int P, bool twin) { return (m2p_nw(P) * (twin ? 2 : 1) + 3) / 4 * 4; }

struct M2PArgs {
    const int *skip; const int4 *items; const int *m2p_cell; int n_items; int np;
    const double4 *tpos; const double4 *cgeo;
    const void *wc;            // W_{m,e} of the tree owner (and twin), already combined and in T (farfield.cuh)
    double kappaA, kappaB; double *outA, *outB;
    int twin; int fp32; cudaStream_t stream;
    int lap;                   // Laplace form (k_m2p_lap): wc holds the C'_f; ggeo = target group centres
    const double4 *ggeo;
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T> struct Chunk;                                   // one 16-byte shared-memory read
template <> struct Chunk<float> { typedef float4 V; static constexpr int N = 4;
    static __device__ __forceinline__ void get(const float *p, float (&c)[4]) { const float4 v = *(const float4 *)p; c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w; } };
template <> struct Chunk<double> { typedef double2 V; static constexpr int N = 2;
    static __device__ __forceinline__ void get(const double *p, double (&c)[2]) { const double2 v = *(const double2 *)p; c[0] = v.x; c[1] = v.y; } };

// Q_m (+ twin) of one cell at offset d: the loops are fully unrolled for the compile-time order, so the
// position in the W stream, the accumulator index and the 16-byte reads are all static.
template <int P, int NS, typename T>
__device__ __forceinline__ void m2p_q(T dx, T dy, T dz, const T *__restrict__ w, T (&q)[P + 1][NS])
{
    constexpr int EPC = Chunk<T>::N;
    T cur[EPC];
    int idx = 0;
#pragma unroll
    for (int m = 0; m <= P; m++)
#pragma unroll
        for (int s = 0; s < NS; s++) q[m][s] = T(0);
    T px = T(1);
#pragma unroll
    for (int ex = 0; ex <= P; ex++) {
        T pxy = px;
#pragma unroll
        for (int ey = 0; ey <= P - ex; ey++) {
            T mono = pxy;
#pragma unroll
            for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++) {
                const int t = ex + ey + ez;
#pragma unroll
                for (int J = 0; J <= (P - t) / 2; J++) {
#pragma unroll
                    for (int s = 0; s < NS; s++) {
                        if (idx % EPC == 0) Chunk<T>::get(w + idx, cur);
                        q[t + J][s] = fma(cur[idx % EPC], mono, q[t + J][s]);
                        idx++;
                    }
                }
                mono *= dz;
            }
            pxy *= dy;
        }
        px *= dx;
    }
}

// sum_m F^(m)(s) q_m for one kernel (kappa = 0: Laplace)
template <int P, int NS, typename T>
__device__ __forceinline__ T m2p_radial(T r, T rinv, T rinv2, T kappa, T kscaled, const T (&q)[P + 1][NS], int s)
{
    const T E = kappa != T(0) ? Real<T>::exp_neg(kscaled, r) : T(1);
    T gm = E * rinv;                                   // F^(0)
    T acc = gm * q[0][s];
    if (P >= 1) {
        T g = -E * (kappa * r + T(1)) * rinv * rinv2;  // F^(1)
        acc = fma(g, q[1][s], acc);
        const T k2 = kappa * kappa;
#pragma unroll
        for (int m = 1; m < P; m++) {
            const T gn = -(T(2 * m + 1) * g - k2 * gm) * rinv2;
            gm = g; g = gn;
            acc = fma(g, q[m + 1][s], acc);
        }
    }
    return acc;
}

// fp32 twin regions: the W of A and B are interleaved in the row, so the pair (Q_m^A, Q_m^B) is one packed
// accumulator and each W pair costs one FFMA2 with the monomial as broadcast operand; the radial part runs on
// the pairs (F_A^(m), F_B^(m)) likewise.  Returns (sum_m F_A^(m) Q_m^A, sum_m F_B^(m) Q_m^B).
template <int P>
__device__ __forceinline__ f2_t m2p_twin_packed(float dx, float dy, float dz, const float *__restrict__ w, float kappaA,
                                                float ksA, float kappaB, float ksB)
{
    f2_t q[P + 1];
#pragma unroll
    for (int m = 0; m <= P; m++) q[m] = 0;
    int idx = 0;
    float4 cur = make_float4(0.f, 0.f, 0.f, 0.f);
    float px = 1.f;
#pragma unroll
    for (int ex = 0; ex <= P; ex++) {
        float pxy = px;
#pragma unroll
        for (int ey = 0; ey <= P - ex; ey++) {
            float mono = pxy;
#pragma unroll
            for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++) {
                const int t = ex + ey + ez;
                const f2_t m2 = f2_pack(mono, mono);
#pragma unroll
                for (int J = 0; J <= (P - t) / 2; J++) {
                    if (idx % 2 == 0) cur = *(const float4 *)(w + 2 * idx);
                    q[t + J] = f2_fma(idx % 2 == 0 ? f2_pack(cur.x, cur.y) : f2_pack(cur.z, cur.w), m2, q[t + J]);
                    idx++;
                }
                mono *= dz;
            }
            pxy *= dy;
        }
        px *= dx;
    }
    const float r2 = dx * dx + dy * dy + dz * dz;
    const float rinv = Real<float>::rsqrt_(r2), rinv2 = rinv * rinv, r = r2 * rinv;
    const float EA = kappaA != 0.f ? Real<float>::exp_neg(ksA, r) : 1.f, EB = kappaB != 0.f ? Real<float>::exp_neg(ksB, r) : 1.f;
    const f2_t ri2 = f2_pack(rinv2, rinv2), kap = f2_pack(kappaA, kappaB), k2 = f2_mul(kap, kap);
    f2_t gm = f2_mul(f2_pack(EA, EB), f2_pack(rinv, rinv));                                    // F^(0)
    f2_t acc = f2_mul(gm, q[0]);
    if (P >= 1) {
        const float nr3 = -rinv * rinv2;
        f2_t g = f2_mul(f2_mul(f2_pack(EA, EB), f2_fma(kap, f2_pack(r, r), f2_pack(1.f, 1.f))), f2_pack(nr3, nr3));   // F^(1)
        acc = f2_fma(g, q[1], acc);
#pragma unroll
        for (int m = 1; m < P; m++) {
            const float c = -(float)(2 * m + 1);
            const f2_t gn = f2_mul(f2_fma(g, f2_pack(c, c), f2_mul(k2, gm)), ri2);             // -[(2m+1) g - k^2 gm] / r^2
            gm = g; g = gn;
            acc = f2_fma(g, q[m + 1], acc);
        }
    }
    return acc;
}

// Work item = (target group, a run of its M2P list).  One thread per target; the W rows of CB cells at a
// time are staged in shared memory and read by all threads as 16-byte broadcasts.  The target offset
// d = x - y_c is always formed in fp64 and then rounded to T, so the fp32 path never subtracts large absolute
// coordinates; accumulation over cells is fp64.  The batches are double-buffered with cp.async (LDGSTS):
// while the threads work on one batch, the rows and centres of the next stream from L2 into the other buffer.
template <int P, bool TWIN, typename T>
__global__ void __launch_bounds__(PYGBE_TG_M2P)
k_m2p(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
      const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const T *__restrict__ wc,
      double kappaA, double kscaledA, double kappaB, double kscaledB, double *__restrict__ outA, double *__restrict__ outB)
{
    constexpr int NS = TWIN ? 2 : 1;
    constexpr int STRIDE = m2p_stride(P, TWIN);
    constexpr int EPC = 16 / (int)sizeof(T);                 // elements per 16-byte chunk
    constexpr int CH = STRIDE / EPC;                         // chunks per cell
    constexpr int CBW = 12288 / (STRIDE * (int)sizeof(T));   // cells per batch: about 12 KB per buffer
    constexpr int CB = CBW < 1 ? 1 : (CBW > 4 ? 4 : CBW);
    __shared__ __align__(16) T s_W[2][CB][STRIDE];
    __shared__ __align__(16) double4 s_c[2][CB];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t = it.x * PYGBE_TG_M2P + threadIdx.x;
    const bool ok = t < np;
    const double4 X = ok ? tpos[t] : make_double4(1e30, 1e30, 1e30, 0);
    double accA = 0.0, accB = 0.0;
    auto stage = [&](int buf, int s0) {
        const int nb = min(CB, it.z - s0);
        for (int i = threadIdx.x; i < nb * CH; i += PYGBE_TG_M2P) {
            const int c_ = i / CH, j = i - c_ * CH;
            cp_async16(&s_W[buf][c_][j * EPC], wc + (long)m2p_cell[s0 + c_] * STRIDE + j * EPC);
        }
        if (threadIdx.x < nb * 2) {
            const int c_ = threadIdx.x >> 1, hf = threadIdx.x & 1;
            cp_async16((char *)&s_c[buf][c_] + 16 * hf, (const char *)(cgeo + m2p_cell[s0 + c_]) + 16 * hf);
        }
        cp_async_commit();
    };
    stage(0, it.y);
    int buf = 0;
    for (int s0 = it.y; s0 < it.z; s0 += CB, buf ^= 1) {
        const int nb = min(CB, it.z - s0);
        const bool more = s0 + CB < it.z;
        if (more) { stage(buf ^ 1, s0 + CB); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
#pragma unroll 1                                             // one copy of the straight-line body: four copies (65 KB of code at P = 8) thrash the instruction cache
        for (int c_ = 0; c_ < nb; c_++) {
            const double4 c = s_c[buf][c_];
            const T dx = (T)(X.x - c.x), dy = (T)(X.y - c.y), dz = (T)(X.z - c.z);
            if constexpr (TWIN && sizeof(T) == 4) {
                float va, vb;
                f2_unpack(m2p_twin_packed<P>(dx, dy, dz, (const float *)s_W[buf][c_], (float)kappaA, (float)kscaledA,
                                             (float)kappaB, (float)kscaledB), va, vb);
                accA += (double)va; accB += (double)vb;
            } else {
                T q[P + 1][NS];
                m2p_q<P, NS, T>(dx, dy, dz, s_W[buf][c_], q);
                const T r2 = dx * dx + dy * dy + dz * dz;
                const T rinv = Real<T>::rsqrt_(r2), rinv2 = rinv * rinv, r = r2 * rinv;
                accA += (double)m2p_radial<P, NS, T>(r, rinv, rinv2, (T)kappaA, (T)kscaledA, q, 0);
                if (TWIN) accB += (double)m2p_radial<P, NS, T>(r, rinv, rinv2, (T)kappaB, (T)kscaledB, q, NS - 1);
            }
        }
        __syncthreads();                                     // buf is refilled two iterations from now
    }
    if (ok) {
        atomicAdd(outA + t, accA);
        if (TWIN) atomicAdd(outB + t, accB);
    }
}

// ------------------------------------------------------------------------------------------------------
// fp32 twin regions, two targets per thread.  The kernel above is bound by the shared-memory data pipe, not by
// issue or the FMA pipe (ncu: l1tex__data_pipe_lsu_wavefronts 79 % of peak while active; every broadcast
// LDS.128 is two wavefronts for four W): with two targets in a thread each W read feeds twice the FMAs.  One
// warp per 64-target group; the monomials of the two targets travel as one packed pair.
template <int P>
__device__ __forceinline__ void m2p_twin_packed2(f2_t dx, f2_t dy, f2_t dz, const float *__restrict__ w, f2_t (&qa)[P + 1],
                                                 f2_t (&qb)[P + 1])
{
#pragma unroll
    for (int m = 0; m <= P; m++) { qa[m] = 0; qb[m] = 0; }
    int idx = 0;
    float4 cur = make_float4(0.f, 0.f, 0.f, 0.f);
    f2_t px = f2_pack(1.f, 1.f);
#pragma unroll
    for (int ex = 0; ex <= P; ex++) {
        f2_t pxy = px;
#pragma unroll
        for (int ey = 0; ey <= P - ex; ey++) {
            f2_t mono = pxy;
#pragma unroll
            for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++) {
                const int t = ex + ey + ez;
                float ma, mb;
                f2_unpack(mono, ma, mb);
                const f2_t m2a = f2_pack(ma, ma), m2b = f2_pack(mb, mb);
#pragma unroll
                for (int J = 0; J <= (P - t) / 2; J++) {
                    if (idx % 2 == 0) cur = *(const float4 *)(w + 2 * idx);
                    const f2_t w2 = idx % 2 == 0 ? f2_pack(cur.x, cur.y) : f2_pack(cur.z, cur.w);
                    qa[t + J] = f2_fma(w2, m2a, qa[t + J]);
                    qb[t + J] = f2_fma(w2, m2b, qb[t + J]);
                    idx++;
                }
                mono = f2_mul(mono, dz);
            }
            pxy = f2_mul(pxy, dy);
        }
        px = f2_mul(px, dx);
    }
}

// (sum_m F_A^(m) Q_m^A, sum_m F_B^(m) Q_m^B) of one target from its packed accumulators
template <int P>
__device__ __forceinline__ f2_t m2p_radial_packed(float dx, float dy, float dz, const f2_t (&q)[P + 1], float kappaA, float ksA,
                                                  float kappaB, float ksB)
{
    const float r2 = dx * dx + dy * dy + dz * dz;
    const float rinv = Real<float>::rsqrt_(r2), rinv2 = rinv * rinv, r = r2 * rinv;
    const float EA = kappaA != 0.f ? Real<float>::exp_neg(ksA, r) : 1.f, EB = kappaB != 0.f ? Real<float>::exp_neg(ksB, r) : 1.f;
    const f2_t ri2 = f2_pack(rinv2, rinv2), kap = f2_pack(kappaA, kappaB), k2 = f2_mul(kap, kap);
    f2_t gm = f2_mul(f2_pack(EA, EB), f2_pack(rinv, rinv));                                    // F^(0)
    f2_t acc = f2_mul(gm, q[0]);
    if (P >= 1) {
        const float nr3 = -rinv * rinv2;
        f2_t g = f2_mul(f2_mul(f2_pack(EA, EB), f2_fma(kap, f2_pack(r, r), f2_pack(1.f, 1.f))), f2_pack(nr3, nr3));   // F^(1)
        acc = f2_fma(g, q[1], acc);
#pragma unroll
        for (int m = 1; m < P; m++) {
            const float c = -(float)(2 * m + 1);
            const f2_t gn = f2_mul(f2_fma(g, f2_pack(c, c), f2_mul(k2, gm)), ri2);             // -[(2m+1) g - k^2 gm] / r^2
            gm = g; g = gn;
            acc = f2_fma(g, q[m + 1], acc);
        }
    }
    return acc;
}

#define M2P2_THREADS (PYGBE_TG_M2P / 2)
// register-cap experiment (-DM2P2_MINB=<CTAs per SM>): caps lose -- 96 regs 0.0533 ms, 80 regs 0.0554, 72 regs 0.0571,
// 64 regs 0.0584 (P = 6, config 1) -- and even a minimum of 1 changes ptxas's allocation (138 regs, 0.0575 ms)
#ifdef M2P2_MINB
#define M2P2_BOUNDS __launch_bounds__(M2P2_THREADS, M2P2_MINB)
#else
#define M2P2_BOUNDS __launch_bounds__(M2P2_THREADS)
#endif
template <int P>
__global__ void M2P2_BOUNDS
k_m2p_twin2(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
            const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const float *__restrict__ wc,
            double kappaA, double kscaledA, double kappaB, double kscaledB, double *__restrict__ outA, double *__restrict__ outB)
{
    constexpr int STRIDE = m2p_stride(P, true);
    constexpr int CH = STRIDE / 4;                           // 16-byte chunks per cell
    constexpr int CBW = 12288 / (STRIDE * 4);
    constexpr int CB = CBW < 1 ? 1 : (CBW > 4 ? 4 : CBW);
    __shared__ __align__(16) float s_W[2][CB][STRIDE];
    __shared__ __align__(16) double4 s_c[2][CB];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t0 = it.x * PYGBE_TG_M2P + threadIdx.x, t1 = t0 + M2P2_THREADS;
    const bool ok0 = t0 < np, ok1 = t1 < np;
    const double4 X0 = ok0 ? tpos[t0] : make_double4(1e30, 1e30, 1e30, 0), X1 = ok1 ? tpos[t1] : make_double4(1e30, 1e30, 1e30, 0);
    const float kA = (float)kappaA, ksA = (float)kscaledA, kB = (float)kappaB, ksB = (float)kscaledB;
    double aA0 = 0.0, aB0 = 0.0, aA1 = 0.0, aB1 = 0.0;
    auto stage = [&](int buf, int s0) {
        const int nb = min(CB, it.z - s0);
        for (int i = threadIdx.x; i < nb * CH; i += M2P2_THREADS) {
            const int c_ = i / CH, j = i - c_ * CH;
            cp_async16(&s_W[buf][c_][j * 4], wc + (long)m2p_cell[s0 + c_] * STRIDE + j * 4);
        }
        if (threadIdx.x < nb * 2) {
            const int c_ = threadIdx.x >> 1, hf = threadIdx.x & 1;
            cp_async16((char *)&s_c[buf][c_] + 16 * hf, (const char *)(cgeo + m2p_cell[s0 + c_]) + 16 * hf);
        }
        cp_async_commit();
    };
    stage(0, it.y);
    int buf = 0;
    for (int s0 = it.y; s0 < it.z; s0 += CB, buf ^= 1) {
        const int nb = min(CB, it.z - s0);
        const bool more = s0 + CB < it.z;
        if (more) { stage(buf ^ 1, s0 + CB); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
#pragma unroll 1                                             // one copy of the straight-line body: four copies (65 KB of code at P = 8) thrash the instruction cache
        for (int c_ = 0; c_ < nb; c_++) {
            const double4 c = s_c[buf][c_];
            const float dx0 = (float)(X0.x - c.x), dy0 = (float)(X0.y - c.y), dz0 = (float)(X0.z - c.z);
            const float dx1 = (float)(X1.x - c.x), dy1 = (float)(X1.y - c.y), dz1 = (float)(X1.z - c.z);
            f2_t qa[P + 1], qb[P + 1];
            m2p_twin_packed2<P>(f2_pack(dx0, dx1), f2_pack(dy0, dy1), f2_pack(dz0, dz1), s_W[buf][c_], qa, qb);
            float va, vb;
            f2_unpack(m2p_radial_packed<P>(dx0, dy0, dz0, qa, kA, ksA, kB, ksB), va, vb);
            aA0 += (double)va; aB0 += (double)vb;
            f2_unpack(m2p_radial_packed<P>(dx1, dy1, dz1, qb, kA, ksA, kB, ksB), va, vb);
            aA1 += (double)va; aB1 += (double)vb;
        }
        __syncthreads();                                     // buf is refilled two iterations from now
    }
    if (ok0) { atomicAdd(outA + t0, aA0); atomicAdd(outB + t0, aB0); }
    if (ok1) { atomicAdd(outA + t1, aA1); atomicAdd(outB + t1, aB1); }
}

// fp32, a tree without twin, two targets per thread: the pair is (target 0, target 1) -- packed monomials,
// packed accumulators Q_m, W as the broadcast operand -- including the radial part.
template <int P>
__global__ void M2P2_BOUNDS
k_m2p_single2(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
              const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const float *__restrict__ wc,
              double kappa, double kscaled, double *__restrict__ out)
{
    constexpr int STRIDE = m2p_stride(P, false);
    constexpr int CH = STRIDE / 4;                           // 16-byte chunks per cell
    constexpr int CBW = 12288 / (STRIDE * 4);
    constexpr int CB = CBW < 1 ? 1 : (CBW > 4 ? 4 : CBW);
    __shared__ __align__(16) float s_W[2][CB][STRIDE];
    __shared__ __align__(16) double4 s_c[2][CB];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t0 = it.x * PYGBE_TG_M2P + threadIdx.x, t1 = t0 + M2P2_THREADS;
    const bool ok0 = t0 < np, ok1 = t1 < np;
    const double4 X0 = ok0 ? tpos[t0] : make_double4(1e30, 1e30, 1e30, 0), X1 = ok1 ? tpos[t1] : make_double4(1e30, 1e30, 1e30, 0);
    const float kap = (float)kappa, ks = (float)kscaled;
    const f2_t kap2 = f2_pack(kap, kap), k2 = f2_pack(kap * kap, kap * kap), one2 = f2_pack(1.f, 1.f);
    double a0 = 0.0, a1 = 0.0;
    auto stage = [&](int buf, int s0) {
        const int nb = min(CB, it.z - s0);
        for (int i = threadIdx.x; i < nb * CH; i += M2P2_THREADS) {
            const int c_ = i / CH, j = i - c_ * CH;
            cp_async16(&s_W[buf][c_][j * 4], wc + (long)m2p_cell[s0 + c_] * STRIDE + j * 4);
        }
        if (threadIdx.x < nb * 2) {
            const int c_ = threadIdx.x >> 1, hf = threadIdx.x & 1;
            cp_async16((char *)&s_c[buf][c_] + 16 * hf, (const char *)(cgeo + m2p_cell[s0 + c_]) + 16 * hf);
        }
        cp_async_commit();
    };
    stage(0, it.y);
    int buf = 0;
    for (int s0 = it.y; s0 < it.z; s0 += CB, buf ^= 1) {
        const int nb = min(CB, it.z - s0);
        const bool more = s0 + CB < it.z;
        if (more) { stage(buf ^ 1, s0 + CB); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
#pragma unroll 1                                             // one copy of the straight-line body: four copies (65 KB of code at P = 8) thrash the instruction cache
        for (int c_ = 0; c_ < nb; c_++) {
            const double4 c = s_c[buf][c_];
            const f2_t dx = f2_pack((float)(X0.x - c.x), (float)(X1.x - c.x)), dy = f2_pack((float)(X0.y - c.y), (float)(X1.y - c.y)),
                       dz = f2_pack((float)(X0.z - c.z), (float)(X1.z - c.z));
            const float *w = s_W[buf][c_];
            f2_t q[P + 1];
#pragma unroll
            for (int m = 0; m <= P; m++) q[m] = 0;
            int idx = 0;
            float cur[4] = {0.f, 0.f, 0.f, 0.f};
            f2_t px = one2;
#pragma unroll
            for (int ex = 0; ex <= P; ex++) {
                f2_t pxy = px;
#pragma unroll
                for (int ey = 0; ey <= P - ex; ey++) {
                    f2_t mono = pxy;
#pragma unroll
                    for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++) {
                        const int t = ex + ey + ez;
#pragma unroll
                        for (int J = 0; J <= (P - t) / 2; J++) {
                            if (idx % 4 == 0) Chunk<float>::get(w + idx, cur);
                            q[t + J] = f2_fma(f2_pack(cur[idx % 4], cur[idx % 4]), mono, q[t + J]);
                            idx++;
                        }
                        mono = f2_mul(mono, dz);
                    }
                    pxy = f2_mul(pxy, dy);
                }
                px = f2_mul(px, dx);
            }
            // radial part, both targets at once
            const f2_t r2 = f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx)));
            float ra, rb;
            f2_unpack(r2, ra, rb);
            const f2_t rinv = f2_pack(Real<float>::rsqrt_(ra), Real<float>::rsqrt_(rb)), rinv2 = f2_mul(rinv, rinv), r = f2_mul(r2, rinv);
            f2_t E = one2;
            if (kap != 0.f) { f2_unpack(r, ra, rb); E = f2_pack(Real<float>::exp_neg(ks, ra), Real<float>::exp_neg(ks, rb)); }
            f2_t gm = f2_mul(E, rinv);                                                        // F^(0)
            f2_t acc = f2_mul(gm, q[0]);
            if (P >= 1) {
                f2_t g = f2_mul(f2_mul(E, f2_fma(kap2, r, one2)), f2_mul(f2_sub(0, rinv), rinv2));   // F^(1)
                acc = f2_fma(g, q[1], acc);
#pragma unroll
                for (int m = 1; m < P; m++) {
                    const float cc = -(float)(2 * m + 1);
                    const f2_t gn = f2_mul(f2_fma(g, f2_pack(cc, cc), f2_mul(k2, gm)), rinv2);
                    gm = g; g = gn;
                    acc = f2_fma(g, q[m + 1], acc);
                }
            }
            float va, vb;
            f2_unpack(acc, va, vb);
            a0 += (double)va; a1 += (double)vb;
        }
        __syncthreads();                                     // buf is refilled two iterations from now
    }
    if (ok0) atomicAdd(out + t0, a0);
    if (ok1) atomicAdd(out + t1, a1);
}

// ------------------------------------------------------------------------------------------------------
// fp64, two targets per thread (one warp per 64-target group).  The one-target kernel above reads one W per
// DFMA through 16-byte broadcasts and sits on the shared-memory data pipe like its fp32 predecessor did (52 %
// of the fp64 pipe at config 1); with two targets every W read feeds two DFMAs.
template <int P, int NS>
__device__ __forceinline__ void m2p_q2(double dx0, double dy0, double dz0, double dx1, double dy1, double dz1,
                                       const double *__restrict__ w, double (&q0)[P + 1][NS], double (&q1)[P + 1][NS])
{
    double cur[2];
    int idx = 0;
#pragma unroll
    for (int m = 0; m <= P; m++)
#pragma unroll
        for (int s = 0; s < NS; s++) { q0[m][s] = 0.0; q1[m][s] = 0.0; }
    double px0 = 1.0, px1 = 1.0;
#pragma unroll
    for (int ex = 0; ex <= P; ex++) {
        double pxy0 = px0, pxy1 = px1;
#pragma unroll
        for (int ey = 0; ey <= P - ex; ey++) {
            double m0 = pxy0, m1 = pxy1;
#pragma unroll
            for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++) {
                const int t = ex + ey + ez;
#pragma unroll
                for (int J = 0; J <= (P - t) / 2; J++) {
#pragma unroll
                    for (int s = 0; s < NS; s++) {
                        if (idx % 2 == 0) Chunk<double>::get(w + idx, cur);
                        q0[t + J][s] = fma(cur[idx % 2], m0, q0[t + J][s]);
                        q1[t + J][s] = fma(cur[idx % 2], m1, q1[t + J][s]);
                        idx++;
                    }
                }
                m0 *= dz0; m1 *= dz1;
            }
            pxy0 *= dy0; pxy1 *= dy1;
        }
        px0 *= dx0; px1 *= dx1;
    }
}

template <int P, bool TWIN>
__global__ void __launch_bounds__(M2P2_THREADS)
k_m2p_dbl2(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
           const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const double *__restrict__ wc,
           double kappaA, double kappaB, double *__restrict__ outA, double *__restrict__ outB)
{
    constexpr int NS = TWIN ? 2 : 1;
    constexpr int STRIDE = m2p_stride(P, TWIN);
    constexpr int CH = STRIDE / 2;                           // 16-byte chunks per cell
    constexpr int CBW = 12288 / (STRIDE * 8);
    constexpr int CB = CBW < 1 ? 1 : (CBW > 4 ? 4 : CBW);
    __shared__ __align__(16) double s_W[2][CB][STRIDE];
    __shared__ __align__(16) double4 s_c[2][CB];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t0 = it.x * PYGBE_TG_M2P + threadIdx.x, t1 = t0 + M2P2_THREADS;
    const bool ok0 = t0 < np, ok1 = t1 < np;
    const double4 X0 = ok0 ? tpos[t0] : make_double4(1e30, 1e30, 1e30, 0), X1 = ok1 ? tpos[t1] : make_double4(1e30, 1e30, 1e30, 0);
    double aA0 = 0.0, aB0 = 0.0, aA1 = 0.0, aB1 = 0.0;
    auto stage = [&](int buf, int s0) {
        const int nb = min(CB, it.z - s0);
        for (int i = threadIdx.x; i < nb * CH; i += M2P2_THREADS) {
            const int c_ = i / CH, j = i - c_ * CH;
            cp_async16(&s_W[buf][c_][j * 2], wc + (long)m2p_cell[s0 + c_] * STRIDE + j * 2);
        }
        if (threadIdx.x < nb * 2) {
            const int c_ = threadIdx.x >> 1, hf = threadIdx.x & 1;
            cp_async16((char *)&s_c[buf][c_] + 16 * hf, (const char *)(cgeo + m2p_cell[s0 + c_]) + 16 * hf);
        }
        cp_async_commit();
    };
    stage(0, it.y);
    int buf = 0;
    for (int s0 = it.y; s0 < it.z; s0 += CB, buf ^= 1) {
        const int nb = min(CB, it.z - s0);
        const bool more = s0 + CB < it.z;
        if (more) { stage(buf ^ 1, s0 + CB); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
#pragma unroll 1                                             // one copy of the straight-line body (instruction cache)
        for (int c_ = 0; c_ < nb; c_++) {
            const double4 c = s_c[buf][c_];
            const double dx0 = X0.x - c.x, dy0 = X0.y - c.y, dz0 = X0.z - c.z;
            const double dx1 = X1.x - c.x, dy1 = X1.y - c.y, dz1 = X1.z - c.z;
            double q0[P + 1][NS], q1[P + 1][NS];
            m2p_q2<P, NS>(dx0, dy0, dz0, dx1, dy1, dz1, s_W[buf][c_], q0, q1);
            {
                const double r2 = dx0 * dx0 + dy0 * dy0 + dz0 * dz0;
                const double rinv = Real<double>::rsqrt_(r2), rinv2 = rinv * rinv, r = r2 * rinv;
                aA0 += m2p_radial<P, NS, double>(r, rinv, rinv2, kappaA, kappaA, q0, 0);
                if (TWIN) aB0 += m2p_radial<P, NS, double>(r, rinv, rinv2, kappaB, kappaB, q0, NS - 1);
            }
            {
                const double r2 = dx1 * dx1 + dy1 * dy1 + dz1 * dz1;
                const double rinv = Real<double>::rsqrt_(r2), rinv2 = rinv * rinv, r = r2 * rinv;
                aA1 += m2p_radial<P, NS, double>(r, rinv, rinv2, kappaA, kappaA, q1, 0);
                if (TWIN) aB1 += m2p_radial<P, NS, double>(r, rinv, rinv2, kappaB, kappaB, q1, NS - 1);
            }
        }
        __syncthreads();                                     // buf is refilled two iterations from now
    }
    if (ok0) { atomicAdd(outA + t0, aA0); if (TWIN) atomicAdd(outB + t0, aB0); }
    if (ok1) { atomicAdd(outA + t1, aA1); if (TWIN) atomicAdd(outB + t1, aB1); }
}

// ------------------------------------------------------------------------------------------------------
// Laplace regions without a twin (kappa = 0: the protein interior and the Stern layer of the multi-surface
// problems): the same truncated series in a form that needs no monomials and no radial
// recurrence.  For G = 1/r every radial derivative is a pure power, F^(m)(s) = (-1)^m (2m-1)!! / r^(2m+1), so
// with the inverted offset u = d / r^2 (|u| = 1/r, d^e = u^e r^(2|e|), r^(-2J) = (ux^2 + uy^2 + uz^2)^J)
//     sum_{|k| <= P} a^k M^k  =  (1/r) sum_{|f| <= P} C_f u^f,
//     C_f = sum_{2i <= f, e = f - 2i, J = |i|}  (J! / i!)  sum_{|j| = J} (-1)^J (2(|e| + J) - 1)!! / (e! 2^J j!)  M^(e + 2j):
// ONE trivariate polynomial of degree P with Nc coefficients per cell (the detraced multipoles; degree-n
// coefficients come from degree-n moments only), evaluated by nested Horner steps in uz, uy, ux: Nc - 1 FMAs per
// (target, cell) -- 164 at P = 8 against 164 multiplies + 295 FMAs of the regrouped form above.  The C_f are formed
// where the W are (P2M / M2M epilogue, farfield.cuh; table built at create, tables.cuh), stored in Horner order
// (ex, ey, ez descending) and normalised by the cell edge a, C'_f = C_f / a^|f| with u' = a d / r^2 (|u'| = a / r
// < theta), so that every intermediate is O(monopole) whatever the units.
//
// Four targets per thread: each coefficient read from shared memory feeds four FMAs (fp32: two packed FFMA2),
// because a broadcast LDS.128 costs two wavefronts for four coefficients and one coefficient per FMA pair would
// tie the shared-memory pipe with the FMA pipe.  A CTA of one warp serves one 64-target group: thread
// (sub, l16) = (tid / 16, tid % 16) owns targets l16 + 16 k, k = 0..3, and the cells sub, sub + 2, ... of every
// staged batch (two cells in flight per warp, warp-level synchronisation only); the partial sums per target
// meet in shared memory at the end of the item.  Offsets are
// formed from group-relative coordinates: x - G in T per target, c - G computed in fp64 and rounded once per
// staged cell, so that the fp32 path subtracts numbers of the size of r, not of the molecule (relative error of
// d about 1e-7; no fp64 arithmetic or conversions in the loop over cells except the accumulation).
static inline __host__ __device__ constexpr int m2p_lap_stride(int P) { return ((P + 1) * (P + 2) * (P + 3) / 6 + 3) / 4 * 4; }

template <typename T> struct LapVec;
template <> struct LapVec<float> {
    f2_t lo, hi;                                                     // targets (0, 1) and (2, 3)
    static __device__ __forceinline__ LapVec make(float a, float b, float c, float d) { LapVec v; v.lo = f2_pack(a, b); v.hi = f2_pack(c, d); return v; }
    static __device__ __forceinline__ LapVec set(float w) { LapVec v; v.lo = f2_pack(w, w); v.hi = v.lo; return v; }
    static __device__ __forceinline__ LapVec fmaw(const LapVec &a, const LapVec &u, float w)      // a u + w
    { const f2_t w2 = f2_pack(w, w); LapVec v; v.lo = f2_fma(a.lo, u.lo, w2); v.hi = f2_fma(a.hi, u.hi, w2); return v; }
    static __device__ __forceinline__ LapVec fmav(const LapVec &a, const LapVec &u, const LapVec &c)   // a u + c
    { LapVec v; v.lo = f2_fma(a.lo, u.lo, c.lo); v.hi = f2_fma(a.hi, u.hi, c.hi); return v; }
    static __device__ __forceinline__ LapVec mul(const LapVec &a, const LapVec &b) { LapVec v; v.lo = f2_mul(a.lo, b.lo); v.hi = f2_mul(a.hi, b.hi); return v; }
    static __device__ __forceinline__ LapVec sub(const LapVec &a, float c) { const f2_t c2 = f2_pack(c, c); LapVec v; v.lo = f2_sub(a.lo, c2); v.hi = f2_sub(a.hi, c2); return v; }
    __device__ __forceinline__ void get(float (&o)[4]) const { f2_unpack(lo, o[0], o[1]); f2_unpack(hi, o[2], o[3]); }
};
template <> struct LapVec<double> {
    double v[4];
    static __device__ __forceinline__ LapVec make(double a, double b, double c, double d) { LapVec r; r.v[0] = a; r.v[1] = b; r.v[2] = c; r.v[3] = d; return r; }
    static __device__ __forceinline__ LapVec set(double w) { return make(w, w, w, w); }
    static __device__ __forceinline__ LapVec fmaw(const LapVec &a, const LapVec &u, double w)
    { LapVec r;
#pragma unroll
      for (int i = 0; i < 4; i++) r.v[i] = fma(a.v[i], u.v[i], w);
      return r; }
    static __device__ __forceinline__ LapVec fmav(const LapVec &a, const LapVec &u, const LapVec &c)
    { LapVec r;
#pragma unroll
      for (int i = 0; i < 4; i++) r.v[i] = fma(a.v[i], u.v[i], c.v[i]);
      return r; }
    static __device__ __forceinline__ LapVec mul(const LapVec &a, const LapVec &b)
    { LapVec r;
#pragma unroll
      for (int i = 0; i < 4; i++) r.v[i] = a.v[i] * b.v[i];
      return r; }
    static __device__ __forceinline__ LapVec sub(const LapVec &a, double c)
    { LapVec r;
#pragma unroll
      for (int i = 0; i < 4; i++) r.v[i] = a.v[i] - c;
      return r; }
    __device__ __forceinline__ void get(double (&o)[4]) const
    {
#pragma unroll
        for (int i = 0; i < 4; i++) o[i] = v[i];
    }
};

// sum_f C'_f u^f by nested Horner steps; w: the cell's coefficients in Horner order (ex, ey, ez descending)
template <int P, typename T>
__device__ __forceinline__ LapVec<T> lap_poly(const LapVec<T> &ux, const LapVec<T> &uy, const LapVec<T> &uz, const T *__restrict__ w)
{
    typedef LapVec<T> V;
    constexpr int EPC = Chunk<T>::N;
    T cur[EPC];
    int idx = 0;
    V ax = V::set(T(0));
#pragma unroll
    for (int ex = P; ex >= 0; ex--) {
        V ay = V::set(T(0));
#pragma unroll
        for (int ey = P - ex; ey >= 0; ey--) {
            V az = V::set(T(0));
#pragma unroll
            for (int ez = P - ex - ey; ez >= 0; ez--) {
                if (idx % EPC == 0) Chunk<T>::get(w + idx, cur);
                const T c = cur[idx % EPC];
                idx++;
                if (ez == P - ex - ey) az = V::set(c); else az = V::fmaw(az, uz, c);
            }
            if (ey == P - ex) ay = az; else ay = V::fmav(ay, uy, az);
        }
        if (ex == P) ax = ay; else ax = V::fmav(ax, ux, ay);
    }
    return ax;
}

#ifndef M2PL_THREADS
#define M2PL_THREADS 32                                              // one warp: two cells in flight, no CTA barrier
#endif
#define M2PL_NSUB (M2PL_THREADS / 16)
// cells per staged batch: a multiple of the subs, at most 12, two buffers within M2PL_SMEM bytes of static shared memory
#ifndef M2PL_SMEM
#define M2PL_SMEM 12288
#endif
template <int P, typename T> struct LapBatch {
    static constexpr int ROW = m2p_lap_stride(P) * (int)sizeof(T);
    static constexpr int FIT = M2PL_SMEM / ROW / 4 * 4;
    static constexpr int CB = FIT < 4 ? 4 : (FIT > 12 ? 12 : FIT);
};
#ifdef M2PL_MINB
#define M2PL_BOUNDS __launch_bounds__(M2PL_THREADS, M2PL_MINB)
#else
#define M2PL_BOUNDS __launch_bounds__(M2PL_THREADS)
#endif
__device__ __forceinline__ void lap_sync()
{
#if M2PL_THREADS == 32
    __syncwarp();
#else
    __syncthreads();
#endif
}
template <int P, typename T>
__global__ void M2PL_BOUNDS
k_m2p_lap(const int *__restrict__ skip, const int4 *__restrict__ items, const int *__restrict__ m2p_cell, int np,
          const double4 *__restrict__ tpos, const double4 *__restrict__ ggeo, const double4 *__restrict__ cgeo,
          const T *__restrict__ wc, double *__restrict__ out)
{
    typedef LapVec<T> V;
    typedef typename Real<T>::vec4 V4;
    constexpr int STRIDE = m2p_lap_stride(P);
    constexpr int EPC = 16 / (int)sizeof(T);
    constexpr int CH = STRIDE / EPC;                                 // 16-byte chunks per cell
    constexpr int M2PL_CB = LapBatch<P, T>::CB;
    __shared__ __align__(16) T s_W[2][M2PL_CB][STRIDE];
    __shared__ __align__(16) V4 s_c[2][M2PL_CB];                     // (c - G, edge)
    __shared__ double s_red[M2PL_NSUB][PYGBE_TG_M2P];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int sub = threadIdx.x >> 4, l16 = threadIdx.x & 15;
    const double4 G = ggeo[2 * it.x];
    T xt[4], yt[4], zt[4];
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const int t = it.x * PYGBE_TG_M2P + l16 + 16 * k;
        const double4 X = t < np ? tpos[t] : make_double4(1e30, 1e30, 1e30, 0);
        xt[k] = (T)(X.x - G.x); yt[k] = (T)(X.y - G.y); zt[k] = (T)(X.z - G.z);
    }
    const V X4 = V::make(xt[0], xt[1], xt[2], xt[3]), Y4 = V::make(yt[0], yt[1], yt[2], yt[3]), Z4 = V::make(zt[0], zt[1], zt[2], zt[3]);
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    double4 pc = make_double4(0, 0, 0, 1);                           // centre of this thread's cell of the batch after the staged one
    auto prefetch = [&](int s0) { if (threadIdx.x < M2PL_CB && s0 + (int)threadIdx.x < it.z) pc = cgeo[m2p_cell[s0 + threadIdx.x]]; };
    auto stage = [&](int buf, int s0) {
        const int nb = min(M2PL_CB, it.z - s0);
        for (int i = threadIdx.x; i < nb * CH; i += M2PL_THREADS) {
            const int c_ = i / CH, j = i - c_ * CH;
            cp_async16(&s_W[buf][c_][j * EPC], wc + (long)m2p_cell[s0 + c_] * STRIDE + j * EPC);
        }
        if ((int)threadIdx.x < nb) {
            V4 v; v.x = (T)(pc.x - G.x); v.y = (T)(pc.y - G.y); v.z = (T)(pc.z - G.z); v.w = (T)pc.w;
            s_c[buf][threadIdx.x] = v;
        }
        cp_async_commit();
    };
    prefetch(it.y);
    stage(0, it.y);
    prefetch(it.y + M2PL_CB);
    int buf = 0;
    for (int s0 = it.y; s0 < it.z; s0 += M2PL_CB, buf ^= 1) {
        const int nb = min(M2PL_CB, it.z - s0);
        const bool more = s0 + M2PL_CB < it.z;
        if (more) { stage(buf ^ 1, s0 + M2PL_CB); prefetch(s0 + 2 * M2PL_CB); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        lap_sync();
#pragma unroll 1                                             // one copy of the straight-line body (instruction cache)
        for (int c_ = sub; c_ < nb; c_ += M2PL_NSUB) {
            const V4 c = s_c[buf][c_];
            const V dx = V::sub(X4, c.x), dy = V::sub(Y4, c.y), dz = V::sub(Z4, c.z);
            const V r2 = V::fmav(dz, dz, V::fmav(dy, dy, V::mul(dx, dx)));
            T r2s[4], ri[4], sc[4];
            r2.get(r2s);
#pragma unroll
            for (int k = 0; k < 4; k++) { ri[k] = Real<T>::rsqrt_(r2s[k]); sc[k] = c.w * (ri[k] * ri[k]); }
            const V S = V::make(sc[0], sc[1], sc[2], sc[3]);
            const V p = lap_poly<P, T>(V::mul(dx, S), V::mul(dy, S), V::mul(dz, S), s_W[buf][c_]);
            T pv[4];
            p.get(pv);
#pragma unroll
            for (int k = 0; k < 4; k++) acc[k] += (double)(pv[k] * ri[k]);
        }
        lap_sync();                                          // buf is refilled two iterations from now
    }
#pragma unroll
    for (int k = 0; k < 4; k++) s_red[sub][l16 + 16 * k] = acc[k];
    lap_sync();
    for (int i = threadIdx.x; i < PYGBE_TG_M2P; i += M2PL_THREADS) {
        const int t = it.x * PYGBE_TG_M2P + i;
        double v = 0.0;
#pragma unroll
        for (int q = 0; q < M2PL_NSUB; q++) v += s_red[q][i];
        if (t < np) atomicAdd(out + t, v);
    }
}
