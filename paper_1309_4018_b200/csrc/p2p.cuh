// p2p.cuh -- the direct near field P2P (a7): "The final step is to directly compute
// interactions for boxes that are too close", :163 "quadrature points serve as sources, collocation
// points as targets".
//
// One kernel template covers
//   T = double : fp64 arithmetic on absolute coordinates (direct mode parity 1e-11);
//   T = float  : fp32 arithmetic on coordinates relative to an anchor cell (absolute fp32
//                coordinates lose 6e-6 in the near sums, cell-local ones 2e-8), rsqrt / ex2 on the SFU,
//                per-tile fp32 partial sums added into fp64 accumulators;
//   TWIN       : the two regions on either side of the same surfaces (eq. 10's Laplace and Yukawa rows)
//                evaluated in one pass: they share d, r^2, 1/r, n.d and differ only by constants
//                (region B's charges are rV * mV and -mK) and by the screening factor.
// Per pair, with d = x - y, t = (mK.d)/r^2 (1/(4 pi) is in the weights):
//   Laplace  (mV - t)/r ;   Yukawa  (mV - t (1 + kappa r)) exp(-kappa r)/r       (eq. 2 / 9)
// A pair at zero distance (K = 1, 4, 7 have a node at the collocation point of the self panel, reading
// A5) contributes nothing: the self panel is replaced by the semi-analytic correction (a8).
#pragma once
#include "common.cuh"
#include "mathx.cuh"
#include "m2p.cuh"       // cp_async helpers

#define P2P_TILE 128

// fp32 source coordinates relative to the centre of the panel's anchor cell (create time, mixed precision).
// The subtraction is done in fp64 and rounded once, exactly as the kernel re-bases the targets, so the
// collocation point of a panel and a Gauss node placed on it give d = 0 exactly.
__global__ void k_make_sposf(int np, int K, const int *__restrict__ panel_anchor, const double4 *__restrict__ cgeo,
                             const double4 *__restrict__ spos, float4 *__restrict__ sposf)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const double4 an = cgeo[panel_anchor[p]];
    for (int g = 0; g < K; g++) {
        double4 s = spos[(long)p * K + g];
        sposf[(long)p * K + g] = make_float4((float)(s.x - an.x), (float)(s.y - an.y), (float)(s.z - an.z), (float)s.w);
    }
}

template <typename T, bool YA, bool TWIN, bool YB>
__device__ __forceinline__ void p2p_pair(T dx, T dy, T dz, T mV, T mKx, T mKy, T mKz, T ksA, T kA, T ksB, T kB,
                                         T rV, T &accA, T &accB)
{
    T r2 = dx * dx + dy * dy + dz * dz;
    T rinv = r2 > T(0) ? Real<T>::rsqrt_(r2) : T(0);
    T mKd = mKx * dx + mKy * dy + mKz * dz;
    T t = mKd * (rinv * rinv);
    T r = r2 * rinv;
    if constexpr (YA) {
        T kr = kA * r;
        accA += (mV - (t + t * kr)) * (rinv * Real<T>::exp_neg(ksA, r));
    } else {
        accA += (mV - t) * rinv;
    }
    if constexpr (TWIN) {
        T mVb = rV * mV;                         // region B: charges rV mV and -mK
        if constexpr (YB) {
            T kr = kB * r;
            accB += (mVb + (t + t * kr)) * (rinv * Real<T>::exp_neg(ksB, r));
        } else {
            accB += (mVb + t) * rinv;
        }
    }
}

// Work item = (target group, a run of source tiles).  tile = (first point, number of points <= P2P_TILE,
// anchor cell, -): for T = float the stored source coordinates are relative to the anchor cell's centre and
// the target is re-based per tile in fp64 (3 subtractions per thread per tile), so every fp32 difference is
// between numbers of the size of a cell, not of the molecule.  Tiles are double-buffered with cp.async
// (LDGSTS): while the threads sum one tile, the points, weights and anchor centre of the next stream into
// the other buffer, and the descriptor of the one after is already in registers (the first version staged
// each tile synchronously: 16 % wait + 9 % scoreboard stalls, profiles/r1b_mixed_path.md).
template <typename T, bool YA, bool TWIN, bool YB>
__global__ void __launch_bounds__(PYGBE_TG)
k_p2p(const int *__restrict__ skip, const int4 *__restrict__ items, const int4 *__restrict__ tiles, int np,
      const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo,
      const typename Real<T>::vec4 *__restrict__ pos, const typename Real<T>::vec4 *__restrict__ chg,
      double kappaA, double kappaB, double rV, double *__restrict__ outA, double *__restrict__ outB)
{
    typedef typename Real<T>::vec4 V4;
    constexpr int V4C = (int)sizeof(V4) / 16;                        // 16-byte chunks per point record
    __shared__ __align__(16) V4 s_pos[2][P2P_TILE];
    __shared__ __align__(16) V4 s_chg[2][P2P_TILE];
    __shared__ __align__(16) double4 s_an[2];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t = it.x * PYGBE_TG + threadIdx.x;
    const bool ok = t < np;
    const double4 X = ok ? tpos[t] : make_double4(0, 0, 0, 0);
    const T kA = (T)kappaA, kB = (T)kappaB, ksA = (T)Real<T>::kscale(kappaA), ksB = (T)Real<T>::kscale(kappaB);
    const T rv = (T)rV;
    double accA = 0.0, accB = 0.0;
    auto stage = [&](int buf, const int4 &tl) {
        for (int i = threadIdx.x; i < tl.y * V4C; i += PYGBE_TG) {
            cp_async16((char *)s_pos[buf] + 16 * i, (const char *)(pos + tl.x) + 16 * i);
            cp_async16((char *)s_chg[buf] + 16 * i, (const char *)(chg + tl.x) + 16 * i);
        }
        if (sizeof(T) == 4 && threadIdx.x < 2)
            cp_async16((char *)&s_an[buf] + 16 * threadIdx.x, (const char *)(cgeo + tl.z) + 16 * threadIdx.x);
        cp_async_commit();
    };
    int4 cur = tiles[it.y];
    int4 nxt = it.y + 1 < it.z ? tiles[it.y + 1] : cur;
    stage(0, cur);
    int buf = 0;
    for (int k = it.y; k < it.z; k++, buf ^= 1) {
        const bool more = k + 1 < it.z;
        if (more) { stage(buf ^ 1, nxt); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        const int n = cur.y;
        cur = nxt;
        if (k + 2 < it.z) nxt = tiles[k + 2];
        __syncthreads();
        T x, y, z;
        if constexpr (sizeof(T) == 4) {
            const double4 an = s_an[buf];
            x = (T)(X.x - an.x); y = (T)(X.y - an.y); z = (T)(X.z - an.z);
        } else {
            x = (T)X.x; y = (T)X.y; z = (T)X.z;
        }
        const V4 *sp = s_pos[buf], *sc = s_chg[buf];
        T a0 = T(0), a1 = T(0), b0 = T(0), b1 = T(0);
        int i = 0;
#pragma unroll 2
        for (; i + 1 < n; i += 2) {
            V4 p = sp[i], c = sc[i], p2 = sp[i + 1], c2 = sc[i + 1];
            p2p_pair<T, YA, TWIN, YB>(x - p.x, y - p.y, z - p.z, c.x, c.y, c.z, c.w, ksA, kA, ksB, kB, rv, a0, b0);
            p2p_pair<T, YA, TWIN, YB>(x - p2.x, y - p2.y, z - p2.z, c2.x, c2.y, c2.z, c2.w, ksA, kA, ksB, kB, rv, a1, b1);
        }
        if (i < n) {
            V4 p = sp[i], c = sc[i];
            p2p_pair<T, YA, TWIN, YB>(x - p.x, y - p.y, z - p.z, c.x, c.y, c.z, c.w, ksA, kA, ksB, kB, rv, a0, b0);
        }
        accA += (double)(a0 + a1);
        if constexpr (TWIN) accB += (double)(b0 + b1);
        __syncthreads();                                             // buf is refilled two iterations from now
    }
    if (ok) {
        atomicAdd(outA + t, accA);
        if constexpr (TWIN) atomicAdd(outB + t, accB);
    }
}
