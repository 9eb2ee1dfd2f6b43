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

#ifndef P2P_TILE
#define P2P_TILE 128
#endif

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

// Work item = (target group, a run of source tiles).  tile = (first segment, last segment + 1, anchor cell,
// 2 * points + self flag), segment = (first point, points): the <= P2P_TILE points of a tile are gathered from
// several runs of Morton-consecutive panels of one anchor cell (build_lists.cuh).  For T = float the stored source coordinates are relative to the anchor cell's centre and
// the target is re-based per tile in fp64 (3 subtractions per thread per tile), so every fp32 difference is
// between numbers of the size of a cell, not of the molecule.  Tiles are double-buffered with cp.async
// (LDGSTS): while the threads sum one tile, the points, weights and anchor centre of the next stream into
// the other buffer, and the descriptor of the one after is already in registers (the first version staged
// each tile synchronously: 16 % wait + 9 % scoreboard stalls, profiles/r1b_mixed_path.md).
template <typename T, bool YA, bool TWIN, bool YB>
__global__ void __launch_bounds__(PYGBE_TG)
k_p2p(const int *__restrict__ skip, const int4 *__restrict__ items, const int4 *__restrict__ tiles,
      const int2 *__restrict__ segs, int np,
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
    auto stage = [&](int buf, const int4 &tl) {                      // gather the tile's segments into consecutive slots
        const int lane = threadIdx.x & 31;
        int off = 0;                                                 // points staged so far
        for (int s0 = tl.x; s0 < tl.y; s0 += 32) {
            const int ns = min(32, tl.y - s0);
            const int2 mine = lane < ns ? segs[s0 + lane] : make_int2(0, 0);
            for (int s = 0; s < ns; s++) {
                const int p0 = __shfl_sync(0xffffffffu, mine.x, s), c = __shfl_sync(0xffffffffu, mine.y, s) * V4C;
                for (int i = threadIdx.x; i < 2 * c; i += PYGBE_TG) {
                    if (i < c) cp_async16((char *)(s_pos[buf] + off) + 16 * i, (const char *)(pos + p0) + 16 * i);
                    else cp_async16((char *)(s_chg[buf] + off) + 16 * (i - c), (const char *)(chg + p0) + 16 * (i - c));
                }
                off += c / V4C;
            }
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
        const int n = cur.w >> 1;
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

// ------------------------------------------------------------------------------------------------------
// Mixed precision, K a multiple of 4: the same sums with packed fp32 arithmetic (add / mul / fma .f32x2:
// FADD2 / FMUL2 / FFMA2 on sm_100), two source points per instruction.  The first fp32 kernel was issue-bound
// at 29 instructions per fused pair (profiles/r2a_regrouped_path.md); packing halves the FP32 issue slots (the
// MUFU rsqrt / ex2 and the zero-distance guard stay scalar).  Sources are stored as quads of four consecutive
// Gauss points, structure-of-arrays inside the quad, so that one LDS.128 yields two register pairs:
//   posq[3 q + {0,1,2}] = (x0..x3), (y0..y3), (z0..z3)   relative to the anchor cell centre (create)
//   chgq[4 q + {0,1,2,3}] = (mV0..3), (mKx0..3), (mKy0..3), (mKz0..3)   (k_prep, every matvec)
// Region B's charges are rV mV and -mK: its sum is accumulated as sum (mV + t (1 + kappa r) / rV) w and
// multiplied by rV once at the end.
struct P2PQuadConst {                                                 // loop invariants, already packed
    f2_t nksA, nksB;            // -kappa log2(e) of regions A and B
    f2_t kA;                    // kappa_A
    f2_t sB, cB;                // -1 / rV and -kappa_B / rV
    f2_t tiny;                  // floor of r^2 in the unguarded tiles
};

// two source points (packed) against one target.  GUARD: the tile holds panels of the group's own targets, a
// pair can be at zero distance (reading A5) and must contribute nothing -> select on r^2 > 0 (two scalar ALU
// instructions per pair).  Every other tile takes the unguarded form: r^2 carries a 1e-30 floor inside its
// first FMA (free, far below one ulp of any real r^2), so that points of a degenerate mesh that coincide after
// rounding give a finite value instead of a NaN.
template <bool YA, bool TWIN, bool YB, bool GUARD>
__device__ __forceinline__ void p2p_pair2(f2_t X, f2_t Y, f2_t Z, f2_t px, f2_t py, f2_t pz, f2_t mV, f2_t mKx, f2_t mKy,
                                          f2_t mKz, const P2PQuadConst &k, f2_t &accA, f2_t &accB)
{
    // the offset is taken with the opposite sign, y - x: r^2 is the same and mKd = -(mK . d), which turns the
    // subtraction mV - t of the Laplace term into the addend of an FMA (one instruction less per pair in the
    // single-region Laplace kernel); the constants sB, cB of region B carry the sign as well
    const f2_t dx = f2_sub(px, X), dy = f2_sub(py, Y), dz = f2_sub(pz, Z);
    const f2_t r2 = f2_fma(dz, dz, f2_fma(dy, dy, GUARD ? f2_mul(dx, dx) : f2_fma(dx, dx, k.tiny)));
    const f2_t mKd = f2_fma(mKz, dz, f2_fma(mKy, dy, f2_mul(mKx, dx)));                    // -(mK . d)
    float r2a, r2b, ia, ib;
    f2_unpack(r2, r2a, r2b);
    if constexpr (GUARD) { ia = r2a > 0.f ? Real<float>::rsqrt_(r2a) : 0.f; ib = r2b > 0.f ? Real<float>::rsqrt_(r2b) : 0.f; }
    else { ia = Real<float>::rsqrt_(r2a); ib = Real<float>::rsqrt_(r2b); }
    const f2_t rinv = f2_pack(ia, ib);
    const f2_t rinv2 = f2_mul(rinv, rinv);
    const f2_t t = f2_mul(mKd, rinv2);                                // -(mK . d) / r^2
    const f2_t r = f2_mul(r2, rinv);
    if constexpr (YA) {
        float ea, eb;
        f2_unpack(f2_mul(r, k.nksA), ea, eb);
        asm("ex2.approx.ftz.f32 %0, %0;" : "+f"(ea));
        asm("ex2.approx.ftz.f32 %0, %0;" : "+f"(eb));
        const f2_t u = f2_fma(f2_mul(t, k.kA), r, t);                 // -(mK . d) (1 + kappa r) / r^2
        accA = f2_fma(f2_add(mV, u), f2_mul(rinv, f2_pack(ea, eb)), accA);
    } else if constexpr (TWIN) {
        accA = f2_fma(f2_add(mV, t), rinv, accA);
    } else {
        accA = f2_fma(f2_fma(mKd, rinv2, mV), rinv, accA);            // (mV - (mK . d) / r^2) / r
    }
    if constexpr (TWIN) {
        if constexpr (YB) {
            float ea, eb;
            f2_unpack(f2_mul(r, k.nksB), ea, eb);
            asm("ex2.approx.ftz.f32 %0, %0;" : "+f"(ea));
            asm("ex2.approx.ftz.f32 %0, %0;" : "+f"(eb));
            const f2_t u = f2_mul(t, f2_fma(k.cB, r, k.sB));          // (mK . d) (1 + kappa r) / (r^2 rV): sB, cB are negated
            accB = f2_fma(f2_add(mV, u), f2_mul(rinv, f2_pack(ea, eb)), accB);
        } else {
            accB = f2_fma(f2_fma(t, k.sB, mV), rinv, accB);           // (mV + (mK . d) / (r^2 rV)) / r
        }
    }
}

// one staged tile of nq quads against one target
template <bool YA, bool TWIN, bool YB, bool GUARD>
__device__ __forceinline__ void p2p_quad_tile(const float4 *__restrict__ sp, const float4 *__restrict__ sc, int nq, f2_t X2,
                                              f2_t Y2, f2_t Z2, const P2PQuadConst &kc, f2_t &a0, f2_t &a1, f2_t &b0, f2_t &b1)
{
#ifndef P2PQ_UNROLL
#define P2PQ_UNROLL 2
#endif
    constexpr int UNR = P2PQ_UNROLL;
#pragma unroll UNR
    for (int q = 0; q < nq; q++) {
        const float4 px = sp[3 * q], py = sp[3 * q + 1], pz = sp[3 * q + 2];
        const float4 mV = sc[4 * q], mKx = sc[4 * q + 1], mKy = sc[4 * q + 2], mKz = sc[4 * q + 3];
        p2p_pair2<YA, TWIN, YB, GUARD>(X2, Y2, Z2, f2_pack(px.x, px.y), f2_pack(py.x, py.y), f2_pack(pz.x, pz.y), f2_pack(mV.x, mV.y),
                                       f2_pack(mKx.x, mKx.y), f2_pack(mKy.x, mKy.y), f2_pack(mKz.x, mKz.y), kc, a0, b0);
        p2p_pair2<YA, TWIN, YB, GUARD>(X2, Y2, Z2, f2_pack(px.z, px.w), f2_pack(py.z, py.w), f2_pack(pz.z, pz.w), f2_pack(mV.z, mV.w),
                                       f2_pack(mKx.z, mKx.w), f2_pack(mKy.z, mKy.w), f2_pack(mKz.z, mKz.w), kc, a1, b1);
    }
}

#define P2P_QTILE (P2P_TILE / 4)                                       // quads per tile
template <bool YA, bool TWIN, bool YB>
#ifndef P2PQ_MINB
#define P2PQ_MINB 16                                                  // 64 registers: 16 CTAs per SM (uncapped: 114 / 8; 12: 0.0859, 16: 0.0842, 20: 0.0848 ms)
#endif
__global__ void __launch_bounds__(PYGBE_TG, P2PQ_MINB)
k_p2p_quad(const int *__restrict__ skip, const int4 *__restrict__ items, const int4 *__restrict__ tiles,
           const int2 *__restrict__ segs, int np,
           const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo, const float4 *__restrict__ posq,
           const float4 *__restrict__ chgq, double kappaA, double kappaB, double rV, double *__restrict__ outA,
           double *__restrict__ outB)
{
    __shared__ __align__(16) float4 s_pos[2][3 * P2P_QTILE];
    __shared__ __align__(16) float4 s_chg[2][4 * P2P_QTILE];
    __shared__ __align__(16) double4 s_an[2];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int t = it.x * PYGBE_TG + threadIdx.x;
    const bool ok = t < np;
    const double4 X = ok ? tpos[t] : make_double4(0, 0, 0, 0);
    P2PQuadConst kc;
    {
        const float a = -(float)Real<float>::kscale(kappaA), b = -(float)Real<float>::kscale(kappaB);
        const float s = -(float)(1.0 / rV), c = -(float)(kappaB / rV), ka = (float)kappaA;      // negated: see p2p_pair2
        kc.nksA = f2_pack(a, a); kc.nksB = f2_pack(b, b); kc.kA = f2_pack(ka, ka); kc.sB = f2_pack(s, s); kc.cB = f2_pack(c, c);
        kc.tiny = f2_pack(1e-30f, 1e-30f);
    }
    double accA = 0.0, accB = 0.0;
    auto stage = [&](int buf, const int4 &tl) {                      // segments = (first point, points), multiples of 4
        const int lane = threadIdx.x & 31;
        int qoff = 0;                                                // quads staged so far
        for (int s0 = tl.x; s0 < tl.y; s0 += 32) {
            const int ns = min(32, tl.y - s0);
            const int2 mine = lane < ns ? segs[s0 + lane] : make_int2(0, 0);
            for (int s = 0; s < ns; s++) {
                const int q0 = __shfl_sync(0xffffffffu, mine.x, s) >> 2, nq = __shfl_sync(0xffffffffu, mine.y, s) >> 2;
                for (int i = threadIdx.x; i < 7 * nq; i += PYGBE_TG) {
                    if (i < 3 * nq) cp_async16(&s_pos[buf][3 * qoff + i], posq + 3 * (long)q0 + i);
                    else cp_async16(&s_chg[buf][4 * qoff + i - 3 * nq], chgq + 4 * (long)q0 + i - 3 * nq);
                }
                qoff += nq;
            }
        }
        if (threadIdx.x < 2)
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
        const int nq = cur.w >> 3;
        const bool self = (cur.w & 1) != 0;
        cur = nxt;
        if (k + 2 < it.z) nxt = tiles[k + 2];
        __syncthreads();
        const double4 an = s_an[buf];
        const float x = (float)(X.x - an.x), y = (float)(X.y - an.y), z = (float)(X.z - an.z);
        const f2_t X2 = f2_pack(x, x), Y2 = f2_pack(y, y), Z2 = f2_pack(z, z);
        const float4 *sp = s_pos[buf], *sc = s_chg[buf];
        f2_t a0 = 0, a1 = 0, b0 = 0, b1 = 0;                          // (+0.f, +0.f)
        if (self) p2p_quad_tile<YA, TWIN, YB, true>(sp, sc, nq, X2, Y2, Z2, kc, a0, a1, b0, b1);     // uniform over the CTA
        else p2p_quad_tile<YA, TWIN, YB, false>(sp, sc, nq, X2, Y2, Z2, kc, a0, a1, b0, b1);
        float lo, hi;
        f2_unpack(f2_add(a0, a1), lo, hi);
        accA += (double)(lo + hi);
        if constexpr (TWIN) { f2_unpack(f2_add(b0, b1), lo, hi); accB += (double)(lo + hi); }
        __syncthreads();                                             // buf is refilled two iterations from now
    }
    if (ok) {
        atomicAdd(outA + t, accA);
        if constexpr (TWIN) atomicAdd(outB + t, rV * accB);
    }
}

// ------------------------------------------------------------------------------------------------------
// Two targets per thread (one warp per 64-target group): every LDS.128 of a source quad serves two targets.
// The single-region kernels (Laplace only: 6.5 packed instructions per pair) sit on the shared-memory data pipe
// with one target per thread (l1tex__data_pipe_lsu_wavefronts 75-82 % of peak, profiles/r3a); the fused twin
// kernel does not (54 %) and keeps one target per thread.
template <bool YA, bool TWIN, bool YB, bool GUARD>
__device__ __forceinline__ void p2p_quad_tile2(const float4 *__restrict__ sp, const float4 *__restrict__ sc, int nq, f2_t X0,
                                               f2_t Y0, f2_t Z0, f2_t X1, f2_t Y1, f2_t Z1, const P2PQuadConst &kc,
                                               f2_t (&a)[4], f2_t (&b)[4])
{
#ifndef P2PQ2_UNROLL
#define P2PQ2_UNROLL 1
#endif
    constexpr int UNR2 = P2PQ2_UNROLL;
#pragma unroll UNR2
    for (int q = 0; q < nq; q++) {
        const float4 px = sp[3 * q], py = sp[3 * q + 1], pz = sp[3 * q + 2];
        const float4 mV = sc[4 * q], mKx = sc[4 * q + 1], mKy = sc[4 * q + 2], mKz = sc[4 * q + 3];
        const f2_t pxl = f2_pack(px.x, px.y), pyl = f2_pack(py.x, py.y), pzl = f2_pack(pz.x, pz.y), mVl = f2_pack(mV.x, mV.y),
                   kxl = f2_pack(mKx.x, mKx.y), kyl = f2_pack(mKy.x, mKy.y), kzl = f2_pack(mKz.x, mKz.y);
        const f2_t pxh = f2_pack(px.z, px.w), pyh = f2_pack(py.z, py.w), pzh = f2_pack(pz.z, pz.w), mVh = f2_pack(mV.z, mV.w),
                   kxh = f2_pack(mKx.z, mKx.w), kyh = f2_pack(mKy.z, mKy.w), kzh = f2_pack(mKz.z, mKz.w);
        p2p_pair2<YA, TWIN, YB, GUARD>(X0, Y0, Z0, pxl, pyl, pzl, mVl, kxl, kyl, kzl, kc, a[0], b[0]);
        p2p_pair2<YA, TWIN, YB, GUARD>(X1, Y1, Z1, pxl, pyl, pzl, mVl, kxl, kyl, kzl, kc, a[1], b[1]);
        p2p_pair2<YA, TWIN, YB, GUARD>(X0, Y0, Z0, pxh, pyh, pzh, mVh, kxh, kyh, kzh, kc, a[2], b[2]);
        p2p_pair2<YA, TWIN, YB, GUARD>(X1, Y1, Z1, pxh, pyh, pzh, mVh, kxh, kyh, kzh, kc, a[3], b[3]);
    }
}

#define P2PQ2_THREADS (PYGBE_TG / 2)
template <bool YA, bool TWIN, bool YB>
__global__ void __launch_bounds__(P2PQ2_THREADS)
k_p2p_quad2(const int *__restrict__ skip, const int4 *__restrict__ items, const int4 *__restrict__ tiles,
            const int2 *__restrict__ segs, int np, const double4 *__restrict__ tpos, const double4 *__restrict__ cgeo,
            const float4 *__restrict__ posq, const float4 *__restrict__ chgq, double kappaA, double kappaB, double rV,
            double *__restrict__ outA, double *__restrict__ outB)
{
    __shared__ __align__(16) float4 s_pos[2][3 * P2P_QTILE];
    __shared__ __align__(16) float4 s_chg[2][4 * P2P_QTILE];
    __shared__ __align__(16) double4 s_an[2];
    if (skip && *skip) return;
    const int4 it = items[blockIdx.x];
    const int lane = threadIdx.x;
    const int t0 = it.x * PYGBE_TG + lane, t1 = t0 + P2PQ2_THREADS;
    const bool ok0 = t0 < np, ok1 = t1 < np;
    const double4 XA = ok0 ? tpos[t0] : make_double4(0, 0, 0, 0), XB = ok1 ? tpos[t1] : make_double4(0, 0, 0, 0);
    P2PQuadConst kc;
    {
        const float a = -(float)Real<float>::kscale(kappaA), b = -(float)Real<float>::kscale(kappaB);
        const float s = -(float)(1.0 / rV), c = -(float)(kappaB / rV), ka = (float)kappaA;      // negated: see p2p_pair2
        kc.nksA = f2_pack(a, a); kc.nksB = f2_pack(b, b); kc.kA = f2_pack(ka, ka); kc.sB = f2_pack(s, s); kc.cB = f2_pack(c, c);
        kc.tiny = f2_pack(1e-30f, 1e-30f);
    }
    double accA0 = 0.0, accB0 = 0.0, accA1 = 0.0, accB1 = 0.0;
    auto stage = [&](int buf, const int4 &tl) {                      // segments = (first point, points), multiples of 4
        int qoff = 0;                                                // quads staged so far
        for (int s0 = tl.x; s0 < tl.y; s0 += 32) {
            const int ns = min(32, tl.y - s0);
            const int2 mine = lane < ns ? segs[s0 + lane] : make_int2(0, 0);
            for (int s = 0; s < ns; s++) {
                const int q0 = __shfl_sync(0xffffffffu, mine.x, s) >> 2, nq = __shfl_sync(0xffffffffu, mine.y, s) >> 2;
                for (int i = lane; i < 7 * nq; i += P2PQ2_THREADS) {
                    if (i < 3 * nq) cp_async16(&s_pos[buf][3 * qoff + i], posq + 3 * (long)q0 + i);
                    else cp_async16(&s_chg[buf][4 * qoff + i - 3 * nq], chgq + 4 * (long)q0 + i - 3 * nq);
                }
                qoff += nq;
            }
        }
        if (lane < 2) cp_async16((char *)&s_an[buf] + 16 * lane, (const char *)(cgeo + tl.z) + 16 * lane);
        cp_async_commit();
    };
    int4 cur = tiles[it.y];
    int4 nxt = it.y + 1 < it.z ? tiles[it.y + 1] : cur;
    stage(0, cur);
    int buf = 0;
    for (int k = it.y; k < it.z; k++, buf ^= 1) {
        const bool more = k + 1 < it.z;
        if (more) { stage(buf ^ 1, nxt); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        const int nq = cur.w >> 3;
        const bool self = (cur.w & 1) != 0;
        cur = nxt;
        if (k + 2 < it.z) nxt = tiles[k + 2];
        __syncwarp();                                                // one warp: every lane's copies have landed
        const double4 an = s_an[buf];
        const float x0 = (float)(XA.x - an.x), y0 = (float)(XA.y - an.y), z0 = (float)(XA.z - an.z);
        const float x1 = (float)(XB.x - an.x), y1 = (float)(XB.y - an.y), z1 = (float)(XB.z - an.z);
        const float4 *sp = s_pos[buf], *sc = s_chg[buf];
        f2_t a[4] = {0, 0, 0, 0}, b[4] = {0, 0, 0, 0};
        if (self) p2p_quad_tile2<YA, TWIN, YB, true>(sp, sc, nq, f2_pack(x0, x0), f2_pack(y0, y0), f2_pack(z0, z0), f2_pack(x1, x1),
                                                      f2_pack(y1, y1), f2_pack(z1, z1), kc, a, b);
        else p2p_quad_tile2<YA, TWIN, YB, false>(sp, sc, nq, f2_pack(x0, x0), f2_pack(y0, y0), f2_pack(z0, z0), f2_pack(x1, x1),
                                                  f2_pack(y1, y1), f2_pack(z1, z1), kc, a, b);
        float lo, hi;
        f2_unpack(f2_add(a[0], a[2]), lo, hi); accA0 += (double)(lo + hi);
        f2_unpack(f2_add(a[1], a[3]), lo, hi); accA1 += (double)(lo + hi);
        if constexpr (TWIN) {
            f2_unpack(f2_add(b[0], b[2]), lo, hi); accB0 += (double)(lo + hi);
            f2_unpack(f2_add(b[1], b[3]), lo, hi); accB1 += (double)(lo + hi);
        }
        __syncwarp();                                                // buf is refilled two iterations from now
    }
    if (ok0) { atomicAdd(outA + t0, accA0); if constexpr (TWIN) atomicAdd(outB + t0, rV * accB0); }
    if (ok1) { atomicAdd(outA + t1, accA1); if constexpr (TWIN) atomicAdd(outB + t1, rV * accB1); }
}

// quad layout of the fp32 source coordinates (create time): see k_make_sposf for the rounding
__global__ void k_make_sposq(int np, int K, const int *__restrict__ panel_anchor, const double4 *__restrict__ cgeo,
                             const double4 *__restrict__ spos, float *__restrict__ posq)
{
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;      // Gauss point
    if (i >= (long)np * K) return;
    const double4 an = cgeo[panel_anchor[i / K]];
    const double4 s = spos[i];
    const long q = i >> 2;
    const int l = (int)(i & 3);
    posq[12 * q + l] = (float)(s.x - an.x); posq[12 * q + 4 + l] = (float)(s.y - an.y); posq[12 * q + 8 + l] = (float)(s.z - an.z);
}
