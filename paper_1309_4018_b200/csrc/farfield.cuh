// farfield.cuh -- P2M (a3) and the upward pass M2M (a4) of the Cartesian Taylor treecode, eq. (13)-(14),
// PAPER.md:144-153, :161.  (M2P lives in m2p.cuh, compiled once per order.)
//
// Two multipole sets per cell (reading A12), from the point charges mV_g (single layer) and the vectors
// mK_g (double layer, normal folded in), d = y_g - y_c:
//     MV^k = sum_g mV_g d^k                       ("m_c^k" of eq. 14)
//     MK^k = sum_g sum_i mK_g,i k_i d^(k - e_i)   (n . grad_y applied to the monomial)
// so that  sum_g [ mV_g G - mK_g . grad_y G ](x) ~ sum_|k|<=P a^k(x, y_c) (MV^k - MK^k).  Keeping the two
// sets apart lets the two regions on either side of the same surfaces ("twin" regions, e.g. eq. 10's
// Laplace and Yukawa rows) share one P2M and one upward pass: their moments are c_a MV + c_b MK with
// different constants.  Layout: mom[cell][set][Nc], fp64.
#pragma once
#include "common.cuh"
#include "tables.cuh"

// ------------------------------------------------------------------------------------------------ P2M
// One CTA per leaf; thread k owns coefficient k of both sets; the leaf's points go through shared memory
// as tables of powers d^0..d^P per axis (HBM traffic: each point read once, 64 B).
#define P2M_THREADS 128
#define P2M_TILE 64
#define P2M_SLOTS ((PYGBE_NCMAX + P2M_THREADS - 1) / P2M_THREADS)
__global__ void __launch_bounds__(P2M_THREADS)
k_p2m(const int *__restrict__ skip, int P, int Nc, int K, const IndexTables *__restrict__ tab,
      const int *__restrict__ leaf_cell, const double4 *__restrict__ cgeo, const int2 *__restrict__ crange,
      const double4 *__restrict__ spos, const double4 *__restrict__ schg, double *__restrict__ mom)
{
    __shared__ double s_pw[P2M_TILE][3][PYGBE_PMAX + 1];
    __shared__ double4 s_chg[P2M_TILE];
    if (skip && *skip) return;
    const int cell = leaf_cell[blockIdx.x];
    const double4 cg = cgeo[cell];
    const int2 rg = crange[cell];
    const long p0 = (long)rg.x * K, p1 = (long)rg.y * K;
    double accV[P2M_SLOTS], accK[P2M_SLOTS];
    int kk[P2M_SLOTS][3];
#pragma unroll
    for (int s = 0; s < P2M_SLOTS; s++) {
        accV[s] = accK[s] = 0.0;
        int k = threadIdx.x + s * P2M_THREADS;
        if (k < Nc) { kk[s][0] = tab->kxyz[k][0]; kk[s][1] = tab->kxyz[k][1]; kk[s][2] = tab->kxyz[k][2]; }
        else { kk[s][0] = kk[s][1] = kk[s][2] = 0; }
    }
    for (long base = p0; base < p1; base += P2M_TILE) {
        int n = (int)min((long)P2M_TILE, p1 - base);
        __syncthreads();
        for (int i = threadIdx.x; i < n * 3; i += P2M_THREADS) {
            int pt = i / 3, a = i - 3 * pt;
            double4 s = spos[base + pt];
            double d = (a == 0 ? s.x - cg.x : (a == 1 ? s.y - cg.y : s.z - cg.z));
            double pw = 1.0;
            for (int e = 0; e <= P; e++) { s_pw[pt][a][e] = pw; pw *= d; }
        }
        for (int i = threadIdx.x; i < n; i += P2M_THREADS) s_chg[i] = schg[base + i];
        __syncthreads();
#pragma unroll
        for (int s = 0; s < P2M_SLOTS; s++) {
            int k = threadIdx.x + s * P2M_THREADS;
            if (k >= Nc) break;
            const int kx = kk[s][0], ky = kk[s][1], kz = kk[s][2];
            double aV = 0.0, aK = 0.0;
            for (int pt = 0; pt < n; pt++) {
                double X = s_pw[pt][0][kx], Y = s_pw[pt][1][ky], Z = s_pw[pt][2][kz];
                double4 c = s_chg[pt];
                aV += c.x * X * Y * Z;
                double t = 0.0;
                if (kx) t += c.y * kx * s_pw[pt][0][kx - 1] * Y * Z;
                if (ky) t += c.z * ky * X * s_pw[pt][1][ky - 1] * Z;
                if (kz) t += c.w * kz * X * Y * s_pw[pt][2][kz - 1];
                aK += t;
            }
            accV[s] += aV; accK[s] += aK;
        }
    }
#pragma unroll
    for (int s = 0; s < P2M_SLOTS; s++) {
        int k = threadIdx.x + s * P2M_THREADS;
        if (k < Nc) { mom[((long)cell * 2) * Nc + k] = accV[s]; mom[((long)cell * 2 + 1) * Nc + k] = accK[s]; }
    }
}

// ------------------------------------------------------------------------------------------------ M2M
// Parent moments from the children's ("shifted and added"), for both sets:
//   M_p^k = sum_children sum_{l <= k} C(k,l) s^(k-l) M_c^l,   s = y_child - y_parent.
// The shift factorises over the axes, so it is applied as three one-dimensional shifts (x, then y, then z)
// through two shared-memory buffers: O(Nc P) work per child instead of O(Nc P^3).  All children of a parent
// are shifted concurrently (work item = (child, coefficient)), then summed.  The index tables are staged
// in shared memory (the first version read them from constant memory with divergent indices and was
// latency-bound: 62 us per launch, profiles/r1a_first_path.md).  One CTA per listed parent cell; launched
// level by level from the deepest upward, and only for the cells whose multipoles are used: those in
// some M2P list and, to build those, all their descendants (build_lists.cuh).
// Dynamic shared memory: 2 buffers x 8 children x 2 Nc doubles.
#define M2M_THREADS 512
static inline size_t m2m_smem_bytes(int Nc) { return (size_t)2 * 8 * 2 * Nc * sizeof(double); }
__global__ void __launch_bounds__(M2M_THREADS)
k_m2m(const int *__restrict__ skip, int P, int Nc, const int *__restrict__ cells, const IndexTables *__restrict__ tab,
      const double4 *__restrict__ cgeo, const int2 *__restrict__ cchild, double *__restrict__ mom)
{
    extern __shared__ double s_dyn[];
    __shared__ double s_pw[8][3][PYGBE_PMAX + 1];
    __shared__ double s_binom[PYGBE_PMAX + 1][PYGBE_PMAX + 1];
    __shared__ short s_idx3[PYGBE_PMAX + 1][PYGBE_PMAX + 1][PYGBE_PMAX + 1];
    __shared__ __align__(16) unsigned char s_k[PYGBE_NCMAX][4];
    if (skip && *skip) return;
    const int cell = cells[blockIdx.x];
    const int2 ch = cchild[cell];
    const int n2 = 2 * Nc, nch = ch.y, nw = nch * n2;
    double *s_a = s_dyn, *s_b = s_dyn + 8 * n2;
    for (int i = threadIdx.x; i < (PYGBE_PMAX + 1) * (PYGBE_PMAX + 1); i += M2M_THREADS)
        (&s_binom[0][0])[i] = (&tab->binom[0][0])[i];
    for (int i = threadIdx.x; i < (PYGBE_PMAX + 1) * (PYGBE_PMAX + 1) * (PYGBE_PMAX + 1); i += M2M_THREADS)
        (&s_idx3[0][0][0])[i] = (&tab->idx3[0][0][0])[i];
    for (int i = threadIdx.x; i < Nc; i += M2M_THREADS)
        *(uchar4 *)s_k[i] = *(const uchar4 *)tab->kxyz[i];
    for (int w = threadIdx.x; w < nw; w += M2M_THREADS) s_a[w] = mom[(long)ch.x * n2 + w];   // children are contiguous
    if (threadIdx.x < nch * 3) {
        const int c = threadIdx.x / 3, a = threadIdx.x - 3 * c;
        const double4 g = cgeo[ch.x + c], pg = cgeo[cell];
        const double sft = a == 0 ? g.x - pg.x : (a == 1 ? g.y - pg.y : g.z - pg.z);
        double pw = 1.0;
        for (int e = 0; e <= P; e++) { s_pw[c][a][e] = pw; pw *= sft; }
    }
    __syncthreads();
    for (int w = threadIdx.x; w < nw; w += M2M_THREADS) {          // shift along x: s_a -> s_b
        const int c = w / n2, e = w - c * n2, so = c * n2 + (e < Nc ? 0 : Nc), k = e < Nc ? e : e - Nc;
        const int kx = s_k[k][0], ky = s_k[k][1], kz = s_k[k][2];
        double a = 0.0;
        for (int l = 0; l <= kx; l++) a += s_binom[kx][l] * s_pw[c][0][kx - l] * s_a[so + s_idx3[l][ky][kz]];
        s_b[w] = a;
    }
    __syncthreads();
    for (int w = threadIdx.x; w < nw; w += M2M_THREADS) {          // shift along y: s_b -> s_a
        const int c = w / n2, e = w - c * n2, so = c * n2 + (e < Nc ? 0 : Nc), k = e < Nc ? e : e - Nc;
        const int kx = s_k[k][0], ky = s_k[k][1], kz = s_k[k][2];
        double a = 0.0;
        for (int l = 0; l <= ky; l++) a += s_binom[ky][l] * s_pw[c][1][ky - l] * s_b[so + s_idx3[kx][l][kz]];
        s_a[w] = a;
    }
    __syncthreads();
    for (int w = threadIdx.x; w < nw; w += M2M_THREADS) {          // shift along z: s_a -> s_b
        const int c = w / n2, e = w - c * n2, so = c * n2 + (e < Nc ? 0 : Nc), k = e < Nc ? e : e - Nc;
        const int kx = s_k[k][0], ky = s_k[k][1], kz = s_k[k][2];
        double a = 0.0;
        for (int l = 0; l <= kz; l++) a += s_binom[kz][l] * s_pw[c][2][kz - l] * s_a[so + s_idx3[kx][ky][l]];
        s_b[w] = a;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < n2; e += M2M_THREADS) {          // sum over the children
        double a = 0.0;
        for (int c = 0; c < nch; c++) a += s_b[c * n2 + e];
        mom[(long)cell * n2 + e] = a;
    }
}
