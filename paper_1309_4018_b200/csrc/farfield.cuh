// farfield.cuh -- P2M (a3), upward pass M2M (a4) and M2P (a6) of the Cartesian Taylor treecode,
// eq. (13)-(14).
//
// One combined multipole per cell serves both layers (reading A12): with point charges mV_g (single
// layer) and vectors mK_g (double layer, normal folded in)
//     M^k = sum_g [ mV_g d^k - sum_i mK_g,i k_i d^(k - e_i) ],   d = y_g - y_c,
// so that  sum_g [ mV_g G - mK_g . grad_y G ](x)  ~  sum_|k|<=P a^k(x, y_c) M^k  with the Taylor
// coefficients a^k = (1/k!) D_y^k G(x, y_c)  (eq. 14).
#pragma once
#include "common.cuh"
#include "tables.cuh"

// ------------------------------------------------------------------------------------------------ P2M
#define P2M_THREADS 128
#define P2M_TILE 64
__global__ void __launch_bounds__(P2M_THREADS)
k_p2m(const int *__restrict__ skip, int P, int Nc, int K, const int *__restrict__ leaf_cell, const double4 *__restrict__ cgeo,
      const int2 *__restrict__ crange, const double4 *__restrict__ spos, const double4 *__restrict__ schg,
      double *__restrict__ mom)
{
    __shared__ double s_pw[P2M_TILE][3][PYGBE_PMAX + 1];
    __shared__ double4 s_chg[P2M_TILE];
    if (skip && *skip) return;
    const int cell = leaf_cell[blockIdx.x];
    const double4 cg = cgeo[cell];
    const int2 rg = crange[cell];
    const long p0 = (long)rg.x * K, p1 = (long)rg.y * K;
    double acc[(PYGBE_NCMAX + P2M_THREADS - 1) / P2M_THREADS];
#pragma unroll
    for (int i = 0; i < (PYGBE_NCMAX + P2M_THREADS - 1) / P2M_THREADS; i++) acc[i] = 0.0;
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
        for (int s = 0; s < (PYGBE_NCMAX + P2M_THREADS - 1) / P2M_THREADS; s++) {
            int k = threadIdx.x + s * P2M_THREADS;
            if (k >= Nc) break;
            int kx = c_kxyz[k][0], ky = c_kxyz[k][1], kz = c_kxyz[k][2];
            double a = 0.0;
            for (int pt = 0; pt < n; pt++) {
                double X = s_pw[pt][0][kx], Y = s_pw[pt][1][ky], Z = s_pw[pt][2][kz];
                double4 c = s_chg[pt];
                double t = c.x * X * Y * Z;
                if (kx) t -= c.y * kx * s_pw[pt][0][kx - 1] * Y * Z;
                if (ky) t -= c.z * ky * X * s_pw[pt][1][ky - 1] * Z;
                if (kz) t -= c.w * kz * X * Y * s_pw[pt][2][kz - 1];
                a += t;
            }
            acc[s] += a;
        }
    }
#pragma unroll
    for (int s = 0; s < (PYGBE_NCMAX + P2M_THREADS - 1) / P2M_THREADS; s++) {
        int k = threadIdx.x + s * P2M_THREADS;
        if (k < Nc) mom[(long)cell * Nc + k] = acc[s];
    }
}

// ------------------------------------------------------------------------------------------------ M2M
// Parent moments from the children's ("shifted and added"):
//   M_p^k = sum_children sum_{l <= k} C(k,l) s^(k-l) M_c^l,   s = y_child - y_parent.
// One CTA per non-leaf cell of the level; launched level by level from the deepest upward.
#define M2M_THREADS 128
__global__ void __launch_bounds__(M2M_THREADS)
k_m2m(const int *__restrict__ skip, int P, int Nc, int cell_begin, int cell_end, const double4 *__restrict__ cgeo,
      const int2 *__restrict__ cchild, double *__restrict__ mom)
{
    __shared__ double s_M[PYGBE_NCMAX];
    __shared__ double s_pw[3][PYGBE_PMAX + 1];
    if (skip && *skip) return;
    const int cell = cell_begin + blockIdx.x;
    if (cell >= cell_end) return;
    const int2 ch = cchild[cell];
    if (ch.y == 0) return;                       // leaf: filled by P2M
    const double4 pg = cgeo[cell];
    double acc[(PYGBE_NCMAX + M2M_THREADS - 1) / M2M_THREADS];
#pragma unroll
    for (int i = 0; i < (PYGBE_NCMAX + M2M_THREADS - 1) / M2M_THREADS; i++) acc[i] = 0.0;
    for (int c = ch.x; c < ch.x + ch.y; c++) {
        __syncthreads();
        for (int i = threadIdx.x; i < Nc; i += M2M_THREADS) s_M[i] = mom[(long)c * Nc + i];
        if (threadIdx.x < 3) {
            double4 g = cgeo[c];
            double s = threadIdx.x == 0 ? g.x - pg.x : (threadIdx.x == 1 ? g.y - pg.y : g.z - pg.z);
            double pw = 1.0;
            for (int e = 0; e <= P; e++) { s_pw[threadIdx.x][e] = pw; pw *= s; }
        }
        __syncthreads();
#pragma unroll
        for (int s = 0; s < (PYGBE_NCMAX + M2M_THREADS - 1) / M2M_THREADS; s++) {
            int k = threadIdx.x + s * M2M_THREADS;
            if (k >= Nc) break;
            int kx = c_kxyz[k][0], ky = c_kxyz[k][1], kz = c_kxyz[k][2];
            double a = 0.0;
            for (int lx = 0; lx <= kx; lx++) {
                double fx = c_binom[kx][lx] * s_pw[0][kx - lx];
                for (int ly = 0; ly <= ky; ly++) {
                    double fy = fx * c_binom[ky][ly] * s_pw[1][ky - ly];
                    for (int lz = 0; lz <= kz; lz++)
                        a += fy * c_binom[kz][lz] * s_pw[2][kz - lz] * s_M[c_idx3[lx][ly][lz]];
                }
            }
            acc[s] += a;
        }
    }
#pragma unroll
    for (int s = 0; s < (PYGBE_NCMAX + M2M_THREADS - 1) / M2M_THREADS; s++) {
        int k = threadIdx.x + s * M2M_THREADS;
        if (k < Nc) mom[(long)cell * Nc + k] = acc[s];
    }
}

