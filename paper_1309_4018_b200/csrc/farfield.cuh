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

// Where a finished cell's multipoles go besides mom: the M2P does not read M^k but the regrouped coefficients
//     W_{m,e} = (-1)^|e| / e!  sum_{|j| = m - |e|} M^(e + 2j) / (2^|j| j!)            (m2p.cuh)
// of the combinations ca MV + cb MK that belong to the tree owner (A) and to its twin region (B, interleaved
// with A's when there is one), in the arithmetic type of the M2P, row stride padded to a multiple of 4.
// Written by the kernel that finishes the cell (P2M for leaves, M2M otherwise) from the sparse table
// (wt_off, wt_k, wt_c) built at create (tables.cuh): entry p of the stream is sum_i wt_c[i] M^(wt_k[i]).
// Laplace regions without a twin take the single polynomial of k_m2p_lap instead (m2p.cuh): same mechanism with
// the table of build_lap_table, each entry divided by the cell edge to the power wt_deg[p].
struct MomOut {
    void *wc;
    double caA, cbA, caB, cbB;
    int fp32, stride, twin, NW;
    const int *wt_off; const short *wt_k; const double *wt_c;      // table of the tree owner's kappa (tables.cuh)
    const int *wtB_off; const short *wtB_k; const double *wtB_c;   // table of the twin's kappa (the reduction depends on kappa)
    const short *wt_deg;            // Laplace form: degree of entry p; nullptr otherwise
    const double4 *cgeo;            // cell geometry (edge length in .w)
};
// mv, mk: the cell's two moment sets in shared memory; all nthreads threads of the CTA call this
__device__ __forceinline__ void wc_store(const MomOut &o, long cell, const double *mv, const double *mk, int tid, int nthreads)
{
    const double inv_edge = o.wt_deg ? 1.0 / o.cgeo[cell].w : 1.0;
    for (int p = tid; p < o.NW; p += nthreads) {
        double wv = 0.0, wk = 0.0;
        for (int i = o.wt_off[p]; i < o.wt_off[p + 1]; i++) {
            const int k = o.wt_k[i];
            const double c = o.wt_c[i];
            wv += c * mv[k]; wk += c * mk[k];
        }
        double a = o.caA * wv + o.cbA * wk, b = 0.0;
        if (o.twin) {
            double bv = 0.0, bk = 0.0;
            for (int i = o.wtB_off[p]; i < o.wtB_off[p + 1]; i++) {
                const int k = o.wtB_k[i];
                const double c = o.wtB_c[i];
                bv += c * mv[k]; bk += c * mk[k];
            }
            b = o.caB * bv + o.cbB * bk;
        }
        if (o.wt_deg) {                                            // C'_f = C_f / edge^|f|
            double s = 1.0;
            for (int d = o.wt_deg[p]; d > 0; d--) s *= inv_edge;
            a *= s; b *= s;
        }
        const long at = cell * o.stride + (o.twin ? 2 * p : p);
        if (o.fp32) { ((float *)o.wc)[at] = (float)a; if (o.twin) ((float *)o.wc)[at + 1] = (float)b; }
        else { ((double *)o.wc)[at] = a; if (o.twin) ((double *)o.wc)[at + 1] = b; }
    }
}

// ------------------------------------------------------------------------------------------------ P2M
// The densities are constant per panel, so a leaf's multipoles are linear in the panel values
// with geometry-only coefficients, computed once at create (k_panel_moments) about the centre of the panel's
// leaf, K-point rule:
//     GV_j^k = sum_g w_g d_g^k,     GK_j^k = sum_g w_g sum_i n_j,i k_i d_g^(k - e_i),     d_g = y_jg - y_c
//     MV^k(leaf) = sum_{j in leaf} (cV_j dphi_j) GV_j^k,      MK^k(leaf) = sum_{j in leaf} (cK_j phi_j) GK_j^k
// (cV, cK: the per-region constants folded into the densities; k_prep leaves the two products in pq).  Each matvec the P2M is
// then a streaming product: 2 Nc doubles read per panel, coalesced, two FMAs per 16 bytes -- HBM / L2 bound
// as SURVEY 8(d) puts it (27.5 MB at 20 480 panels and P = 6) instead of the ALU- and latency-bound
// monomial loop over the Gauss points of the first versions (29 us -> see profiles/r2a_regrouped_path.md).
// pmom[panel][set][Nc], panels in the region's Morton order; fp64, or fp32 in mixed precision (TM = float: the
// M2P reads fp32 coefficients anyway, the stream is half as long -- 1.4 instead of 2.85 GB for the 1.08 M panels of
// the Stern-layer region of config 4 at P = 8 -- and the sums over the panels of a leaf stay fp64).
#define PMOM_THREADS 128
template <typename TM>
__global__ void __launch_bounds__(PMOM_THREADS)
k_panel_moments(int P, int Nc, int K, const IndexTables *__restrict__ tab, const int *__restrict__ leaf_cell,
                const double4 *__restrict__ cgeo, const int2 *__restrict__ crange,
                const double4 *__restrict__ spos, const double4 *__restrict__ pnrm, TM *__restrict__ pmom)
{
    const int cell = leaf_cell[blockIdx.x];
    const double4 cg = cgeo[cell];
    const int2 rg = crange[cell];
    const long nitem = (long)(rg.y - rg.x) * Nc;
    for (long it = threadIdx.x; it < nitem; it += PMOM_THREADS) {
        const int j = rg.x + (int)(it / Nc), k = (int)(it % Nc);
        const int kx = tab->kxyz[k][0], ky = tab->kxyz[k][1], kz = tab->kxyz[k][2];
        const double4 n = pnrm[j];
        double gv = 0.0, gk = 0.0;
        for (int g = 0; g < K; g++) {
            const double4 s = spos[(long)j * K + g];
            const double dx = s.x - cg.x, dy = s.y - cg.y, dz = s.z - cg.z;
            // X1 = dx^(kx-1) (or 0), X = dx^kx, likewise for y and z
            double X1 = 0.0, X = 1.0, Y1 = 0.0, Y = 1.0, Z1 = 0.0, Z = 1.0;
            for (int e = 0; e < kx; e++) { X1 = X; X *= dx; }
            for (int e = 0; e < ky; e++) { Y1 = Y; Y *= dy; }
            for (int e = 0; e < kz; e++) { Z1 = Z; Z *= dz; }
            gv += s.w * X * Y * Z;
            gk += s.w * (n.x * kx * X1 * Y * Z + n.y * ky * X * Y1 * Z + n.z * kz * X * Y * Z1);
        }
        pmom[((long)j * 2) * Nc + k] = (TM)gv;
        pmom[((long)j * 2 + 1) * Nc + k] = (TM)gk;
    }
}

// CTAs take needed leaves grid-stride (4 CTAs per SM with nsplit = 1 in the narrowed pass, matvec.cuh; one CTA per leaf at
// full width); one work item (split s, coefficient k) per thread: split s takes every nsplit-th
// panel of the leaf; the partial sums meet in shared memory in a fixed order (deterministic).
#define P2M_MAXT 512
static inline int p2m_nsplit(int Nc) { return Nc >= 192 ? 1 : (Nc >= 96 ? 2 : (256 / Nc > 8 ? 8 : 256 / Nc)); }
static inline int p2m_threads(int Nc) { return (p2m_nsplit(Nc) * Nc + 31) / 32 * 32; }
template <typename TM>
__global__ void __launch_bounds__(P2M_MAXT)
k_p2m(const int *__restrict__ skip, int Nc, int nsplit, int n_leaves, const int4 *__restrict__ rec, const double2 *__restrict__ pq,
      const TM *__restrict__ pmom, double *__restrict__ mom, MomOut mo)
{
    __shared__ double s_part[2][P2M_MAXT];
    if (skip && *skip) return;
    const int t = threadIdx.x;
    const int sp = t / Nc, k = t - sp * Nc;
    const bool active = sp < nsplit;
    for (int leaf = blockIdx.x; leaf < n_leaves; leaf += gridDim.x) {
    const int4 rc = rec[leaf];                                     // (cell, first panel, end panel, -)
    const int cell = rc.x;
    double aV = 0.0, aK = 0.0;
    if (active) {
#pragma unroll 8
        for (int j = rc.y + sp; j < rc.z; j += nsplit) {
            const double2 q = pq[j];                               // (cV dphi, cK phi) of panel j, from k_prep
            aV += q.x * (double)pmom[((long)j * 2) * Nc + k];
            aK += q.y * (double)pmom[((long)j * 2 + 1) * Nc + k];
        }
        if (sp > 0) { s_part[0][t] = aV; s_part[1][t] = aK; }
    }
    __syncthreads();
    if (active && sp == 0) {
        for (int j = 1; j < nsplit; j++) { aV += s_part[0][t + j * Nc]; aK += s_part[1][t + j * Nc]; }
        mom[((long)cell * 2) * Nc + k] = aV;
        mom[((long)cell * 2 + 1) * Nc + k] = aK;
    }
    __syncthreads();
    if (active && sp == 0) { s_part[0][k] = aV; s_part[1][k] = aK; }
    __syncthreads();
    wc_store(mo, cell, s_part[0], s_part[1], t, blockDim.x);
    __syncthreads();                                               // s_part is rewritten by the next leaf
    }
}

// ------------------------------------------------------------------------------------------------ M2M
// Parent moments from the children's ("shifted and added"), for both sets:
//   M_p^k = sum_children sum_{l <= k} C(k,l) s^(k-l) M_c^l,   s = y_child - y_parent.
// The shift factorises over the axes: three one-dimensional passes (x, then y, then z).  In a pass the
// coefficients split into independent lines along the axis (all k with the other two indices (u, v) fixed,
// u + v <= P, length L = P - u - v + 1), and on a line the shift is the binomial transform
//   b_m <- sum_{l <= m} C(m,l) s^(m-l) b_l,
// computed in registers without binomials or powers by L - 1 sweeps  b_m += s b_(m-1), m = L-1 .. i  (i = 1 ..
// L-1).  One thread owns one line of one (child, set): it loads the line, sweeps, and stores it back in
// place; a __syncthreads separates the passes; then the children are summed.  (The first version looped
// over binomial terms through shared-memory tables per coefficient: ~1100 dependent instructions per warp
// and cell, 12 us per level.)
//
// The whole upward pass is ONE launch of persistent CTAs.  Cells are listed deepest level first -- only those
// whose multipoles are used: the ones in some M2P list and, to build those, all their descendants
// (build_lists.cuh) -- and handed out by an atomic ticket; a parent waits for the ready flag of each internal
// child.  A child's ticket is always smaller than its parent's, so the CTA holding it is already running: no
// deadlock whatever the residency.  Ready flags hold the number of the upward pass (sync[2], kept on the device; never reset); the last CTA to leave
// resets the ticket.  Children are read with ld.global.cg (written by other SMs during this launch).
// rec[i] = (cell, first child, number of children, bit c set if child c is internal).
// Dynamic shared memory: 8 children x 2 Nc doubles.
#define M2M_THREADS 512
#define M2M_SLOTS 3                      // 16 (P+1)(P+2)/2 lines <= 3 x 512 at P = 12
static inline size_t m2m_smem_bytes(int Nc) { return (size_t)8 * 2 * Nc * sizeof(double); }

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// one pass over the lines this thread owns; AXIS = 0, 1, 2
template <int PM, int AXIS>
__device__ __forceinline__ void m2m_pass(int P, int Nc, int nch, const int *line, double *s_m,
                                         const short (*s_idx3)[PYGBE_PMAX + 1][PYGBE_PMAX + 1], const double (*s_sh)[3])
{
#pragma unroll
    for (int sl = 0; sl < M2M_SLOTS; sl++) {
        const int q = line[sl];                                      // packed (child, set, u, v) or -1
        if (q < 0) continue;
        const int c = q >> 16, set = (q >> 8) & 1, u = (q >> 4) & 15, v = q & 15;
        if (c >= nch) continue;
        const int L = P - u - v + 1;
        double *m = s_m + (c * 2 + set) * Nc;
        const double s = s_sh[c][AXIS];
        double b[PM + 1];
        short id[PM + 1];
#pragma unroll
        for (int l = 0; l <= PM; l++) {
            id[l] = l < L ? (AXIS == 0 ? s_idx3[l][u][v] : (AXIS == 1 ? s_idx3[u][l][v] : s_idx3[u][v][l])) : (short)0;
            b[l] = l < L ? m[id[l]] : 0.0;
        }
#pragma unroll
        for (int i = 1; i <= PM; i++)
#pragma unroll
            for (int mm = PM; mm >= i; mm--) b[mm] = fma(s, b[mm - 1], b[mm]);
#pragma unroll
        for (int l = 1; l <= PM; l++)
            if (l < L) m[id[l]] = b[l];
    }
}

template <int PM>
__global__ void __launch_bounds__(M2M_THREADS)
k_m2m(const int *__restrict__ skip, int P, int Nc, int n_cells, const int4 *__restrict__ rec,
      const IndexTables *__restrict__ tab, const double4 *__restrict__ cgeo, double *mom, MomOut mo,
      int *sync, int *ready)
{
    extern __shared__ double s_m[];
    __shared__ short s_idx3[PYGBE_PMAX + 1][PYGBE_PMAX + 1][PYGBE_PMAX + 1];
    __shared__ double s_sh[8][3];
    __shared__ int s_ticket;
    if (skip && *skip) return;
    // ready flags hold the number of the upward pass that built the cell; sync[2] counts the passes and is advanced by
    // the last CTA to leave (after every CTA has read it), so that a captured launch needs no per-launch argument
    const int epoch = ld_acquire(sync + 2) + 1;
    const int n2 = 2 * Nc, nl = (P + 1) * (P + 2) / 2;
    for (int i = threadIdx.x; i < (PYGBE_PMAX + 1) * (PYGBE_PMAX + 1) * (PYGBE_PMAX + 1); i += M2M_THREADS)
        (&s_idx3[0][0][0])[i] = (&tab->idx3[0][0][0])[i];
    // the lines this thread owns: the same for every cell
    int line[M2M_SLOTS];
#pragma unroll
    for (int sl = 0; sl < M2M_SLOTS; sl++) {
        const int w = threadIdx.x + sl * M2M_THREADS;
        line[sl] = -1;
        if (w < 16 * nl) {
            const int cs = w / nl;
            int j = w - cs * nl, u = 0;
            while (j >= P - u + 1) { j -= P - u + 1; u++; }           // line j -> (u, v), u + v <= P
            line[sl] = ((cs >> 1) << 16) | ((cs & 1) << 8) | (u << 4) | j;
        }
    }
    for (;;) {
        __syncthreads();                                             // previous cell is done with shared memory
        if (threadIdx.x == 0) s_ticket = atomicAdd(&sync[0], 1);
        __syncthreads();
        if (s_ticket >= n_cells) break;
        const int4 rc = rec[s_ticket];
        const int cell = rc.x, ch0 = rc.y, nch = rc.z;
        if (threadIdx.x < nch && ((rc.w >> threadIdx.x) & 1))        // internal child: wait until it is built
            while (ld_acquire(ready + ch0 + threadIdx.x) != epoch) __nanosleep(32);
        if (threadIdx.x >= 32 && threadIdx.x < 32 + nch * 3) {
            const int c = (threadIdx.x - 32) / 3, a = (threadIdx.x - 32) - 3 * c;
            const double4 g = cgeo[ch0 + c], pg = cgeo[cell];
            s_sh[c][a] = a == 0 ? g.x - pg.x : (a == 1 ? g.y - pg.y : g.z - pg.z);
        }
        __syncthreads();
        for (int w = threadIdx.x; w < nch * n2; w += M2M_THREADS) s_m[w] = __ldcg(mom + (long)ch0 * n2 + w);   // children are contiguous
        __syncthreads();
        m2m_pass<PM, 0>(P, Nc, nch, line, s_m, s_idx3, s_sh);
        __syncthreads();
        m2m_pass<PM, 1>(P, Nc, nch, line, s_m, s_idx3, s_sh);
        __syncthreads();
        m2m_pass<PM, 2>(P, Nc, nch, line, s_m, s_idx3, s_sh);
        __syncthreads();
        for (int k = threadIdx.x; k < Nc; k += M2M_THREADS) {          // sum over the children
            double mv = 0.0, mk = 0.0;
            for (int c = 0; c < nch; c++) { mv += s_m[c * n2 + k]; mk += s_m[c * n2 + Nc + k]; }
            mom[(long)cell * n2 + k] = mv;
            mom[(long)cell * n2 + Nc + k] = mk;
            s_m[k] = mv; s_m[Nc + k] = mk;                           // only this thread read these two
        }
        __syncthreads();
        wc_store(mo, cell, s_m, s_m + Nc, threadIdx.x, M2M_THREADS);
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) st_release(ready + cell, epoch);
    }
    if (threadIdx.x == 0) {
        const int d = atomicAdd(&sync[1], 1);
        if (d == (int)gridDim.x - 1) { sync[2] = epoch; sync[1] = 0; __threadfence(); sync[0] = 0; }
    }
}

struct M2MLaunch {
    const int *skip; int P, Nc, n_cells, grid; const int4 *rec; const IndexTables *tab; const double4 *cgeo;
    double *mom; MomOut mo; int *sync, *ready; cudaStream_t stream;
};
template <int PM> static void m2m_go(const M2MLaunch &a)
{
    k_m2m<PM><<<a.grid, M2M_THREADS, m2m_smem_bytes(a.Nc), a.stream>>>(a.skip, a.P, a.Nc, a.n_cells, a.rec, a.tab, a.cgeo,
                                                                      a.mom, a.mo, a.sync, a.ready);
}
static void m2m_launch(const M2MLaunch &a)
{
    if (a.P <= 4) m2m_go<4>(a);
    else if (a.P <= 6) m2m_go<6>(a);
    else if (a.P <= 8) m2m_go<8>(a);
    else m2m_go<PYGBE_PMAX>(a);
}
static cudaError_t m2m_configure()
{
    cudaError_t e = cudaFuncSetAttribute(k_m2m<PYGBE_PMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)m2m_smem_bytes(PYGBE_NCMAX));
    return e;
}
