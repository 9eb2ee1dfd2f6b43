// tree.cuh -- panel geometry (a1), Morton-sorted octree (a2), target groups and the warp-cooperative
// MAC traversal that emits the M2P / P2P interaction lists (a5).  PAPER.md:155-159, eq. (15).
#pragma once
#include "common.cuh"
#include "tables.cuh"
#include "blockops.cuh"

// ------------------------------------------------------------------------------------------ geometry
// flat triangles, collocation at the panel centre.  flags[0] is raised for a
// degenerate (zero-area or non-finite) triangle.
__global__ void k_panel_geometry(const double *__restrict__ tri, long npan, double4 *__restrict__ gcen,
                                 double4 *__restrict__ gnrm, int *flags)
{
    long j = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (j >= npan) return;
    const double *t = tri + 9 * j;
    double ux = t[3] - t[0], uy = t[4] - t[1], uz = t[5] - t[2];
    double vx = t[6] - t[0], vy = t[7] - t[1], vz = t[8] - t[2];
    double cx = uy * vz - uz * vy, cy = uz * vx - ux * vz, cz = ux * vy - uy * vx;
    double len = sqrt(cx * cx + cy * cy + cz * cz);
    if (!(len > 0.0) || !isfinite(len)) { atomicExch(flags, 1); len = 1.0; }
    double A = 0.5 * len;
    gcen[j] = make_double4((t[0] + t[3] + t[6]) / 3.0, (t[1] + t[4] + t[7]) / 3.0,
                           (t[2] + t[5] + t[8]) / 3.0, sqrt(2.0 * A));
    gnrm[j] = make_double4(cx / len, cy / len, cz / len, A);
}

// ------------------------------------------------------------------------------------------- Morton
__device__ __forceinline__ unsigned long long spread3(unsigned long long v)
{   // 21 bits -> every third bit
    v &= 0x1fffffULL;
    v = (v | v << 32) & 0x1f00000000ffffULL;
    v = (v | v << 16) & 0x1f0000ff0000ffULL;
    v = (v | v << 8) & 0x100f00f00f00f00fULL;
    v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
    v = (v | v << 2) & 0x1249249249249249ULL;
    return v;
}

// Key of a panel = Morton code of its centroid in the region's root cube (reading A11: the K Gauss
// points travel with their panel).  lo = corner of the root cube, scale = 2^21 / edge.
__global__ void k_region_keys(const double4 *__restrict__ gcen, const int *__restrict__ gid, int np,
                              double lox, double loy, double loz, double scale,
                              unsigned long long *__restrict__ keys, int *__restrict__ iota)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    double4 c = gcen[gid[p]];
    const double top = 2097151.0;
    unsigned long long qx = (unsigned long long)fmin(fmax((c.x - lox) * scale, 0.0), top);
    unsigned long long qy = (unsigned long long)fmin(fmax((c.y - loy) * scale, 0.0), top);
    unsigned long long qz = (unsigned long long)fmin(fmax((c.z - loz) * scale, 0.0), top);
    keys[p] = (spread3(qx) << 2) | (spread3(qy) << 1) | spread3(qz);
    iota[p] = p;
}

// Gather the region's per-panel data into Morton order and generate the Gauss points
// y_g = sum_v b_gv p_v with weight w_g A_j / (4 pi)  (the 1/(4 pi) of eq. (2), :55-58).
__global__ void k_region_gather(int np, int K, QuadTables q, const int *__restrict__ perm,
                                const int *__restrict__ gid_u, const int *__restrict__ phi_u,
                                const int *__restrict__ dphi_u, const int *__restrict__ row_u,
                                const double *__restrict__ cV_u, const double *__restrict__ cK_u,
                                const double *__restrict__ tri, const double4 *__restrict__ gcen,
                                const double4 *__restrict__ gnrm, int *__restrict__ gid,
                                int *__restrict__ phi_idx, int *__restrict__ dphi_idx,
                                int *__restrict__ row_idx, double *__restrict__ cV, double *__restrict__ cK,
                                double4 *__restrict__ tpos, double4 *__restrict__ pnrm,
                                double4 *__restrict__ spos)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    int u = perm[p];
    int j = gid_u[u];
    gid[p] = j; phi_idx[p] = phi_u[u]; dphi_idx[p] = dphi_u[u]; row_idx[p] = row_u[u];
    cV[p] = cV_u[u]; cK[p] = cK_u[u];
    tpos[p] = gcen[j];
    double4 nA = gnrm[j];
    pnrm[p] = nA;
    const double *t = tri + 9 * (long)j;
    const double inv4pi = 0.07957747154594767;
    for (int g = 0; g < K; g++) {
        double b0 = q.bK[g][0], b1 = q.bK[g][1], b2 = q.bK[g][2];
        double4 y = make_double4(b0 * t[0] + b1 * t[3] + b2 * t[6], b0 * t[1] + b1 * t[4] + b2 * t[7],
                                 b0 * t[2] + b1 * t[5] + b2 * t[8], q.wK[g] * nA.w * inv4pi);
        // a node at the centroid (K = 1, 4, 7) must coincide with the collocation point bit for bit, so
        // that the self pair has r = 0 exactly and is dropped by the P2P kernel (reading A5)
        if (b0 == b1 && b1 == b2) { double4 c = gcen[j]; y.x = c.x; y.y = c.y; y.z = c.z; }
        spos[(long)p * K + g] = y;
    }
}

// ------------------------------------------------------------------------------------------- octree
// Cells are key prefixes of the sorted panel keys.  One level is split per launch by ONE CTA so that the
// numbering of the cells is deterministic (an exclusive scan over the cells of the level hands out the
// child slots).  A cell is split when it holds more than ncrit panels ("less than NCRIT
// sources" per twig).
#define SPLIT_THREADS 1024
__global__ void __launch_bounds__(SPLIT_THREADS)
k_split_level(const unsigned long long *__restrict__ keys, int level, int lvl_begin, int lvl_end, int ncrit,
              int maxcells, double4 *cgeo, int2 *crange, int2 *cchild, int *cparent,
              unsigned long long *ckey, int *ncells_io)
{
    __shared__ int s_base;
    if (threadIdx.x == 0) s_base = *ncells_io;
    __syncthreads();
    const int shift = 3 * (PYGBE_MAXLEVEL - 1 - level);
    for (int c0 = lvl_begin; c0 < lvl_end; c0 += SPLIT_THREADS) {
        int c = c0 + threadIdx.x;
        int bounds[9];
        int nchild = 0;
        if (c < lvl_end) {
            int2 r = crange[c];
            if (r.y - r.x > ncrit && level < PYGBE_MAXLEVEL) {
                unsigned long long pre = ckey[c];
                bounds[0] = r.x; bounds[8] = r.y;
                for (int d = 1; d < 8; d++) {
                    unsigned long long want = ((pre << 3) | (unsigned long long)d) << shift;
                    int lo = r.x, hi = r.y;
                    while (lo < hi) {
                        int mid = (lo + hi) >> 1;
                        if (keys[mid] < want) lo = mid + 1; else hi = mid;
                    }
                    bounds[d] = lo;
                }
                for (int d = 0; d < 8; d++) nchild += (bounds[d + 1] > bounds[d]);
            }
        }
        int off, total;
        block_exclusive_sum<SPLIT_THREADS>(nchild, off, total);
        int base = s_base;
        __syncthreads();
        if (nchild > 0) {
            int first = base + off;
            if (first + nchild <= maxcells) {
                double4 g = cgeo[c];
                unsigned long long pre = ckey[c];
                double q = 0.25 * g.w;
                int k = 0;
                for (int d = 0; d < 8; d++) {
                    if (bounds[d + 1] <= bounds[d]) continue;
                    int cc = first + k++;
                    // key bit layout: x is the most significant bit of each digit
                    cgeo[cc] = make_double4(g.x + ((d & 4) ? q : -q), g.y + ((d & 2) ? q : -q),
                                            g.z + ((d & 1) ? q : -q), 0.5 * g.w);
                    crange[cc] = make_int2(bounds[d], bounds[d + 1]);
                    cchild[cc] = make_int2(-1, 0);
                    cparent[cc] = c;
                    ckey[cc] = (pre << 3) | (unsigned long long)d;
                }
            }
            cchild[c] = make_int2(first, nchild);
        }
        if (threadIdx.x == 0) s_base = base + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) *ncells_io = s_base;
}

// ------------------------------------------------------------------------------------ target groups
// A group = PYGBE_TG Morton-consecutive collocation points (reading A9: the MAC is tested for the
// whole group against its bounding sphere and bounding box, which is stricter than the per-target test
// of eq. 15).  ggeo[2g] = (centre, radius), ggeo[2g+1] = half extents of the box about the same centre.
__global__ void __launch_bounds__(PYGBE_TG)
k_group_geometry(const double4 *__restrict__ tpos, int np, double4 *__restrict__ ggeo)
{
    __shared__ double s_c[3];
    int g = blockIdx.x;
    int t = g * PYGBE_TG + threadIdx.x;
    bool ok = t < np;
    double4 x = ok ? tpos[t] : make_double4(0, 0, 0, 0);
    const double big = 1e300;
    double mn[3], mx[3];
    double v[3] = {x.x, x.y, x.z};
    for (int a = 0; a < 3; a++) {
        mn[a] = block_reduce<PYGBE_TG>(ok ? v[a] : big, OpMin());
        __syncthreads();
        mx[a] = block_reduce<PYGBE_TG>(ok ? v[a] : -big, OpMax());
        __syncthreads();
        if (threadIdx.x == 0) s_c[a] = 0.5 * (mn[a] + mx[a]);
    }
    __syncthreads();
    double dx = x.x - s_c[0], dy = x.y - s_c[1], dz = x.z - s_c[2];
    double r = ok ? sqrt(dx * dx + dy * dy + dz * dz) : 0.0;
    double rmax = block_reduce<PYGBE_TG>(r, OpMax());
    if (threadIdx.x == 0) {
        ggeo[2 * g] = make_double4(s_c[0], s_c[1], s_c[2], rmax);
        ggeo[2 * g + 1] = make_double4(0.5 * (mx[0] - mn[0]), 0.5 * (mx[1] - mn[1]), 0.5 * (mx[2] - mn[2]), 0.0);
    }
}

// longest panel L = sqrt(2A) of every cell (tpos.w), one warp per cell: the near-field guard of the traversal
__global__ void __launch_bounds__(128)
k_cell_lmax(int ncells, const int2 *__restrict__ crange, const double4 *__restrict__ tpos, double *__restrict__ clmax)
{
    const int c = (int)((blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (c >= ncells) return;
    const int2 r = crange[c];
    double m = 0.0;
    for (int p = r.x + lane; p < r.y; p += 32) m = fmax(m, tpos[p].w);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) clmax[c] = m;
}

// ---------------------------------------------------------------------------------------- traversal
// One warp per target group walks the tree from the root.  A cell is accepted for the
// Taylor expansion when the MAC of eq. (15) holds for every target of the group (reading A9):
//      theta * dist > r_b                             (reading A8: r_b = cell edge, y_c = cell centre)
// with dist = min |x - y_c| over the group.  A lower bound from the group's bounding sphere and box decides
// most cells; where it fails but the farthest possible target would pass, the minimum is taken over the
// group's own points (exact = 1; with the bound alone the direct lists were 27 % longer at config 1)
// and, so that the near-singular region is always inside the direct list ("in practice,
// the near-singular region is always contained in an area where the MAC criterion is not met"), when
// additionally every panel centroid of the cell is farther than thres * Lmax(cell) from every target, Lmax(cell)
// the longest panel of that cell (the longest panel of the whole region made the direct lists of the irregular
// molecular meshes 10 % longer):
//      dist - (sqrt(3)/2) r_b > thres * Lmax(cell).
// Accepted cells go to the M2P list; leaves that fail go to the P2P list (as cell ids); other cells
// are opened.  Pass 1 (fill == 0) counts, pass 2 writes.  The lane that owns child d of the popped
// cell tests it; ballots keep the output order deterministic (Morton order).
#define TRAV_WARPS 4
#define TRAV_STACK 256
__global__ void __launch_bounds__(TRAV_WARPS * 32)
k_traverse(int ng, const double4 *__restrict__ tpos, int np, int exact, const double4 *__restrict__ ggeo,
           const double4 *__restrict__ cgeo,
           const int2 *__restrict__ crange, const int2 *__restrict__ cchild, double theta,
           double thres, const double *__restrict__ clmax, int small_leaf, int fill, int *__restrict__ m2p_cnt, int *__restrict__ p2p_cnt,
           const int *__restrict__ m2p_off, const int *__restrict__ p2p_off, int *__restrict__ m2p_cell,
           int *__restrict__ p2p_leaf, int *overflow)
{
    __shared__ int s_stack[TRAV_WARPS][TRAV_STACK];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = blockIdx.x * TRAV_WARPS + warp;
    if (g >= ng) return;
    int *stack = s_stack[warp];
    const double4 G = ggeo[2 * g], H = ggeo[2 * g + 1];
    // the group's own targets, PYGBE_TG / 32 per lane (exact minimum distance of the undecided cells)
    double tx[PYGBE_TG / 32], ty[PYGBE_TG / 32], tz[PYGBE_TG / 32];
#pragma unroll
    for (int k = 0; k < PYGBE_TG / 32; k++) {
        const int t = g * PYGBE_TG + k * 32 + lane;
        const double4 x = tpos[min(t, np - 1)];                      // a ragged last group repeats its last target
        tx[k] = x.x; ty[k] = x.y; tz[k] = x.z;
    }
    int nm = 0, npp = 0, sp = 0;
    const int mbase = fill ? m2p_off[g] : 0, pbase = fill ? p2p_off[g] : 0;
    // the root is tested like a child of a virtual parent
    int first = 0, count = 1;
    while (true) {
        int c = (lane < count) ? first + lane : -1;
        bool acc = false, leaf = false, open = false, maybe = false;
        double dist = 0.0, rb = 0.0, near_dist = 0.0;
        if (c >= 0) {
            double4 cg = cgeo[c];
            double dx = G.x - cg.x, dy = G.y - cg.y, dz = G.z - cg.z;
            // lower bound of the distance from the cell centre to any target of the group: the better of
            // the bounding sphere and the bounding box
            double bx = fmax(fabs(dx) - H.x, 0.0), by = fmax(fabs(dy) - H.y, 0.0), bz = fmax(fabs(dz) - H.z, 0.0);
            const double dc = sqrt(dx * dx + dy * dy + dz * dz);
            dist = fmax(dc - G.w, sqrt(bx * bx + by * by + bz * bz));
            rb = cg.w;
            near_dist = thres * clmax[c];
            acc = (theta * dist > rb) && (dist - 0.8660254037844387 * rb > near_dist);
            // undecided: the bound fails, but the farthest any target can be (dc + radius) would pass
            const double far = dc + G.w;
            maybe = !acc && (theta * far > rb) && (far - 0.8660254037844387 * rb > near_dist);
        }
        if (exact) {
            // eq. (15) for every target of the group against the undecided cells: the minimum over the group's
            // own points instead of its bounding volume (accepts 5-10 % closer cells; still reading A9)
            unsigned mm = __ballot_sync(0xffffffffu, maybe);
            while (mm) {
                const int k = __ffs(mm) - 1;
                mm &= mm - 1;
                const double4 cg = cgeo[first + k];
                double d2 = 1e300;
#pragma unroll
                for (int j = 0; j < PYGBE_TG / 32; j++) {
                    const double ex = tx[j] - cg.x, ey = ty[j] - cg.y, ez = tz[j] - cg.z;
                    d2 = fmin(d2, ex * ex + ey * ey + ez * ez);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) d2 = fmin(d2, __shfl_xor_sync(0xffffffffu, d2, o));
                if (lane == k) {
                    dist = sqrt(d2);
                    acc = (theta * dist > rb) && (dist - 0.8660254037844387 * rb > near_dist);
                }
            }
        }
        if (c >= 0) {
            if (acc && cchild[c].y == 0) {
                // an accepted leaf with so few panels that summing its points directly (exact) costs fewer
                // instructions than one Taylor evaluation goes to the direct list instead
                int2 r = crange[c];
                if (r.y - r.x <= small_leaf) { acc = false; leaf = true; }
            } else if (!acc) {
                leaf = cchild[c].y == 0;
                open = !leaf;
            }
        }
        unsigned ma = __ballot_sync(0xffffffffu, acc);
        unsigned ml = __ballot_sync(0xffffffffu, leaf);
        unsigned mo = __ballot_sync(0xffffffffu, open);
        unsigned below = (1u << lane) - 1u;
        if (acc && fill) m2p_cell[mbase + nm + __popc(ma & below)] = c;
        if (leaf && fill) p2p_leaf[pbase + npp + __popc(ml & below)] = c;
        nm += __popc(ma);
        npp += __popc(ml);
        // push the cells to open in reverse so that they pop in Morton order
        int no = __popc(mo);
        if (open) {
            int slot = sp + (no - 1 - __popc(mo & below));
            if (slot < TRAV_STACK) stack[slot] = c; else atomicExch(overflow, 1);
        }
        sp = min(sp + no, TRAV_STACK);
        __syncwarp();
        if (sp == 0) break;
        int top = stack[sp - 1];
        sp--;
        int2 ch = cchild[top];
        first = ch.x; count = ch.y;
        __syncwarp();
    }
    if (lane == 0 && !fill) { m2p_cnt[g] = nm; p2p_cnt[g] = npp; }
}
