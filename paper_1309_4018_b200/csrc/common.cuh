// common.cuh -- shared declarations of libpygbe (CUDA, sm_100a).  See include/pygbe.h for the ABI and
// DESIGN.md for the data layout.  Paper citations are PAPER.md:<line>.
#pragma once
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <cmath>
#include <vector>
#include <algorithm>
#include <chrono>
#include <utility>
#include <cstdlib>
#include "../../include/pygbe.h"

#define PYGBE_PMAX 12
#define PYGBE_NCMAX 455              // (P+1)(P+2)(P+3)/6 at P = 12
#ifndef PYGBE_TG
#define PYGBE_TG 64                  // targets per group = threads per CTA of the P2P / M2P kernels
#endif
#define PYGBE_MAXLEVEL 21            // 21 bits per dimension in the 63-bit Morton key

void pygbe_set_error(const char *fmt, ...);

#define CUDA_TRY(expr)                                                                                \
    do {                                                                                              \
        cudaError_t e_ = (expr);                                                                      \
        if (e_ != cudaSuccess) {                                                                      \
            pygbe_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e_));    \
            return PYGBE_ECUDA;                                                                       \
        }                                                                                             \
    } while (0)

#define TRY(expr)                                                                                     \
    do {                                                                                              \
        int rc_ = (expr);                                                                             \
        if (rc_ != PYGBE_OK) return rc_;                                                              \
    } while (0)

// Launch bookkeeping: every kernel launch of the library goes through LAUNCH so that
// pygbe_stats().kernel_launches is a count, not a guess.
#define LAUNCH(h, kernel, grid, block, smem, ...)                                                     \
    do {                                                                                              \
        kernel<<<(grid), (block), (smem), (h)->stream>>>(__VA_ARGS__);                                \
        (h)->launches++;                                                                              \
    } while (0)

static inline int nc_of(int P) { return (P + 1) * (P + 2) * (P + 3) / 6; }
static inline int cdiv(long a, long b) { return (int)((a + b - 1) / b); }

// Tuning knobs are environment variables only in builds with -DPYGBE_TUNING (experiments); the
// product build compiles the defaults in and reads no environment.
#ifdef PYGBE_TUNING
static inline const char *tune_env(const char *name) { return getenv(name); }
#else
static inline const char *tune_env(const char *) { return nullptr; }
#endif

// ---------------------------------------------------------------------------------------------------
// Device memory owned by a handle.  Two sources (include/pygbe.h "Memory"):
//   workspace  one block supplied by the caller (pygbe_options.workspace, e.g. a torch uint8 tensor), carved
//              up by a host-side first-fit allocator with coalescing free list (a few hundred blocks per
//              handle; every alloc / free is a host call, the device never sees the bookkeeping);
//   pool       no workspace given: blocks from a library-owned stream-ordered pool (cudaMallocFromPoolAsync),
//              never the device's default pool, released in pygbe_destroy.
// In both modes the same allocator runs on offsets, so high_water is the workspace size that the sequence of
// allocations made so far needs: pygbe_workspace_size is a dry run in pool mode that reads it.  Blocks are
// 256-byte aligned.  Freed blocks are reused at once: everything that touches them is ordered on the handle's
// stream (side streams join it through events before any free).
struct DeviceArena {
    struct Block { size_t off, size; void *ptr; };
    std::vector<Block> used;                    // live blocks
    std::vector<std::pair<size_t, size_t>> holes;   // free (offset, size) below top, sorted by offset
    size_t top = 0;                             // end of the highest live block
    size_t bytes = 0;                           // live bytes (rounded to the alignment)
    size_t high_water = 0;                      // max of top so far
    char *base = nullptr;                       // workspace mode: caller's block
    size_t capacity = 0;
    cudaMemPool_t pool = nullptr;               // pool mode
    cudaStream_t stream = nullptr;
    static size_t round_up(size_t n) { return (n + 255) & ~(size_t)255; }
    size_t place(size_t n)                      // first fit; returns the offset
    {
        for (size_t i = 0; i < holes.size(); i++)
            if (holes[i].second >= n) {
                const size_t off = holes[i].first;
                if (holes[i].second == n) holes.erase(holes.begin() + i);
                else { holes[i].first += n; holes[i].second -= n; }
                return off;
            }
        const size_t off = top;
        top += n;
        high_water = std::max(high_water, top);
        return off;
    }
    void unplace(size_t off, size_t n)
    {
        size_t i = 0;
        while (i < holes.size() && holes[i].first < off) i++;
        holes.insert(holes.begin() + i, std::make_pair(off, n));
        if (i + 1 < holes.size() && holes[i].first + holes[i].second == holes[i + 1].first) {
            holes[i].second += holes[i + 1].second; holes.erase(holes.begin() + i + 1);
        }
        if (i > 0 && holes[i - 1].first + holes[i - 1].second == holes[i].first) {
            holes[i - 1].second += holes[i].second; holes.erase(holes.begin() + i);
        }
        if (!holes.empty() && holes.back().first + holes.back().second == top) { top = holes.back().first; holes.pop_back(); }
    }
    bool dry = false;                           // size query: alloc_big only books the space
    // The large arrays that no sizing step reads (panel moments, multipoles, correction values, Krylov basis): in a
    // size query they are only booked, not allocated -- the dry run of the 1.08 M-panel complex then touches 1.5 GB
    // instead of 8 GB.  The pointer returned in that case is a placeholder that must not be dereferenced.
    template <class T> int alloc_big(T **p, size_t n)
    {
        if (!dry) return alloc(p, n);
        if (n == 0) n = 1;
        const size_t sz = round_up(n * sizeof(T));
        const size_t off = place(sz);
        void *q = (void *)(((uintptr_t)1 << 48) + off);
        used.push_back({off, sz, q});
        bytes += sz;
        *p = (T *)q;
        return PYGBE_OK;
    }
    static bool placeholder(const void *q) { return ((uintptr_t)q >> 48) == 1; }
    template <class T> int alloc(T **p, size_t n)
    {
        *p = nullptr;
        if (n == 0) n = 1;
        const size_t sz = round_up(n * sizeof(T));
        const size_t off = place(sz);
        void *q = nullptr;
        if (base) {
            if (off + sz > capacity) {
                unplace(off, sz);
                pygbe_set_error("workspace too small: %zu bytes given, at least %zu needed (pygbe_workspace_size)", capacity, off + sz);
                return PYGBE_ENOMEM;
            }
            q = base + off;
        } else {
            cudaError_t e = pool ? cudaMallocFromPoolAsync(&q, sz, pool, stream) : cudaMallocAsync(&q, sz, stream);
            if (e != cudaSuccess) {
                unplace(off, sz);
                pygbe_set_error("device allocation of %zu bytes failed: %s", sz, cudaGetErrorString(e));
                return PYGBE_ENOMEM;
            }
        }
        used.push_back({off, sz, q});
        bytes += sz;
        *p = (T *)q;
        return PYGBE_OK;
    }
    void release_one(void *q)
    {
        if (!q) return;
        for (size_t i = 0; i < used.size(); i++)
            if (used[i].ptr == q) {
                if (!base && !placeholder(q)) cudaFreeAsync(q, stream);
                bytes -= used[i].size;
                unplace(used[i].off, used[i].size);
                used.erase(used.begin() + i);
                return;
            }
    }
    void release()
    {
        if (!base) for (const Block &b : used) if (!placeholder(b.ptr)) cudaFreeAsync(b.ptr, stream);
        used.clear(); holes.clear();
        top = 0; bytes = 0;
    }
};

// ---------------------------------------------------------------------------------------------------
// One region Omega of the multi-surface problem: its boundary panels are both the
// sources (K Gauss points each) and the targets (centroids) of one N-body sum with the region's kernel.
struct Region {
    int id = 0;
    int twin_of = -1;               // >= 0: shares tree, order, lists and moments with that region
    int twin = -1;                  // >= 0: the region that shares this one's structures
    double twin_rV = 0;             // twin charges: mV_B = twin_rV * mV_A, mK_B = -mK_A
    int *perm = nullptr;            // sorted position -> position in the unsorted boundary list
    int *panel_anchor = nullptr;    // anchor cell of each panel (mixed precision)
    double eps = 1, kappa = 0;
    bool yukawa = false;
    int np = 0, npts = 0;           // boundary panels, Gauss points (np * K)
    // per panel, Morton-sorted order -------------------------------------------------------------
    int *gid = nullptr;             // global panel id
    int *phi_idx = nullptr, *dphi_idx = nullptr, *row_idx = nullptr;   // positions in x / y
    double *cV = nullptr, *cK = nullptr;   // sigma_S c_S and sigma_S of the panel's surface
    double4 *tpos = nullptr;        // collocation point (x,y,z, L = sqrt(2A))
    double4 *pnrm = nullptr;        // unit normal (x,y,z) and area
    // per Gauss point (K consecutive per panel) ------------------------------------------------------
    double4 *spos = nullptr;        // (x, y, z, w_g A_j / 4pi)
    double4 *schg = nullptr;        // per matvec: (mV, mKx, mKy, mKz)
    float4 *sposf = nullptr;        // mixed precision: position relative to the anchor cell centre, weight
    bool quad = false;              // sposf / schgf hold quads of four points, structure-of-arrays (packed P2P, p2p.cuh)
    float4 *schgf = nullptr;
    double *pphi = nullptr, *pdphi = nullptr;   // per matvec: gathered densities
    double2 *pq = nullptr;          // per matvec: (cV dphi, cK phi) per panel, the weights of the panel moments (P2M)
    double *out = nullptr;          // per matvec: sum_S sigma_S [c_S V dphi - K phi] at each target
    double *corr = nullptr;         // per matvec: the singular / near-singular correction of that sum (k_near)
    // octree ----------------------------------------------------------------------------------------
    unsigned long long *keys = nullptr;
    int ncells = 0, nleaves = 0, depth = 0;
    double4 *cgeo = nullptr;        // cell centre (x,y,z) and edge length r_b
    int2 *crange = nullptr;         // panel range [lo, hi)
    int2 *cchild = nullptr;         // (first child, number of children)
    int *cparent = nullptr;
    unsigned long long *ckey = nullptr;
    std::vector<int> level_begin;   // host: cells of level l are [level_begin[l], level_begin[l+1])
    int *leaf_cell = nullptr;       // leaves in Morton order
    // cells whose multipoles are needed: those in some M2P list and all their descendants
    int *p2m_cells = nullptr; int n_p2m = 0;        // needed leaves (P2M)
    int4 *p2m_rec = nullptr;                        // per needed leaf: (cell, first panel, end panel, 0)
    int4 *m2m_rec = nullptr; int n_m2m = 0;         // needed internal cells, deepest level first: (cell, first child, n children, internal-child mask)
    double *pmom = nullptr;                         // [np][2][Nc] geometry-only panel moments about the panel's leaf centre (P2M), fp64
    float *pmomf = nullptr;                         // the same in fp32 (mixed precision; pmom is then not allocated)
    int *up_sync = nullptr;                         // [4] ticket and exit counters of the upward pass, number of passes so far
    int *cready = nullptr;                          // [ncells] matvec number at which the cell's multipoles were built
    double Lmax = 0;                // max panel length sqrt(2A) on this region's boundary
    double root_c[3] = {0, 0, 0}, root_edge = 1;
    // target groups and interaction lists -----------------------------------------------------------
    int ng = 0;
    double4 *ggeo = nullptr;        // group centre and radius
    int *m2p_off = nullptr, *m2p_cell = nullptr;
    int *p2p_off = nullptr;
    int4 *p2p_rng = nullptr;        // merged source panel ranges (lo, hi, anchor cell, -)
    int n_p2p_items = 0, n_m2p_items = 0;
    int4 *p2p_items = nullptr;      // (group, first tile, last tile + 1, source panels) over p2p_sub
    int4 *p2p_sub = nullptr;        // tiles: (first segment, last segment + 1, anchor cell, 2 * points + self flag)
    int2 *p2p_seg = nullptr;        // segments of the tiles: (first point, points), whole panels
    int4 *m2p_items = nullptr;      // (group, first list slot, last slot+1, unused)
    long p2p_pairs = 0, m2p_evals = 0;
    // multipoles ------------------------------------------------------------------------------------
    double *mom = nullptr;          // [ncells][2][Nc]: MV, MK (farfield.cuh), shared by twin regions
    const int *wt_off = nullptr; const short *wt_k = nullptr; const double *wt_c = nullptr;   // the W table of this region's kappa (handle-owned)
    bool lap = false;               // tree owner, kappa = 0, no twin: wc holds the Nc coefficients C'_f of k_m2p_lap instead
    long p2m_panels = 0, m2m_children = 0;   // panels streamed by one P2M launch, child cells read by one M2M launch
    void *wc = nullptr;             // tree owner: [ncells][m2p_stride(P, twin)] regrouped multipoles W_{m,e} of this region and,
                                    // interleaved, of its twin, in float or double (m2p.cuh; written by P2M / M2M)
    // singular / near-singular corrections (CSR over targets) ----------------------------------------
    int *corr_off = nullptr, *corr_col = nullptr;
    double2 *corr_val = nullptr;    // (sigma c (fine - coarse)_V, sigma (fine - coarse)_K)
    long corr_nnz = 0;
    // charges of this region -------------------------------------------------------------------------
    int nq = 0;
    double4 *qpos = nullptr;        // (x, y, z, q)
    int *qid = nullptr;             // caller's charge index
};

// A vector that a kernel reads or writes, resolved on the device so that one captured launch (CUDA graph) serves
// every caller buffer and every Krylov vector: base pointer taken from a device slot (or given directly), plus
// sel[0] * stride elements (the column of the Krylov basis the iteration is at).
struct VecRef {
    const double *const *slot;      // device slot holding the base pointer, or nullptr
    const double *ptr;              // base pointer when slot == nullptr
    const int *sel; long stride;    // optional column selector
    __device__ __forceinline__ const double *get() const
    {
        const double *b = slot ? *slot : ptr;
        return b + (sel ? (long)sel[0] * stride : 0L);
    }
};
static inline VecRef vec_direct(const double *p) { VecRef v; v.slot = nullptr; v.ptr = p; v.sel = nullptr; v.stride = 0; return v; }
static inline VecRef vec_slot(const double *const *s, const int *sel = nullptr, long stride = 0) { VecRef v; v.slot = s; v.ptr = nullptr; v.sel = sel; v.stride = stride; return v; }

// An instantiated CUDA graph of a fixed launch sequence, with what identifies the sequence (pointers, sizes, tol)
struct GraphSlot {
    cudaGraphExec_t exec = nullptr;
    long key[6] = {0, 0, 0, 0, 0, 0};
    long nlaunch = 0, nmatvec = 0;
    bool failed = false;            // capture or instantiation failed once: direct launches from then on
};

struct GmresWork {
    int m = 0;                      // restart length the buffers were sized for
    long n = 0;
    double *V = nullptr;            // [(m+1)][n]
    double *w = nullptr, *b = nullptr;
    double *H = nullptr;            // [(m+1)][m] column-major by column j: H[j*(m+1) + i]
    double *h1 = nullptr, *h2 = nullptr, *cs = nullptr, *sn = nullptr, *g = nullptr, *yk = nullptr;
    double *scal = nullptr;         // [0]=bnorm [1]=beta [2]=rel [3]=nrm2 scratch
    int *flags = nullptr;           // [0]=done [1]=k at convergence
};

struct pygbe_handle {
    int device = 0, n_sm = 148;
    cudaStream_t stream = nullptr;
    int K = 4, P = 6, Nc = 84, Kfine = 19, Nk = 5, ncrit = 0, precision = 0;
    double theta = 0.5, thres = 2.0;
    long npan = 0, nq = 0;
    int nsurf = 0, nreg = 0;
    std::vector<long> surf_first, surf_count;
    std::vector<int> rin, rout;
    std::vector<double> eps, kappa;
    DeviceArena mem;
    // global panel geometry (caller order)
    double *tri = nullptr;          // [npan][9]
    double4 *gcen = nullptr;        // centroid, L
    double4 *gnrm = nullptr;        // normal, area
    std::vector<Region> regions;
    GmresWork gm;
    double *phi_reac = nullptr;     // [nq]
    struct IndexTables *itab = nullptr;   // device copy of the multi-index tables
    int NW = 0;                           // W_{m,e} per moment set (m2p_nw(P)) and the table that forms them (tables.cuh)
    struct WDev { double kappa; int *off; short *k; double *c; };
    std::vector<WDev> wtabs;              // one reduced W table per distinct kappa among the regions (tables.cuh)
    int *lt_off = nullptr; short *lt_k = nullptr, *lt_deg = nullptr; double *lt_c = nullptr;   // Laplace form (build_lap_table), Nc entries
    cudaStream_t side = nullptr;    // far-field chain (P2M, M2M, M2P) runs here, concurrently with P2P
    cudaStream_t side2 = nullptr;   // near-field correction SpMV runs here
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_join2 = nullptr;
    // CUDA graphs: the kernel sequence of a matvec (7+ launches on three streams) and of a block of GMRES iterations is
    // captured once on capst and replayed with one cudaGraphLaunch on the caller's stream (which may be the legacy
    // default stream, where capture itself is not allowed)
    cudaStream_t capst = nullptr;
    bool use_graphs = true;
    const double **io = nullptr;    // device slots: [0], [1] x and y of pygbe_matvec; [2], [3] input base and output of the GMRES iteration
    const double *io_host[4] = {nullptr, nullptr, nullptr, nullptr};   // what the slots hold
    GraphSlot g_matvec, g_iter;
    long graph_launches = 0;
    char graph_note[160] = "";      // why a capture failed, if one did
    bool overlap = true;
    // The upward pass (P2M stream, M2M) is bandwidth- and latency-bound and runs beside the FMA-bound P2P; at full
    // width its CTAs (high priority, 350-512 threads, few of them busy) take the thread slots of every SM and the P2P
    // waits, so the two run one after the other.  Capped at 4 unsplit (P2M) / 1 (M2M) CTAs per SM they share the SMs:
    // 16.5 -> 15.3 ms per matvec on the 1.08 M-panel complex, 0.138 -> 0.132 ms on config 1 (every configuration
    // measured gains 4-10 %).
    bool narrow_upward = false;
    // optional block-diagonal right preconditioner of GMRES (pygbe_options.precond)
    int precond = 0;
    bool dry = false;               // size query (pygbe_workspace_size): allocate as create does, compute no values
    int group_mac = 0;              // pygbe_options.group_mac
    double *dq = nullptr;           // [nq] charges in the caller's order (energy)
    double4 *pinv = nullptr;        // per global panel: inverse of [[1/2, -V_in], [1/2, c V_out]] as (a, b, c, d)
    int2 *pidx = nullptr;           // per global panel: positions of (phi, dphi) = (row_in, row_out) in x / y
    double *zbuf = nullptr;         // [2 npan] scratch
    double *scratch = nullptr;      // small device scratch (16 doubles)
    double *xh = nullptr, *yh = nullptr;   // device staging for the *_host entry points
    int *pinned_flags = nullptr;    // host pinned, 4 ints
    double *pinned_scal = nullptr;  // host pinned, 8 doubles
    std::vector<double> qxyz, qq;   // host copies of the charges
    std::vector<int> qreg;
    long launches = 0, n_matvec = 0, kernels_per_matvec = 0;
    // optional per-stage CUDA-event timers (pygbe_profile / pygbe_stage_times)
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<int> ev_stage;          // stage started at event i (-1 = end marker)
    std::vector<int> ev_region;         // tree owner the launch after event i works on (-1: none)
    struct LaunchAcc { int stage, region; double ms; int launches; };
    std::vector<LaunchAcc> launch_acc;  // per (stage, region) accumulators of pygbe_launch_times
    size_t ev_used = 0;
    double stage_ms[PYGBE_N_STAGES] = {0};
    long stage_launches[PYGBE_N_STAGES] = {0};
    double create_ms = 0, last_solve_ms = 0;
    int last_iters = 0;
};
