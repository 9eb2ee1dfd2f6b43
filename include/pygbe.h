/*
 * pygbe.h -- C ABI of libpygbe: the treecode-accelerated boundary-element matrix-vector product of the
 * linearised Poisson-Boltzmann equation (PyGBe, arXiv:1309.4018) and the ring around it (right-hand
 * side, restarted GMRES, reaction potential / solvation energy), hand-written CUDA for sm_100a.
 *
 * Citations are PAPER.md:<line> (+ section / equation).  "Reading Ax" refers to DESIGN.md.
 *
 * Conventions
 *   Units        Angstrom, elementary charges, energies in kJ/mol
 *                (C0 = qe^2 N_A 1e7 / eps0 = 17459.1429 kJ A /(mol e^2), reading A17).
 *   Surfaces     closed triangulated surfaces; triangles counter-clockwise seen from region_out, so the
 *                unit normal points region_in -> region_out (reading A3).  Every surface separates
 *                exactly two regions.  Disjoint closed components with identical (region_in,
 *                region_out) may be passed as one surface.
 *   Regions      region r has permittivity eps[r] and inverse Debye length kappa[r] (1/Angstrom);
 *                kappa[r] == 0 selects the Laplace kernel 1/(4 pi r), otherwise the Yukawa kernel
 *                exp(-kappa r)/(4 pi r) (eq. 2).
 *   Unknowns     surfaces in creation order; for surface s with N_s panels (caller's triangle order)
 *                x = [ phi_s (N_s) ; dphi/dn_s (N_s) ], the derivative taken on the region_in side
 *                along the normal (eq. 10 unknown [phi_1 ; dphi_1/dn]).
 *   Rows         y = [ equation of region_in(s) collocated on s (N_s) ; equation of region_out(s) (N_s) ].
 *                Row of region Omega collocated on panel i of surface T (eq. 9/10, PAPER.md:98-108;
 *                several surfaces: PAPER.md:121-133, reading A4):
 *                   1/2 phi_T,i - sum_{S in dOmega} sigma_S [ c_S (V_TS dphi_S)_i - (K_TS phi_S)_i ]
 *                sigma_S = +1, c_S = 1 when Omega = region_in(S); sigma_S = -1,
 *                c_S = eps[region_in(S)]/eps[region_out(S)] when Omega = region_out(S).
 *                Green's functions carry 1/(4 pi); the right-hand side is sum_k q_k G(x_i,r_k)/eps.
 *   Memory       pointers marked HOST are host memory, read during the call and never retained;
 *                pointers marked DEVICE are device memory on the handle's device, owned by the caller
 *                (e.g. torch tensors), fp64, pygbe_num_unknowns() long.  Internal device memory: if
 *                pygbe_options.workspace is given, EVERY device array of the handle (geometry, tree,
 *                lists, corrections, multipoles, GMRES basis, staging) is carved out of that block and
 *                the library allocates nothing else on the device; its size is queried first with
 *                pygbe_workspace_size, and a block that is too small gives PYGBE_ENOMEM.  The block stays
 *                owned by the caller and must outlive the handle.  Without a workspace the library takes
 *                its memory from a pool of its own (never the device's default pool) and returns it in
 *                pygbe_destroy.  pygbe_stats reports the bytes in use either way.
 *   Stream       all work of a handle is issued on the stream given in pygbe_options (a cudaStream_t,
 *                e.g. torch.cuda.current_stream().cuda_stream; NULL = legacy default stream).  Calls
 *                taking DEVICE pointers are asynchronous unless stated; one handle is not re-entrant.
 *   Errors       every call returns PYGBE_OK (0) or a negative code; nothing throws or aborts across
 *                the ABI; pygbe_last_error() gives a thread-local message.  A failed pygbe_create
 *                leaves *out = NULL.
 */
#ifndef PYGBE_H
#define PYGBE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PYGBE_OK        0
#define PYGBE_EINVAL   (-1)  /* null pointer, bad size, unsupported K / P, theta < 0, bad region ids,  */
                             /* open / inconsistently oriented mesh, zero-area triangle, region graph  */
                             /* (regions = nodes, surfaces = edges) not a tree                         */
#define PYGBE_ENOMEM   (-2)  /* device or host allocation failed, or the workspace is too small         */
#define PYGBE_ECUDA    (-3)  /* a CUDA call or kernel failed                                           */
#define PYGBE_ENOCONV  (-4)  /* GMRES reached max_iter; x and the residual are still returned          */

#define PYGBE_PRECISION_FP64  0  /* every kernel in fp64                                               */
#define PYGBE_PRECISION_MIXED 1  /* P2P / M2P arithmetic in fp32 (cell-local coordinates), fp64        */
                                 /* accumulation, fp64 near-field corrections, fp64 GMRES              */

typedef struct pygbe_handle pygbe_handle; /* opaque, owned by the library */

/* One closed surface ("flat triangular panels"). HOST pointers. */
typedef struct {
    const double  *vertices;   int64_t n_vertices;   /* [n_vertices][3], Angstrom                    */
    const int32_t *triangles;  int64_t n_triangles;  /* [n_triangles][3], 0-based vertex ids         */
    int32_t region_in, region_out;
} pygbe_surface;

/* Point charges (eq. 1). HOST pointers; region == NULL puts all charges in region 0. */
typedef struct {
    const double  *xyz;    /* [n][3] Angstrom */
    const double  *q;      /* [n] units of e  */
    const int32_t *region; /* [n] or NULL     */
    int64_t n;
} pygbe_charges;

/* Options; zero-initialise and set what you need (0 selects the default given in brackets). */
typedef struct {
    int32_t K_fine;     /* Gauss points in the near-singular region [19]  (Tables 4, 6)  */
    double  thres;      /* near-singular radius in units of L = sqrt(2 A_j) [2.0] (Table 6; A7);       */
                        /* negative disables the near-singular rule (self panels are still analytic)   */
    int32_t N_k;        /* Gauss-Legendre points per side of the semi-analytic self integral [5]       */
    int32_t ncrit;      /* max source panels per octree leaf (NCRIT of PAPER.md:155, in panels) [auto] */
    int32_t precision;  /* PYGBE_PRECISION_* [FP64]                                                    */
    int32_t device;     /* CUDA device ordinal [0]                                                     */
    void   *stream;     /* cudaStream_t [NULL]                                                         */
    int32_t check_mesh; /* 1: verify closedness / orientation on the host in create [0]                */
    int32_t precond;    /* GMRES right preconditioner: 0 none (the paper names none) [0];        */
                        /* 1 block-diagonal: per panel the 2x2 block [[1/2, -V_ii^in], [1/2, c V_ii^out]] of   */
                        /* its two rows and two unknowns (self integrals only).  Same stopping test, since a   */
                        /* right preconditioner leaves the residual b - A x unchanged                          */
    int32_t group_mac;  /* MAC of a target group (reading A9): 0 eq. (15) for every target of the group, decided  */
                        /* from the group's own points where its bounding volume cannot [0]; 1 bounding volume  */
                        /* only (stricter: longer direct lists, smaller error)                                  */
    void   *workspace;  /* DEVICE block that holds every internal array of the handle, or NULL [NULL]: see      */
                        /* "Memory" above; 256-byte aligned, owned by the caller, must outlive the handle        */
    size_t  workspace_bytes;   /* size of that block; at least what pygbe_workspace_size returned                */
    int32_t reserved[4];
} pygbe_options;

/* Counters and timings filled by pygbe_stats. */
typedef struct {
    int64_t n_panels, n_unknowns, n_regions, n_surfaces, n_charges;
    int64_t n_points;            /* Gauss points summed over regions (a point bounding 2 regions x2)   */
    int64_t n_cells, n_leaves, n_groups, tree_depth;
    int64_t p2p_pairs;           /* (target, Gauss point) pairs evaluated directly per matvec          */
    int64_t m2p_evals;           /* (target, accepted cell) Taylor evaluations per matvec              */
    int64_t direct_equiv;        /* sum_regions N_targets x N_points: interactions of the dense matvec */
    int64_t near_nnz;            /* entries of the singular / near-singular correction (a8)            */
    int64_t device_bytes;        /* internal device memory in use by the handle (workspace or pool)    */
    int64_t workspace_high_water;/* workspace bytes the allocations made so far needed at their peak   */
    int64_t n_matvec;            /* matvecs executed so far                                            */
    int64_t kernels_per_matvec;  /* kernel launches one pygbe_matvec issues                            */
    int64_t kernel_launches;     /* all kernel launches issued by this handle so far (inside graphs too) */
    int64_t graph_launches;      /* cudaGraphLaunch calls so far: a matvec is one graph, `poll` GMRES  */
                                 /* iterations are one graph; 0 if capture is unavailable              */
    double  create_ms, last_solve_ms;
    int32_t last_iters;
    int32_t P, K, precision;
    double  theta;
} pygbe_stats_t;

/*
 * Build everything that depends on geometry only ("compute the tree structure and
 * interaction list only once"): panel geometry and Gauss points (a1), Morton-sorted octree per region
 * (a2), traversal with the multipole-acceptance criterion theta > r_b / r_tb (eq. 15, PAPER.md:155-159;
 * reading A8: r_b = cell edge, r_tb = distance to the cell centre) into M2P / P2P lists (a5), and the
 * singular / near-singular corrections (a8).
 *   K      Gauss points per panel, one of 1, 3, 4, 7
 *   P      order of the Cartesian Taylor expansion, 1..12        (eq. 13-14)
 *   theta  MAC parameter, >= 0; theta == 0 never accepts a cell, i.e. direct O(N^2) summation
 * Synchronous.  All HOST inputs are copied.
 */
int pygbe_create(const pygbe_surface *surfaces, int32_t n_surfaces, const pygbe_charges *charges,
                 const double *eps, const double *kappa, int32_t n_regions,
                 int32_t K, int32_t P, double theta, const pygbe_options *opt, pygbe_handle **out);

void pygbe_destroy(pygbe_handle *h);

/* Size in bytes of the workspace that pygbe_create with the same arguments needs, including the buffers of
 * pygbe_solve for a restart length of gmres_restart (<= 0: 100), of the *_host entry points and of
 * pygbe_energy ("workspace supplied by the caller, size queried first").  The interaction lists depend on the
 * geometry, so this is a dry run of create's sizing (tree, traversal, list and correction patterns; no
 * values are computed) in memory of the library's own pool, released before returning.  opt->workspace is
 * ignored.  Synchronous; same argument checks and error codes as pygbe_create. */
int pygbe_workspace_size(const pygbe_surface *surfaces, int32_t n_surfaces, const pygbe_charges *charges,
                         const double *eps, const double *kappa, int32_t n_regions,
                         int32_t K, int32_t P, double theta, const pygbe_options *opt,
                         int32_t gmres_restart, size_t *bytes);

/* 2 * total number of panels; < 0 on a NULL handle. */
int64_t pygbe_num_unknowns(const pygbe_handle *h);

/* y = A x: one evaluation of the treecode: P2M (eq. 14), upward pass, M2P with the
 * Laplace / Yukawa recurrences, P2P, near-field corrections, block combination (eq. 10).
 * x_dev, y_dev: DEVICE, must not alias.  Asynchronous on the handle's stream. */
int pygbe_matvec(pygbe_handle *h, const double *x_dev, double *y_dev);

/* Same with HOST buffers: copies x to the device, runs the matvec, copies y back, synchronises. */
int pygbe_matvec_host(pygbe_handle *h, const double *x_host, double *y_host);

/* b = right-hand side, eq. (9)/(11) with the 1/(4 pi) of eq. (9) (reading A2).
 * b_dev: DEVICE.  Asynchronous. */
int pygbe_rhs(pygbe_handle *h, double *b_dev);

/* Restarted GMRES, x0 = 0, no preconditioner unless pygbe_options.precond, stop at
 * ||b - A x|| / ||b|| <= tol (reading A16).  The whole iteration runs on the device; the host only polls flags.
 * A cycle ends when the Arnoldi / Givens estimate of the residual reaches tol; convergence is DECLARED only when
 * the residual recomputed from b - A x with one more matvec is within tol, and that recomputed value is what
 * rel_resid returns.  If the two keep disagreeing (tol below what the operator's arithmetic attains: about 1e-6
 * relative for PYGBE_PRECISION_MIXED, 1e-12 for FP64 with the treecode's non-deterministic summation order) the
 * call returns PYGBE_ENOCONV.  A breakdown (zero pivot) leaves that direction out instead of dividing by zero.
 * x_dev: DEVICE, receives the solution.  iters (matvecs inside Arnoldi steps), rel_resid: HOST, may be NULL.
 * Synchronous.  Returns PYGBE_ENOCONV if max_iter iterations did not reach tol (x and rel_resid still returned).
 * In a caller-supplied workspace the GMRES buffers were sized for the gmres_restart given to
 * pygbe_workspace_size: a longer restart gives PYGBE_ENOMEM. */
int pygbe_solve(pygbe_handle *h, double tol, int32_t restart, int32_t max_iter, double *x_dev,
                int32_t *iters, double *rel_resid);

/* HOST-buffer convenience: solve and copy x back (x_host may be NULL), then evaluate the energies. */
int pygbe_solve_host(pygbe_handle *h, double tol, int32_t restart, int32_t max_iter, double *x_host,
                     int32_t *iters, double *rel_resid, double *E_solv_kJ_per_mol,
                     double *E_coul_kJ_per_mol);

/* Reaction potential at the charges (eq. 4) and dG_solv = 1/2 sum q_k phi_reac(r_k)
 * (eq. 6); Coulomb energy of the charges (eq. 8).
 * x_dev: DEVICE.  Outputs HOST, either may be NULL.  Synchronous. */
int pygbe_energy(pygbe_handle *h, const double *x_dev, double *E_solv_kJ_per_mol,
                 double *E_coul_kJ_per_mol);

/* phi_reac at every charge, in the caller's charge order (units e/Angstrom, i.e. before C0).
 * phi_dev: DEVICE [n_charges].  Asynchronous. */
int pygbe_reaction_potential(pygbe_handle *h, const double *x_dev, double *phi_dev);

int pygbe_stats(const pygbe_handle *h, pygbe_stats_t *out);

/* Per-stage CUDA-event timers of the matvec (SURVEY 5 "tracing / profiling").  pygbe_profile(h, 1) resets
 * and enables them, pygbe_profile(h, 0) disables; while enabled every matvec records one event per stage
 * start on the handle's stream (so a profiled matvec is a little slower: never quote its total time).
 * pygbe_stage_times synchronises and returns the accumulated milliseconds and kernel-launch counts per
 * stage since enabling: ms and launches are HOST arrays of PYGBE_N_STAGES entries (launches may be NULL). */
#define PYGBE_STAGE_PREP    0  /* density weighting (a9 input side)             */
#define PYGBE_STAGE_P2M     1  /* a3                                            */
#define PYGBE_STAGE_M2M     2  /* a4                                            */
#define PYGBE_STAGE_M2P     3  /* a6                                            */
#define PYGBE_STAGE_P2P     4  /* a7                                            */
#define PYGBE_STAGE_NEAR    5  /* a8 correction SpMV                            */
#define PYGBE_STAGE_COMBINE 6  /* a9 block combination                          */
#define PYGBE_N_STAGES      8
int pygbe_profile(pygbe_handle *h, int enable);
int pygbe_stage_times(pygbe_handle *h, double *ms, int64_t *launches);

/* The same timers per kernel launch of a matvec, i.e. per (stage, tree): accumulated milliseconds and number
 * of launches since pygbe_profile(h, 1), the work one launch does and the bytes it has to move at least
 * (inputs read once + outputs written once), from which bench.py forms the roofline numbers.
 * out: HOST array of max_out records; *n_out receives the number written.  Synchronises the stream. */
typedef struct {
    int32_t stage;       /* PYGBE_STAGE_*                                                                 */
    int32_t region;      /* region id of the tree owner the launch works on                               */
    int32_t twin_region; /* region fused into the same launch (twin regions), or -1                       */
    int32_t launches;    /* launches accumulated                                                          */
    double  ms;          /* accumulated milliseconds                                                      */
    int64_t units;       /* per launch: P2P (target, Gauss point) pairs; M2P (target, cell) evaluations   */
                         /* (a fused twin pair counts once here); P2M panels; M2M cells; else rows / points */
    int64_t bytes;       /* per launch: algorithmic bytes (HBM-bound stages; 0 where not meaningful)      */
    char    kernel[64];  /* kernel name                                                                   */
} pygbe_launch_info;
int pygbe_launch_times(pygbe_handle *h, pygbe_launch_info *out, int32_t max_out, int32_t *n_out);

/* Thread-local message of the last failing call ("" if none). */
const char *pygbe_last_error(void);

/* ALU roofline denominators measured on `device` with dependent-FMA / MUFU micro-kernels (synchronous,
 * ~100 ms): out5[0] = fp32 FMA TFLOP/s, out5[1] = fp64 FMA TFLOP/s, out5[2] = MUFU.RSQ Gop/s, out5[3] = TFLOP/s
 * of an fp32 FMUL + three-register FFMA mix over 24 live registers (the practical ceiling of the instruction mix of the
 * regrouped M2P / P2P; FMA = 2 flops, MUL = 1), out5[4] = TFLOP/s of the bare Horner stream of the Laplace-form M2P
 * (packed FFMA2 with a broadcast coefficient from shared memory, P = 8: the ceiling of k_m2p_lap's pattern).
 * out5: HOST, 5 doubles. */
int pygbe_alu_peaks(int32_t device, double *out5);

/* The north star's tensor-core question, measured (csrc/mma_probe.cuh; not on the product path): per (64-target
 * group, cell) the regrouped M2P is the product [64 x Nc] * [Nc x (P+1)] with a target-specific left operand.  On
 * synthetic far-field data (8192 groups x 32 cells, Yukawa, single moment set) it times and checks against fp64
 * direct sums four variants v = 0..3: the production CUDA-core kernel; only the write of the monomial tile to shared
 * memory that any tensor-core form needs first; tile + TF32 tensor-core contraction (mma.sync m16n8k8) + radial part
 * in one pass; the same with the 3 x TF32 split.  out12[3 v] = ms per launch, out12[3 v + 1] = rel-L2 error (NaN for
 * the tile-only variant), out12[3 v + 2] = (group, cell) pairs per launch.  P = 6 or 8.  out12: HOST.  Synchronous. */
int pygbe_mma_probe(int32_t device, int32_t P, double *out12);

/* ONE entry point that allocates nothing (csrc/noalloc.cu), for callers that cannot call cudaMalloc (CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the Coulomb energy of n point charges in one region of
 * permittivity eps (eq. 8),  E = 1/2 C0 sum_{k != l} q_k q_l / (4 pi eps r_kl)  in kJ/mol -- the term
 * pygbe_energy returns as E_coul, without a handle.  Its scratch (the charges packed as (x, y, z, q) records and the
 * accumulator) is a file-scope static __device__ array of PYGBE_NOALLOC_MAX_CHARGES records, 512.25 KB, which every GPU
 * that loads the library holds until the process exits.  The call issues three kernels on `stream` and calls no
 * cudaMalloc, cudaFree or allocating library routine; n > PYGBE_NOALLOC_MAX_CHARGES is rejected with PYGBE_EINVAL.
 * xyz_dev [n][3], q_dev [n]: DEVICE, read only;  E_dev [1]: DEVICE, written.  Asynchronous.  The array is shared by
 * every call and keeps the last call's contents (each call rewrites what it uses and clears the accumulator): calls
 * that overlap on the GPU -- two streams, two host threads -- race on it; serialise them.  pygbe_noalloc_setup takes
 * the array's device address (once per device; also done by the first call) so that later calls do no set-up work. */
#define PYGBE_NOALLOC_MAX_CHARGES 16384
int pygbe_noalloc_setup(int32_t device);
int pygbe_coulomb_energy_noalloc(int32_t device, void *stream, const double *xyz_dev, const double *q_dev, int64_t n,
                                 double eps, double *E_dev);

/* Host-only (no GPU needed): the sparse coefficient tables that the P2M / M2M epilogue applies to a cell's Cartesian
 * moments (canonical order: total order n, then kx descending, then ky descending) to form the M2P's input.
 *   which = 0  regrouped form on harmonically reduced moments for the kernel exp(-kappa r)/r: entry p of the
 *              stream -- ex, ey ascending, ez in {0, 1}, |e| <= P, then J = 0 .. (P - |e|)/2 -- is W_{m = |e| + J, e};
 *   which = 1  Laplace form: entry p -- fx, fy, fz descending, |f| <= P -- is C_f, the coefficient of (d / r^2)^f; deg[p] = |f|.
 * Entry p = sum_{i in [off[p], off[p+1])} c[i] * M^(k[i]).  With off == NULL only the sizes are returned.
 * off: HOST int32 [cap_entries + 1]; k: int16 [cap_nnz]; c: double [cap_nnz]; deg: int16 [cap_entries] or NULL. */
int pygbe_host_table(int32_t which, int32_t P, double kappa, int32_t cap_entries, int32_t cap_nnz, int32_t *n_entries,
                     int32_t *n_nnz, int32_t *off, int16_t *k, double *c, int16_t *deg);

/* Library / build identification, e.g. "pygbe-b200 0.3 sm_100a". */
const char *pygbe_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PYGBE_H */
