// gmres.cuh -- device-resident restarted GMRES (a11).  PAPER.md:169 "PyGBe uses a Krylov method ... one
// evaluation of the treecode per iteration"; tolerances Tables 1, 3 (:197-203, :223-227); reading A16.
// Arnoldi with classical Gram-Schmidt applied twice (CGS2: two batched dot passes instead of j
// sequential ones), Givens rotations and the convergence test run in kernels; every kernel returns
// immediately once flags[0] ("stop") is set, so the host can queue iterations ahead and only polls.
// flags: [0] stop -- the Arnoldi estimate |g_(j+1)| / |b| reached tol, or the recomputed residual did; [1] columns
// built in the current cycle; [2] iterations (matvecs inside Arnoldi steps) so far; [3] converged -- set only by
// k_gm_begin, i.e. only when the residual b - A x recomputed with a matvec is within tol (the estimate alone
// does not see the rounding of the operator: fp32 kernels, treecode, atomics).
#pragma once
#include "common.cuh"
#include "tables.cuh"
#include "nearfield.cuh"
#include "blockops.cuh"

#define GM_THREADS 256
#define GM_ROWS_PER_CTA 2048
#define GM_MAXVEC 256              // Gram-Schmidt coefficients staged in shared memory per pass of k_gm_arnoldi

// Start of a cycle: r = b - w (w = A x, or 0 on the first cycle); beta^2 accumulated in scal[3].
__global__ void __launch_bounds__(GM_THREADS)
k_gm_residual(const int *__restrict__ flags, long n, const double *__restrict__ b, const double *__restrict__ w,
              int use_w, double *__restrict__ r, double *__restrict__ scal)
{
    if (flags[0]) return;
    long i = (long)blockIdx.x * GM_THREADS + threadIdx.x;
    double v = 0.0;
    if (i < n) { v = b[i] - (use_w ? w[i] : 0.0); r[i] = v; }
    double s = block_sum<GM_THREADS>(v * v);
    if (threadIdx.x == 0) atomicAdd(scal + 3, s);
}

// beta = sqrt(scal[3]); first cycle: bnorm = beta.  g = beta e_0; done if beta/bnorm <= tol.
__global__ void k_gm_begin(int *flags, double *scal, double *g, int m, int first, double tol)
{
    if (flags[0]) return;
    double beta = sqrt(scal[3]);
    if (first) scal[0] = beta;
    scal[1] = beta;
    double bn = scal[0];
    scal[2] = bn > 0.0 ? beta / bn : 0.0;
    for (int i = 0; i <= m; i++) g[i] = 0.0;
    g[0] = beta;
    flags[1] = 0;
    if (bn == 0.0 || beta / bn <= tol) { flags[0] = 1; flags[3] = 1; }
    scal[3] = 0.0;
}

// dst = src * (1/s) with s = sqrt(*s2) if is_sq else *s2
__global__ void __launch_bounds__(GM_THREADS)
k_gm_scale(const int *__restrict__ flags, long n, const double *__restrict__ src, const double *__restrict__ s2,
           int is_sq, double *__restrict__ dst)
{
    if (flags[0]) return;
    long i = (long)blockIdx.x * GM_THREADS + threadIdx.x;
    if (i >= n) return;
    double s = is_sq ? sqrt(*s2) : *s2;
    dst[i] = s > 0.0 ? src[i] / s : 0.0;
}

// Back substitution R y = g for the k = flags[1] columns built in this cycle (single thread, k <= m).
__global__ void k_gm_solve_small(const int *__restrict__ flags, int m, const double *__restrict__ H,
                                 const double *__restrict__ g, double *__restrict__ yk)
{
    int k = flags[1];
    for (int i = k - 1; i >= 0; i--) {
        double s = g[i];
        for (int c = i + 1; c < k; c++) s -= H[(long)c * (m + 1) + i] * yk[c];
        const double piv = H[(long)i * (m + 1) + i];
        yk[i] = piv != 0.0 ? s / piv : 0.0;              // zero pivot: breakdown on a singular operator, leave the direction out
    }
}

// x += sum_{i < k} yk[i] V_i
__global__ void __launch_bounds__(GM_THREADS)
k_gm_update(const int *__restrict__ flags, long n, const double *__restrict__ V, const double *__restrict__ yk,
            double *__restrict__ x)
{
    long r = (long)blockIdx.x * GM_THREADS + threadIdx.x;
    if (r >= n) return;
    int k = flags[1];
    double acc = x[r];
    for (int i = 0; i < k; i++) acc += yk[i] * V[(long)i * n + r];
    x[r] = acc;
}

// ---------------------------------------------------------------------------------- block-diagonal M^-1
// Per panel the 2x2 block that couples its two unknowns (phi, dphi/dn) with its two rows (equation of
// region_in, equation of region_out) through the self integrals only:
//     M_j = [[1/2, -V_in,jj], [1/2, c V_out,jj]],   c = eps_in/eps_out,   K_jj = 0.
// pinv[j] = M_j^-1 = (a, b; c, d).  Built once in create.
__global__ void k_precond_build(long npan, QuadTables q, const double *__restrict__ tri,
                                const double4 *__restrict__ pk, double4 *__restrict__ pinv)
{
    long j = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (j >= npan) return;
    const double inv4pi = 0.07957747154594767;
    const double4 k = pk[j];                     // kappa_in, kappa_out, eps_in / eps_out
    const double vin = self_integral(tri + 9 * j, k.x, q) * inv4pi;
    const double vout = self_integral(tri + 9 * j, k.y, q) * inv4pi * k.z;
    const double det = 0.5 * vout + 0.5 * vin;
    pinv[j] = make_double4(vout / det, vin / det, -0.5 / det, 0.5 / det);
}

// z (= or +=) M^-1 u, panel by panel.
__global__ void __launch_bounds__(GM_THREADS)
k_precond_apply(const int *__restrict__ flags, int respect_done, long npan, const double4 *__restrict__ pinv,
                const int2 *__restrict__ pidx, VecRef ur, int add, double *__restrict__ z)
{
    if (respect_done && flags[0]) return;
    long j = (long)blockIdx.x * GM_THREADS + threadIdx.x;
    if (j >= npan) return;
    const double *__restrict__ u = ur.get();
    const int2 ix = pidx[j];
    const double4 m = pinv[j];
    const double u0 = u[ix.x], u1 = u[ix.y];
    const double z0 = m.x * u0 + m.y * u1, z1 = m.z * u0 + m.w * u1;
    if (add) { z[ix.x] += z0; z[ix.y] += z1; } else { z[ix.x] = z0; z[ix.y] = z1; }
}

// ---------------------------------------------------------------------------------- fused Arnoldi step
// One cooperative launch per GMRES iteration instead of nine small ones (zero, dots, axpys, dots, axpys, norm,
// scale, Givens: ~35 us of launch gaps next to a 0.17 ms matvec at config 1).  Each CTA owns a slice of rows;
// the phases are separated by grid-wide barriers:
//   1  h1[i] += V_i . w (slice partials, atomics)                          [h1 is zero on entry]
//   2  w -= sum_i h1[i] V_i on the slice, then h2[i] += V_i . w            (second Gram-Schmidt pass, CGS2)
//   3  w -= sum_i h2[i] V_i, nrm2 += |w|^2
//   4  V_(j+1) = w / sqrt(nrm2) on the slice; one thread: Hessenberg column, Givens, convergence test
// The summation order of the partial dot products is not fixed (atomics, reading A19).
#include <cooperative_groups.h>
__global__ void __launch_bounds__(GM_THREADS)
k_gm_arnoldi(int *flags, double *V, long n, int m, double *w, double *h1, double *h2, double *nrm2, double *H,
             double *cs, double *sn, double *g, double *scal, double tol)
{
    namespace cgx = cooperative_groups;
    if (flags[0]) return;                                    // uniform: set before this launch or not at all
    cgx::grid_group grid = cgx::this_grid();
    // the step number is the count of columns built so far; it is read here by every CTA and rewritten only after
    // the last grid-wide barrier, so one captured launch serves every step
    const int j = flags[1];
    const int nvec = j + 1;
    const long per = (n + gridDim.x - 1) / gridDim.x;
    const long lo = (long)blockIdx.x * per, hi = min(n, lo + per);
    double *vn = V + (long)(j + 1) * n;
    if (blockIdx.x == 0) {
        for (int i = threadIdx.x; i < nvec; i += GM_THREADS) h2[i] = 0.0;
        if (threadIdx.x == 0) *nrm2 = 0.0;
    }
    // The dots of a slice are spread over the warps (warp k takes V_k, V_(k+8), ...; lanes stride over the rows,
    // one shuffle reduction and one atomic per vector) instead of one block reduction with two CTA barriers per
    // vector, which made the step grow by 2.7 us per basis vector (profiles/r2b_launches.csv: 14 ... 50 us).
    __shared__ double s_h[GM_MAXVEC];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    auto slice_dots = [&](double *hout) {
        for (int i = warp; i < nvec; i += GM_THREADS / 32) {
            const double *v = V + (long)i * n;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
            long r = lo + lane;
            for (; r + 96 < hi; r += 128) {
                a0 += v[r] * w[r]; a1 += v[r + 32] * w[r + 32]; a2 += v[r + 64] * w[r + 64]; a3 += v[r + 96] * w[r + 96];
            }
            for (; r < hi; r += 32) a0 += v[r] * w[r];
            double acc = (a0 + a1) + (a2 + a3);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) atomicAdd(hout + i, acc);
        }
    };
    auto slice_update = [&](const double *hin, bool want_norm) {   // w -= sum_i hin[i] V_i on the slice
        double part = 0.0;
        for (int i0 = 0; i0 < nvec; i0 += GM_MAXVEC) {             // coefficients through shared memory, GM_MAXVEC at a time
            const int nv = min(GM_MAXVEC, nvec - i0);
            for (int i = threadIdx.x; i < nv; i += GM_THREADS) s_h[i] = __ldcg(hin + i0 + i);
            __syncthreads();
            const double *Vb = V + (long)i0 * n;
            const bool last = i0 + nv == nvec;
            for (long r = lo + threadIdx.x; r < hi; r += GM_THREADS) {
                double a0 = w[r], a1 = 0.0, a2 = 0.0, a3 = 0.0;
                int i = 0;
                for (; i + 3 < nv; i += 4) {
                    a0 -= s_h[i] * Vb[(long)i * n + r]; a1 -= s_h[i + 1] * Vb[(long)(i + 1) * n + r];
                    a2 -= s_h[i + 2] * Vb[(long)(i + 2) * n + r]; a3 -= s_h[i + 3] * Vb[(long)(i + 3) * n + r];
                }
                for (; i < nv; i++) a0 -= s_h[i] * Vb[(long)i * n + r];
                const double acc = (a0 + a1) + (a2 + a3);
                w[r] = acc;
                if (last) part += acc * acc;
            }
            __syncthreads();                                 // the slice of w is complete, s_h may be rewritten
        }
        return want_norm ? part : 0.0;
    };
    // phase 1
    slice_dots(h1);
    grid.sync();
    // phase 2
    slice_update(h1, false);
    slice_dots(h2);
    grid.sync();
    // phase 3
    {
        const double part = slice_update(h2, true);
        const double s = block_sum<GM_THREADS>(part);
        if (threadIdx.x == 0) atomicAdd(nrm2, s);
    }
    grid.sync();
    // phase 4
    const double nn = sqrt(__ldcg(nrm2));
    for (long r = lo + threadIdx.x; r < hi; r += GM_THREADS) vn[r] = nn > 0.0 ? w[r] / nn : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        double *col = H + (long)j * (m + 1);
        for (int i = 0; i <= j; i++) col[i] = __ldcg(h1 + i) + __ldcg(h2 + i);
        col[j + 1] = nn;
        for (int i = 0; i < j; i++) {
            double t = cs[i] * col[i] + sn[i] * col[i + 1];
            col[i + 1] = -sn[i] * col[i] + cs[i] * col[i + 1];
            col[i] = t;
        }
        double d = hypot(col[j], col[j + 1]);
        double c = d > 0.0 ? col[j] / d : 1.0, s = d > 0.0 ? col[j + 1] / d : 0.0;
        cs[j] = c; sn[j] = s;
        col[j] = d; col[j + 1] = 0.0;
        g[j + 1] = -s * g[j];
        g[j] = c * g[j];
        double rel = fabs(g[j + 1]) / scal[0];
        scal[2] = rel;
        flags[1] = j + 1;
        flags[2] += 1;                       // total iterations
        if (rel <= tol) flags[0] = 1;
        for (int i = 0; i <= j + 1; i++) h1[i] = 0.0;        // invariant: h1 is zero when the next step starts
    }
}
