// solve.cuh -- right-hand side (a10), device-resident restarted GMRES driver (a11), energies (a12, a13).
#pragma once
#include "matvec.cuh"
#include "gmres.cuh"

static int ensure_host_staging(pygbe_handle *h)
{
    if (!h->xh) { TRY(h->mem.alloc_big(&h->xh, 2 * h->npan)); TRY(h->mem.alloc_big(&h->yh, 2 * h->npan)); }
    return PYGBE_OK;
}

static int ensure_energy_scratch(pygbe_handle *h)
{
    if (!h->dq && h->nq > 0) {
        TRY(h->mem.alloc_big(&h->dq, h->nq));
        if (!h->dry) CUDA_TRY(cudaMemcpyAsync(h->dq, h->qq.data(), h->nq * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    }
    return PYGBE_OK;
}


// ---------------------------------------------------------------------------------------------- rhs
extern "C" int pygbe_rhs(pygbe_handle *h, double *b_dev)
{
    if (!h || !b_dev) { pygbe_set_error("rhs: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaMemsetAsync(b_dev, 0, 2 * h->npan * sizeof(double), h->stream));
    const double inv4pi = 0.07957747154594767;
    for (Region &R : h->regions) {
        if (R.nq == 0 || R.np == 0) continue;
        if (R.yukawa)
            LAUNCH(h, k_rhs<true>, cdiv(R.np, 128), 128, 0, R.np, R.tpos, R.row_idx, R.nq, R.qpos, R.kappa, inv4pi / R.eps, b_dev);
        else
            LAUNCH(h, k_rhs<false>, cdiv(R.np, 128), 128, 0, R.np, R.tpos, R.row_idx, R.nq, R.qpos, R.kappa, inv4pi / R.eps, b_dev);
    }
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}

// -------------------------------------------------------------------------------------------- gmres
static int ensure_gmres(pygbe_handle *h, int m)
{
    GmresWork &G = h->gm;
    long n = 2 * h->npan;
    if (G.V && G.m >= m) return PYGBE_OK;
    if (G.V) {
        for (void *q : {(void *)G.V, (void *)G.H, (void *)G.h1, (void *)G.h2, (void *)G.cs, (void *)G.sn, (void *)G.g, (void *)G.yk})
            h->mem.release_one(q);
    }
    G.m = m; G.n = n;
    TRY(h->mem.alloc_big(&G.V, (size_t)(m + 1) * n));
    TRY(h->mem.alloc(&G.H, (size_t)(m + 1) * m));
    TRY(h->mem.alloc(&G.h1, m + 2)); TRY(h->mem.alloc(&G.h2, m + 2)); TRY(h->mem.alloc(&G.cs, m + 1));
    TRY(h->mem.alloc(&G.sn, m + 1)); TRY(h->mem.alloc(&G.g, m + 2)); TRY(h->mem.alloc(&G.yk, m + 1));
    if (!G.w) {
        TRY(h->mem.alloc_big(&G.w, n)); TRY(h->mem.alloc_big(&G.b, n)); TRY(h->mem.alloc(&G.scal, 8)); TRY(h->mem.alloc(&G.flags, 4));
    }
    return PYGBE_OK;
}

extern "C" int pygbe_solve(pygbe_handle *h, double tol, int32_t restart, int32_t max_iter, double *x_dev,
                           int32_t *iters, double *rel_resid)
{
    if (!h || !x_dev) { pygbe_set_error("solve: null pointer"); return PYGBE_EINVAL; }
    if (!(tol > 0.0) || restart < 1 || max_iter < 1) { pygbe_set_error("solve: bad tol / restart / max_iter"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    double t0 = now_ms();
    const long n = 2 * h->npan;
    const int m = std::min(restart, max_iter);
    TRY(ensure_gmres(h, m));
    GmresWork &G = h->gm;
    const int ldh = G.m + 1;     // H was sized with G.m
    (void)ldh;
    cudaStream_t st = h->stream;
    const int gridn = cdiv(n, GM_THREADS), gridd = cdiv(n, GM_ROWS_PER_CTA);
    TRY(pygbe_rhs(h, G.b));
    CUDA_TRY(cudaMemsetAsync(x_dev, 0, n * sizeof(double), st));
    CUDA_TRY(cudaMemsetAsync(G.flags, 0, 4 * sizeof(int), st));
    CUDA_TRY(cudaMemsetAsync(G.scal, 0, 8 * sizeof(double), st));
    const int poll = n < 200000 ? 4 : 1;
    int arn_grid = 1;
    {
        int occ = 1;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_gm_arnoldi, GM_THREADS, 0));
        const long arn_rows = tune_env("PYGBE_ARN_ROWS") ? std::max(32L, atol(tune_env("PYGBE_ARN_ROWS"))) : 256L;   // tuning
        arn_grid = (int)std::max(1L, std::min((long)occ * h->n_sm, (long)cdiv(n, arn_rows)));
    }
    CUDA_TRY(cudaMemsetAsync(G.h1, 0, (size_t)(G.m + 2) * sizeof(double), st));   // k_gm_arnoldi keeps h1 zero between steps
    const bool pc = h->precond == 1 && h->pinv != nullptr;
    TRY(set_slots(h, 2, G.V, G.w));                                 // input base and output of the iteration's matvec
    // Cycle = [residual b - A x by a matvec, convergence test on it] + up to m Arnoldi steps + update of x.  A cycle
    // ends early when the Arnoldi estimate reaches tol; convergence is declared only by the next cycle's recomputed
    // residual (one extra matvec per solve).  If that residual is above tol the iteration simply goes on; after
    // three such disagreements tol is below what the operator's arithmetic attains and the solve returns ENOCONV
    // with the true residual (PRECISION_MIXED: about 1e-6 relative).
    int total = 0, converged = 0, disagreements = 0;
    bool first = true;
    while (!converged) {
        if (!first) {
            CUDA_TRY(cudaMemsetAsync(G.flags, 0, sizeof(int), st));             // clear "stop", keep the counters
            CUDA_TRY(cudaMemsetAsync(G.scal + 3, 0, sizeof(double), st));
            TRY(matvec_run(h, x_dev, G.w));
        }
        LAUNCH(h, k_gm_residual, gridn, GM_THREADS, 0, G.flags, n, G.b, G.w, first ? 0 : 1, G.V, G.scal);
        LAUNCH(h, k_gm_begin, 1, 1, 0, G.flags, G.scal, G.g, G.m, first ? 1 : 0, tol);
        LAUNCH(h, k_gm_scale, gridn, GM_THREADS, 0, G.flags, n, G.V, G.scal + 1, 0, G.V);
        const int mc = std::min(m, max_iter - total);
        if (!first || mc <= 0) {                          // the verdict of k_gm_begin on the recomputed residual, before queueing a cycle
            CUDA_TRY(cudaMemcpyAsync(h->pinned_flags, G.flags, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaMemcpyAsync(h->pinned_scal, G.scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            if (h->pinned_flags[3]) { converged = 1; break; }
            if (mc <= 0) break;                           // out of iterations
        }
        first = false;
        // One Arnoldi step = [M^-1 v_j] + matvec + one cooperative launch (CGS2, normalisation, Givens, convergence
        // estimate; gmres.cuh).  The step number lives on the device (flags[1]), so the same launches serve every
        // step: `poll` of them are captured once as a CUDA graph and replayed; the host reads the flags in between.
        auto one_step = [&]() -> int {
            if (pc) {           // right preconditioning: w = A (M^-1 v_j)
                LAUNCH(h, k_precond_apply, cdiv(h->npan, GM_THREADS), GM_THREADS, 0, G.flags, 1, h->npan, h->pinv, h->pidx,
                       vec_slot(h->io + 2, G.flags + 1, n), 0, h->zbuf);
                TRY(matvec_impl(h, vec_direct(h->zbuf), vec_slot(h->io + 3), G.flags));
            } else {
                TRY(matvec_impl(h, vec_slot(h->io + 2, G.flags + 1, n), vec_slot(h->io + 3), G.flags));
            }
            long nn = n; int mm = G.m; double tl = tol;
            double *nrm2 = G.scal + 3;
            void *args[] = {&G.flags, &G.V, &nn, &mm, &G.w, &G.h1, &G.h2, &nrm2, &G.H, &G.cs, &G.sn, &G.g, &G.scal, &tl};
            CUDA_TRY(cudaLaunchCooperativeKernel((const void *)k_gm_arnoldi, dim3(arn_grid), dim3(GM_THREADS), args, 0, h->stream));
            h->launches++;
            return PYGBE_OK;
        };
        bool graph = h->use_graphs && !h->profile && !h->g_iter.failed;
        if (graph) {
            long tolbits; memcpy(&tolbits, &tol, sizeof(tolbits));
            const long key[6] = {(long)(uintptr_t)G.V, (long)G.m, tolbits, (long)poll, (long)pc, (long)arn_grid};
            if (!h->g_iter.exec || memcmp(key, h->g_iter.key, sizeof(key)) != 0) {
                graph = graph_capture(h, h->g_iter, [&]() -> int { for (int q = 0; q < poll; q++) TRY(one_step()); return PYGBE_OK; });
                if (graph) memcpy(h->g_iter.key, key, sizeof(key));
            }
        }
        for (int j = 0; j < mc;) {
            if (graph && j + poll <= mc) { TRY(graph_launch(h, h->g_iter)); j += poll; }
            else { TRY(one_step()); j++; if (j % poll != 0 && j != mc) continue; }
            CUDA_TRY(cudaMemcpyAsync(h->pinned_flags, G.flags, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            if (h->pinned_flags[0]) break;
        }
        LAUNCH(h, k_gm_solve_small, 1, 1, 0, G.flags, G.m, G.H, G.g, G.yk);
        if (pc) {               // x += M^-1 (V y)
            CUDA_TRY(cudaMemsetAsync(h->zbuf, 0, n * sizeof(double), st));
            LAUNCH(h, k_gm_update, gridn, GM_THREADS, 0, G.flags, n, G.V, G.yk, h->zbuf);
            LAUNCH(h, k_precond_apply, cdiv(h->npan, GM_THREADS), GM_THREADS, 0, G.flags, 0, h->npan, h->pinv, h->pidx, vec_direct(h->zbuf), 1, x_dev);
        } else {
            LAUNCH(h, k_gm_update, gridn, GM_THREADS, 0, G.flags, n, G.V, G.yk, x_dev);
        }
        CUDA_TRY(cudaMemcpyAsync(h->pinned_flags, G.flags, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaMemcpyAsync(h->pinned_scal, G.scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        total = h->pinned_flags[2];
        if (h->pinned_flags[3]) { converged = 1; break; }                       // b = 0, or the recomputed residual was within tol
        if (h->pinned_flags[0] && ++disagreements > 3) {                        // the estimate keeps saying "done", the residual does not
            CUDA_TRY(cudaMemsetAsync(G.flags, 0, sizeof(int), st));
            CUDA_TRY(cudaMemsetAsync(G.scal + 3, 0, sizeof(double), st));
            TRY(matvec_run(h, x_dev, G.w));
            LAUNCH(h, k_gm_residual, gridn, GM_THREADS, 0, G.flags, n, G.b, G.w, 1, G.V, G.scal);
            LAUNCH(h, k_gm_begin, 1, 1, 0, G.flags, G.scal, G.g, G.m, 0, tol);
            CUDA_TRY(cudaMemcpyAsync(h->pinned_flags, G.flags, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaMemcpyAsync(h->pinned_scal, G.scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            converged = h->pinned_flags[3];
            break;
        }
    }
    CUDA_TRY(cudaGetLastError());
    h->last_iters = total;
    h->last_solve_ms = now_ms() - t0;
    if (iters) *iters = total;
    if (rel_resid) *rel_resid = h->pinned_scal[2];
    if (!converged) {
        pygbe_set_error("GMRES: %d iterations, relative residual %.3e > tol %.3e%s", total, h->pinned_scal[2], tol,
                        disagreements > 3 ? " (the Arnoldi estimate is below tol but the recomputed residual b - A x is not: tol is below what this precision attains)" : "");
        return PYGBE_ENOCONV;
    }
    return PYGBE_OK;
}

// ------------------------------------------------------------------------------------------- energy
extern "C" int pygbe_reaction_potential(pygbe_handle *h, const double *x_dev, double *phi_dev)
{
    if (!h || !x_dev || !phi_dev) { pygbe_set_error("reaction_potential: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    if (h->nq == 0) return PYGBE_OK;
    CUDA_TRY(cudaMemsetAsync(phi_dev, 0, h->nq * sizeof(double), h->stream));
    for (Region &R : h->regions) {
        if (R.nq == 0) continue;
        LAUNCH(h, k_prep, cdiv((long)R.np * h->K, 256), 256, 0, nullptr, R.np, h->K, vec_direct(x_dev), R.phi_idx, R.dphi_idx, R.cV, R.cK, R.pnrm,
               R.spos, R.schg, (float4 *)nullptr, 0, R.pphi, R.pdphi, R.pq, R.out, (double *)nullptr);
        // chunks of Gauss points on grid.y: at most 65535 of them
        const long en_chunks = cdiv(R.npts, EN_CHUNK);
        if (en_chunks > 65535) { pygbe_set_error("reaction potential: region %d has too many Gauss points (%d)", R.id, R.npts); return PYGBE_EINVAL; }
        dim3 grid(R.nq, (unsigned)en_chunks);
        if (R.yukawa) LAUNCH(h, k_reaction<true>, grid, EN_THREADS, 0, R.npts, R.spos, R.schg, R.nq, R.qpos, R.qid, R.kappa, phi_dev);
        else LAUNCH(h, k_reaction<false>, grid, EN_THREADS, 0, R.npts, R.spos, R.schg, R.nq, R.qpos, R.qid, R.kappa, phi_dev);
    }
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}

static double unit_C0()
{   // reading A17: qe^2 N_A 1e-3 1e10 / eps0 in kJ Angstrom / (mol e^2); reproduces PAPER.md:229
    const double qe = 1.60217646e-19, NA = 6.0221415e23, eps0 = 8.854187818e-12;
    return qe * qe * NA * 1e7 / eps0;
}

extern "C" int pygbe_energy(pygbe_handle *h, const double *x_dev, double *E_solv, double *E_coul)
{
    if (!h || !x_dev) { pygbe_set_error("energy: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    const double C0 = unit_C0();
    if (E_solv) *E_solv = 0.0;
    if (E_coul) *E_coul = 0.0;
    if (h->nq == 0) return PYGBE_OK;
    if (E_solv) {
        TRY(pygbe_reaction_potential(h, x_dev, h->phi_reac));
        TRY(ensure_energy_scratch(h));
        LAUNCH(h, k_dot_q, 1, 256, 0, (int)h->nq, h->dq, h->phi_reac, h->scratch);
        CUDA_TRY(cudaMemcpyAsync(h->pinned_scal, h->scratch, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        *E_solv = 0.5 * C0 * h->pinned_scal[0];
    }
    if (E_coul) {
        double tot = 0.0;
        for (Region &R : h->regions) {
            if (R.nq < 2) continue;
            CUDA_TRY(cudaMemsetAsync(h->scratch + 1, 0, sizeof(double), h->stream));
            LAUNCH(h, k_coulomb, cdiv(R.nq, 128), 128, 0, R.nq, R.qpos, h->scratch + 1);
            CUDA_TRY(cudaMemcpyAsync(h->pinned_scal + 1, h->scratch + 1, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
            CUDA_TRY(cudaStreamSynchronize(h->stream));
            tot += h->pinned_scal[1] / (4.0 * 3.14159265358979323846 * R.eps);
        }
        *E_coul = 0.5 * C0 * tot;
    }
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}

extern "C" int pygbe_solve_host(pygbe_handle *h, double tol, int32_t restart, int32_t max_iter, double *x_host,
                                int32_t *iters, double *rel_resid, double *E_solv, double *E_coul)
{
    if (!h) { pygbe_set_error("solve_host: null handle"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    TRY(ensure_host_staging(h));
    int rc = pygbe_solve(h, tol, restart, max_iter, h->xh, iters, rel_resid);
    if (rc != PYGBE_OK && rc != PYGBE_ENOCONV) return rc;
    if (x_host) {
        CUDA_TRY(cudaMemcpyAsync(x_host, h->xh, 2 * h->npan * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
    }
    TRY(pygbe_energy(h, h->xh, E_solv, E_coul));
    return rc;
}

