// build_region.cuh -- everything pygbe_create derives from geometry for one region ("compute
// the tree structure and interaction list only once"): boundary bookkeeping (reading A4), Morton sort,
// octree (a2), target groups + MAC traversal (a5), work items, near-field corrections (a8).
// Host code sizes buffers, scans counts and cuts work items; geometry and lists are made by kernels.
#pragma once
#include "common.cuh"
#include "host_util.cuh"
#include "tables.cuh"
#include "tree.cuh"
#include "nearfield.cuh"
#include "p2p.cuh"
#include "build_lists.cuh"

struct Boundary {
    std::vector<int> gid, phi, dphi, row;
    std::vector<double> cV, cK;
    std::vector<int> surfaces;
};

// Boundary panels of region `id` in surface order, with sigma_S c_S and sigma_S (reading A4):
//   sigma = +1, c = 1 if the region is region_in(S); sigma = -1, c = eps_in(S)/eps_out(S) if region_out(S).
static void collect_boundary(const pygbe_handle *h, int id, Boundary &b)
{
    size_t total = 0;
    for (int s = 0; s < h->nsurf; s++)
        if (h->rin[s] == id || h->rout[s] == id) total += (size_t)h->surf_count[s];
    b.gid.resize(total); b.phi.resize(total); b.dphi.resize(total); b.row.resize(total); b.cV.resize(total); b.cK.resize(total);
    size_t at = 0;
    for (int s = 0; s < h->nsurf; s++) {
        double sigma, c;
        int half;
        if (h->rin[s] == id) { sigma = 1.0; c = 1.0; half = 0; }
        else if (h->rout[s] == id) { sigma = -1.0; c = h->eps[h->rin[s]] / h->eps[h->rout[s]]; half = 1; }
        else continue;
        b.surfaces.push_back(s);
        const long o = h->surf_first[s], N = h->surf_count[s];
#pragma omp parallel for schedule(static) if (N > 20000)
        for (long j = 0; j < N; j++) {
            b.gid[at + j] = (int)(o + j);
            b.phi[at + j] = (int)(2 * o + j);
            b.dphi[at + j] = (int)(2 * o + N + j);
            b.row[at + j] = (int)(2 * o + half * N + j);
            b.cV[at + j] = sigma * c;
            b.cK[at + j] = sigma;
        }
        at += (size_t)N;
    }
}

// Singular / near-singular corrections of region R (a8).  With share != nullptr the sparsity pattern of the
// twin region is reused (same geometry, same lists) and only the values are computed with R's kernel.
static int build_corrections(pygbe_handle *h, Region &R, const QuadTables &qt, const Region *share)
{
    if (share) {
        R.corr_off = share->corr_off; R.corr_col = share->corr_col; R.corr_nnz = share->corr_nnz;
    } else {
        int *d_cnt;
        TRY(h->mem.alloc(&d_cnt, R.np));
        const double thres2 = h->thres > 0 ? h->thres * h->thres : 0.0;
        LAUNCH(h, k_near_find, cdiv((long)R.np * 32, 128), 128, 0, R.np, R.tpos, R.pnrm, R.p2p_off, R.p2p_rng, thres2, 0, d_cnt, nullptr, nullptr);
        std::vector<int> cnt;
        TRY(download(h, cnt, d_cnt, (size_t)R.np));
        std::vector<int> off(R.np + 1, 0);
        long nself = 0;
        for (int t = 0; t < R.np; t++) { off[t + 1] = off[t] + cnt[t]; nself += cnt[t] > 0; }
        R.corr_nnz = off[R.np];
        if (nself != R.np) { pygbe_set_error("internal: a target's own panel is missing from its P2P list"); return PYGBE_ECUDA; }
        TRY(upload(h, &R.corr_off, off));
        TRY(h->mem.alloc(&R.corr_col, R.corr_nnz));
        LAUNCH(h, k_near_find, cdiv((long)R.np * 32, 128), 128, 0, R.np, R.tpos, R.pnrm, R.p2p_off, R.p2p_rng, thres2, 1, d_cnt, R.corr_off, R.corr_col);
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        h->mem.release_one(d_cnt);
    }
    TRY(h->mem.alloc_big(&R.corr_val, R.corr_nnz));
    if (!h->dry) LAUNCH(h, k_near_values, cdiv((long)R.np * 32, 128), 128, 0, R.np, qt, R.yukawa, R.kappa, R.corr_off, R.corr_col, R.gid, h->tri,
           R.tpos, R.pnrm, R.spos, R.cV, R.cK, R.corr_val);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return PYGBE_OK;
}

// Region B lies on the other side of exactly the same surfaces as region A (already built): it shares A's
// Morton order, tree, groups, lists, Gauss points and multipoles; it owns its constants, rows, corrections
// and accumulator.
static int build_region_twin(pygbe_handle *h, Region &B, Region &A, const QuadTables &qt)
{
    Boundary b;
    collect_boundary(h, B.id, b);
    const int id = B.id, nq = B.nq;
    const double eps = B.eps, kappa = B.kappa;
    const bool yuk = B.yukawa;
    B = A;                                  // alias every shared device pointer and the host metadata
    B.id = id; B.eps = eps; B.kappa = kappa; B.yukawa = yuk; B.nq = nq;
    B.twin_of = A.id; B.twin = -1; A.twin = B.id;
    B.qpos = nullptr; B.qid = nullptr;
    // p2p_pairs / m2p_evals stay A's: the counts are (target, source, region) triples, fused or not
    int *d_row_u; double *d_cV_u, *d_cK_u;
    TRY(upload(h, &d_row_u, b.row)); TRY(upload(h, &d_cV_u, b.cV)); TRY(upload(h, &d_cK_u, b.cK));
    TRY(h->mem.alloc(&B.row_idx, B.np)); TRY(h->mem.alloc(&B.cV, B.np)); TRY(h->mem.alloc(&B.cK, B.np));
    TRY(h->mem.alloc(&B.out, B.np)); TRY(h->mem.alloc(&B.corr, B.np));
    LAUNCH(h, k_gather_twin, cdiv(B.np, 256), 256, 0, B.np, A.perm, d_row_u, d_cV_u, d_cK_u, B.row_idx, B.cV, B.cK);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (void *q : {(void *)d_row_u, (void *)d_cV_u, (void *)d_cK_u}) h->mem.release_one(q);
    // constant ratio between the twins' charges: mV_B = rV mV_A, mK_B = -mK_A
    A.twin_rV = b.cV[0] / 1.0;
    {
        Boundary a;
        collect_boundary(h, A.id, a);
        A.twin_rV = b.cV[0] / a.cV[0];
        for (size_t i = 0; i < a.cV.size(); i++)
            if (std::fabs(b.cV[i] - A.twin_rV * a.cV[i]) > 1e-14 * std::fabs(b.cV[i]) || b.cK[i] != -a.cK[i]) {
                pygbe_set_error("internal: twin regions %d/%d do not have a constant charge ratio", A.id, B.id);
                return PYGBE_EINVAL;
            }
    }
    TRY(build_corrections(h, B, qt, &A));
    return PYGBE_OK;
}
