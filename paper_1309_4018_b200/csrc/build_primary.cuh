// build_primary.cuh -- build of a region that owns its tree (see build_region.cuh for the twin case).
#pragma once
#include "build_region.cuh"
#include "farfield.cuh"

static int build_region_primary(pygbe_handle *h, Region &R, const std::vector<double> &tri_host, const QuadTables &qt)
{
    const int K = h->K;
    Boundary b;
    collect_boundary(h, R.id, b);
    R.np = (int)b.gid.size();
    R.npts = R.np * K;
    if (R.np == 0) return PYGBE_OK;
    // root cube around the centroids; longest panel (for the near-field guard of the traversal)
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    double Lmax = 0.0;
    {
        double l0 = 1e300, l1 = 1e300, l2 = 1e300, h0 = -1e300, h1 = -1e300, h2 = -1e300;      // min / max are order-independent
#pragma omp parallel for schedule(static) reduction(min : l0, l1, l2) reduction(max : h0, h1, h2, Lmax) if (R.np > 20000)
        for (int p = 0; p < R.np; p++) {
            const double *t = tri_host.data() + 9 * (size_t)b.gid[p];
            double ux = t[3] - t[0], uy = t[4] - t[1], uz = t[5] - t[2];
            double vx = t[6] - t[0], vy = t[7] - t[1], vz = t[8] - t[2];
            double cx = uy * vz - uz * vy, cy = uz * vx - ux * vz, cz = ux * vy - uy * vx;
            Lmax = std::max(Lmax, std::sqrt(std::sqrt(cx * cx + cy * cy + cz * cz)));   // sqrt(2A), 2A = |cross|
            const double c0 = (t[0] + t[3] + t[6]) / 3.0, c1 = (t[1] + t[4] + t[7]) / 3.0, c2 = (t[2] + t[5] + t[8]) / 3.0;
            l0 = std::min(l0, c0); l1 = std::min(l1, c1); l2 = std::min(l2, c2);
            h0 = std::max(h0, c0); h1 = std::max(h1, c1); h2 = std::max(h2, c2);
        }
        lo[0] = l0; lo[1] = l1; lo[2] = l2; hi[0] = h0; hi[1] = h1; hi[2] = h2;
    }
    R.Lmax = Lmax;
    const double edge = std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]}) * (1.0 + 1e-6) + 1e-9;
    for (int a = 0; a < 3; a++) R.root_c[a] = 0.5 * (lo[a] + hi[a]);
    R.root_edge = edge;

    dbg_t("boundary + bbox (host)");
    // ---- Morton keys, sort, gather into sorted order, Gauss points
    int *d_gid_u, *d_phi_u, *d_dphi_u, *d_row_u, *d_iota;
    double *d_cV_u, *d_cK_u;
    unsigned long long *d_keys_u;
    TRY(upload(h, &d_gid_u, b.gid)); TRY(upload(h, &d_phi_u, b.phi)); TRY(upload(h, &d_dphi_u, b.dphi));
    TRY(upload(h, &d_row_u, b.row)); TRY(upload(h, &d_cV_u, b.cV)); TRY(upload(h, &d_cK_u, b.cK));
    TRY(h->mem.alloc(&d_iota, R.np)); TRY(h->mem.alloc(&R.perm, R.np));
    TRY(h->mem.alloc(&d_keys_u, R.np)); TRY(h->mem.alloc(&R.keys, R.np));
    LAUNCH(h, k_region_keys, cdiv(R.np, 256), 256, 0, h->gcen, d_gid_u, R.np, R.root_c[0] - 0.5 * edge,
           R.root_c[1] - 0.5 * edge, R.root_c[2] - 0.5 * edge, 2097152.0 / edge, d_keys_u, d_iota);
    {   // stable radix sort of (Morton key, panel) by the 63 key bits (blockops.cuh)
        int *hist;
        TRY(h->mem.alloc(&hist, (size_t)256 * radix_sort_ctas(R.np)));
        TRY(radix_sort_pairs(d_keys_u, d_iota, R.keys, R.perm, R.np, 63, hist, h->stream, &h->launches));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        h->mem.release_one(hist);
    }
    TRY(h->mem.alloc(&R.gid, R.np)); TRY(h->mem.alloc(&R.phi_idx, R.np)); TRY(h->mem.alloc(&R.dphi_idx, R.np));
    TRY(h->mem.alloc(&R.row_idx, R.np)); TRY(h->mem.alloc(&R.cV, R.np)); TRY(h->mem.alloc(&R.cK, R.np));
    TRY(h->mem.alloc(&R.tpos, R.np)); TRY(h->mem.alloc(&R.pnrm, R.np));
    TRY(h->mem.alloc(&R.spos, R.npts)); TRY(h->mem.alloc(&R.schg, R.npts));
    TRY(h->mem.alloc(&R.pphi, R.np)); TRY(h->mem.alloc(&R.pdphi, R.np)); TRY(h->mem.alloc(&R.out, R.np)); TRY(h->mem.alloc(&R.corr, R.np)); TRY(h->mem.alloc(&R.pq, R.np));
    LAUNCH(h, k_region_gather, cdiv(R.np, 128), 128, 0, R.np, K, qt, R.perm, d_gid_u, d_phi_u, d_dphi_u, d_row_u,
           d_cV_u, d_cK_u, h->tri, h->gcen, h->gnrm, R.gid, R.phi_idx, R.dphi_idx, R.row_idx, R.cV, R.cK, R.tpos,
           R.pnrm, R.spos);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (void *q : {(void *)d_gid_u, (void *)d_phi_u, (void *)d_dphi_u, (void *)d_row_u, (void *)d_iota,
                    (void *)d_cV_u, (void *)d_cK_u, (void *)d_keys_u})
        h->mem.release_one(q);
    dbg_t("keys, sort, gather");
    TRY(build_tree_and_lists(h, R));
    dbg_t("tree + lists total");
    TRY(build_corrections(h, R, qt, nullptr));
    dbg_t("corrections");
    if (R.n_m2p_items > 0) {
        TRY(h->mem.alloc_big(&R.mom, (size_t)R.ncells * 2 * h->Nc));
        const bool f32 = h->precision == PYGBE_PRECISION_MIXED;
        if (f32) TRY(h->mem.alloc_big(&R.pmomf, (size_t)R.np * 2 * h->Nc)); else TRY(h->mem.alloc_big(&R.pmom, (size_t)R.np * 2 * h->Nc));
        if (R.n_p2m > 0 && !h->dry) {
            if (f32) LAUNCH(h, k_panel_moments<float>, R.n_p2m, PMOM_THREADS, 0, h->P, h->Nc, h->K, h->itab, R.p2m_cells, R.cgeo, R.crange,
                            R.spos, R.pnrm, R.pmomf);
            else LAUNCH(h, k_panel_moments<double>, R.n_p2m, PMOM_THREADS, 0, h->P, h->Nc, h->K, h->itab, R.p2m_cells, R.cgeo, R.crange,
                        R.spos, R.pnrm, R.pmom);
        }
    }
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}
