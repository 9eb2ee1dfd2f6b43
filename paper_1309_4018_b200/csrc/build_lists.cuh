// build_lists.cuh -- octree (a2), target groups, MAC traversal (a5) and work items of one region.
#pragma once
#include "common.cuh"
#include "host_util.cuh"
#include "tree.cuh"
#include "p2p.cuh"

// Per-panel constants of a twin region, gathered into the primary region's Morton order.
__global__ void k_gather_twin(int np, const int *__restrict__ perm, const int *__restrict__ row_u,
                              const double *__restrict__ cV_u, const double *__restrict__ cK_u,
                              int *__restrict__ row_idx, double *__restrict__ cV, double *__restrict__ cK)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    int u = perm[p];
    row_idx[p] = row_u[u]; cV[p] = cV_u[u]; cK[p] = cK_u[u];
}

static int build_tree_and_lists(pygbe_handle *h, Region &R)
{
    const int K = h->K;
    const double edge = R.root_edge;
    // ---- octree: split level by level until no cell holds more than ncrit panels
    const int ncrit = h->ncrit;
    long maxcells = 64 + 8L * (R.np / std::max(1, ncrit) + 1) * 12;
    int *d_ncells;
    TRY(h->mem.alloc(&R.cgeo, maxcells)); TRY(h->mem.alloc(&R.crange, maxcells)); TRY(h->mem.alloc(&R.cchild, maxcells));
    TRY(h->mem.alloc(&R.cparent, maxcells)); TRY(h->mem.alloc(&R.ckey, maxcells)); TRY(h->mem.alloc(&d_ncells, 1));
    {
        double4 g0 = make_double4(R.root_c[0], R.root_c[1], R.root_c[2], edge);
        int2 r0 = make_int2(0, R.np), c0 = make_int2(-1, 0);
        int par = -1, one = 1;
        unsigned long long k0 = 0;
        CUDA_TRY(cudaMemcpyAsync(R.cgeo, &g0, sizeof(g0), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaMemcpyAsync(R.crange, &r0, sizeof(r0), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaMemcpyAsync(R.cchild, &c0, sizeof(c0), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaMemcpyAsync(R.cparent, &par, sizeof(par), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaMemcpyAsync(R.ckey, &k0, sizeof(k0), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaMemcpyAsync(d_ncells, &one, sizeof(one), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
    }
    R.level_begin.clear();
    R.level_begin.push_back(0);
    int ncells = 1;
    for (int level = 0; level <= PYGBE_MAXLEVEL; level++) {
        int b = R.level_begin[level], e = ncells;
        R.level_begin.push_back(e);
        if (b == e) { R.level_begin.pop_back(); break; }
        LAUNCH(h, k_split_level, 1, SPLIT_THREADS, 0, R.keys, level, b, e, ncrit, (int)maxcells, R.cgeo, R.crange,
               R.cchild, R.cparent, R.ckey, d_ncells);
        CUDA_TRY(cudaMemcpyAsync(&ncells, d_ncells, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        if (ncells > maxcells) { pygbe_set_error("octree needs %d cells, capacity %ld", ncells, maxcells); return PYGBE_ENOMEM; }
    }
    R.ncells = ncells;
    R.depth = (int)R.level_begin.size() - 1;      // number of levels
    h->mem.release_one(d_ncells);
    std::vector<int2> crange_h, cchild_h;
    std::vector<int> cparent_h;
    TRY(download(h, crange_h, R.crange, (size_t)ncells));
    TRY(download(h, cchild_h, R.cchild, (size_t)ncells));
    TRY(download(h, cparent_h, R.cparent, (size_t)ncells));
    std::vector<int> clevel(ncells, 0);
    for (int l = 0; l < R.depth; l++)
        for (int c = R.level_begin[l]; c < R.level_begin[l + 1]; c++) clevel[c] = l;
    std::vector<int> leaves;
    for (int c = 0; c < ncells; c++)
        if (cchild_h[c].y == 0) leaves.push_back(c);
    std::sort(leaves.begin(), leaves.end(), [&](int a, int b) { return crange_h[a].x < crange_h[b].x; });
    R.nleaves = (int)leaves.size();
    TRY(upload(h, &R.leaf_cell, leaves));

    dbg_t("  octree split + download");
    // ---- anchors (mixed precision): the ancestor of each leaf at the level where cells are <= 16 A wide
    const bool mixed = h->precision == PYGBE_PRECISION_MIXED;
    std::vector<int> anchor_of(ncells, 0);
    if (mixed) {
        int alevel = 0;
        const double anchor_edge = tune_env("PYGBE_ANCHOR_EDGE") ? atof(tune_env("PYGBE_ANCHOR_EDGE")) : 16.0;   // tuning
        while (edge / (double)(1 << alevel) > anchor_edge && alevel < PYGBE_MAXLEVEL) alevel++;
        std::vector<int> panel_anchor(R.np, 0);
        for (int c : leaves) {
            int a = c;
            while (clevel[a] > alevel) a = cparent_h[a];
            anchor_of[c] = a;
            for (int p = crange_h[c].x; p < crange_h[c].y; p++) panel_anchor[p] = a;
        }
        TRY(upload(h, &R.panel_anchor, panel_anchor));
        TRY(h->mem.alloc(&R.sposf, R.npts)); TRY(h->mem.alloc(&R.schgf, R.npts));
        R.quad = K % 4 == 0;                  // packed-fp32 P2P on quads of Gauss points (p2p.cuh)
        if (R.quad) LAUNCH(h, k_make_sposq, cdiv(R.npts, 256), 256, 0, R.np, K, R.panel_anchor, R.cgeo, R.spos, (float *)R.sposf);
        else LAUNCH(h, k_make_sposf, cdiv(R.np, 128), 128, 0, R.np, K, R.panel_anchor, R.cgeo, R.spos, R.sposf);
    }

    // ---- target groups + traversal (count, offsets, fill)
    R.ng = cdiv(R.np, PYGBE_TG);
    TRY(h->mem.alloc(&R.ggeo, 2 * (size_t)R.ng));
    LAUNCH(h, k_group_geometry, R.ng, PYGBE_TG, 0, R.tpos, R.np, R.ggeo);
    int *d_mcnt, *d_pcnt, *d_over;
    TRY(h->mem.alloc(&d_mcnt, R.ng)); TRY(h->mem.alloc(&d_pcnt, R.ng)); TRY(h->mem.alloc(&d_over, 1));
    CUDA_TRY(cudaMemsetAsync(d_over, 0, sizeof(int), h->stream));
    double *d_clmax;
    TRY(h->mem.alloc(&d_clmax, (size_t)ncells));
    LAUNCH(h, k_cell_lmax, cdiv((long)ncells * 32, 128), 128, 0, ncells, R.crange, R.tpos, d_clmax);
    const double thres_guard = h->thres > 0 ? h->thres : 0.0;
    // break-even between one Taylor evaluation and the direct sum over a leaf's points: a regrouped M2P
    // evaluation costs Nc - 1 + NW FMA-pipe instructions per region, a P2P pair ~14 per region, and the sweep of
    // profiles/r2a_regrouped_path.md puts the optimum at ~16 points for P = 6 (344 instructions) in both precisions
    // (the Laplace form costs Nc - 1 FMAs)
    // (regrouped form on reduced moments: (P+1)^2 monomials + NW FMAs per region)
    int small_leaf = (int)(16.0 * (R.lap ? (double)h->Nc : (h->P + 1.0) * (h->P + 1.0) + 2.0 * h->NW) / 344.0 / K);
    if (const char *e = tune_env("PYGBE_SMALL_LEAF")) small_leaf = atoi(e);                     // tuning
    const int exact_mac = h->group_mac == 0 ? 1 : 0;             // 1 = group MAC on the group's own points
    LAUNCH(h, k_traverse, cdiv(R.ng, TRAV_WARPS), TRAV_WARPS * 32, 0, R.ng, R.tpos, R.np, exact_mac, R.ggeo, R.cgeo, R.crange, R.cchild,
           h->theta, thres_guard, d_clmax, small_leaf, 0, d_mcnt, d_pcnt, nullptr, nullptr, nullptr, nullptr, d_over);
    std::vector<int> mcnt, pcnt;
    TRY(download(h, mcnt, d_mcnt, (size_t)R.ng));
    TRY(download(h, pcnt, d_pcnt, (size_t)R.ng));
    std::vector<int> moff(R.ng + 1, 0), poff(R.ng + 1, 0);
    for (int g = 0; g < R.ng; g++) { moff[g + 1] = moff[g] + mcnt[g]; poff[g + 1] = poff[g] + pcnt[g]; }
    int *d_poff_raw, *d_pleaf_raw;
    TRY(upload(h, &R.m2p_off, moff)); TRY(upload(h, &d_poff_raw, poff));
    TRY(h->mem.alloc(&R.m2p_cell, moff[R.ng])); TRY(h->mem.alloc(&d_pleaf_raw, poff[R.ng]));
    LAUNCH(h, k_traverse, cdiv(R.ng, TRAV_WARPS), TRAV_WARPS * 32, 0, R.ng, R.tpos, R.np, exact_mac, R.ggeo, R.cgeo, R.crange, R.cchild,
           h->theta, thres_guard, d_clmax, small_leaf, 1, d_mcnt, d_pcnt, R.m2p_off, d_poff_raw, R.m2p_cell, d_pleaf_raw, d_over);
    std::vector<int> pleaf;
    TRY(download(h, pleaf, d_pleaf_raw, (size_t)poff[R.ng]));
    {   // multipoles are needed for the listed cells and, to build those by M2M, for all their descendants
        std::vector<int> mcell;
        TRY(download(h, mcell, R.m2p_cell, (size_t)moff[R.ng]));
        std::vector<char> need(ncells, 0);
        for (int c : mcell) need[c] = 1;
        for (int c = 1; c < ncells; c++)                  // parents precede children in the numbering
            if (need[cparent_h[c]]) need[c] = 1;
        std::vector<int> p2m_cells;
        std::vector<int4> m2m_rec;
        for (int c : leaves) if (need[c]) p2m_cells.push_back(c);
        for (int l = R.depth - 1; l >= 0; l--)              // deepest level first: children before parents
            for (int c = R.level_begin[l]; c < R.level_begin[l + 1]; c++)
                if (need[c] && cchild_h[c].y > 0) {
                    int mask = 0;
                    for (int k = 0; k < cchild_h[c].y; k++)
                        if (cchild_h[cchild_h[c].x + k].y > 0) mask |= 1 << k;
                    m2m_rec.push_back(make_int4(c, cchild_h[c].x, cchild_h[c].y, mask));
                }
        R.n_m2m = (int)m2m_rec.size();
        R.n_p2m = (int)p2m_cells.size();
        R.p2m_panels = 0; R.m2m_children = 0;
        for (int c : p2m_cells) R.p2m_panels += crange_h[c].y - crange_h[c].x;
        for (const int4 &m : m2m_rec) R.m2m_children += m.z;
        TRY(upload(h, &R.p2m_cells, p2m_cells)); TRY(upload(h, &R.m2m_rec, m2m_rec));
        std::vector<int4> p2m_rec;
        for (int c : p2m_cells) p2m_rec.push_back(make_int4(c, crange_h[c].x, crange_h[c].y, 0));
        TRY(upload(h, &R.p2m_rec, p2m_rec));
        TRY(h->mem.alloc(&R.up_sync, 4)); TRY(h->mem.alloc(&R.cready, (size_t)ncells));
        CUDA_TRY(cudaMemsetAsync(R.up_sync, 0, 4 * sizeof(int), h->stream));
        CUDA_TRY(cudaMemsetAsync(R.cready, 0, (size_t)ncells * sizeof(int), h->stream));
    }
    int over = 0;
    CUDA_TRY(cudaMemcpy(&over, d_over, sizeof(int), cudaMemcpyDeviceToHost));
    if (over) { pygbe_set_error("traversal stack overflow"); return PYGBE_ECUDA; }
    for (void *q : {(void *)d_mcnt, (void *)d_pcnt, (void *)d_over, (void *)d_poff_raw, (void *)d_pleaf_raw, (void *)d_clmax})
        h->mem.release_one(q);

    dbg_t("  anchors, groups, traversal");
    // ---- P2P lists: leaves -> panel ranges sorted by position; adjacent ranges with the same anchor merge.
    // Host work over ~17 k groups x ~30 leaves at 1 M panels: every group is independent, so the loops run in
    // parallel (OpenMP) into per-group slots and are compacted by prefix sums; the result does not depend on the
    // number of threads.
    const int ng = R.ng;
    const bool par = R.np > 20000;
    std::vector<int4> prng_raw((size_t)poff[ng]);       // merged ranges of group g at [poff[g], poff[g] + rcnt[g])
    std::vector<int> rcnt(ng, 0);
    long total_src_panels = 0, p2p_pairs = 0, m2p_evals = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : total_src_panels, p2p_pairs, m2p_evals) if (par)
    for (int g = 0; g < ng; g++) {
        int4 *dst = prng_raw.data() + poff[g];
        const int nl = poff[g + 1] - poff[g];
        for (int r = 0; r < nl; r++) {
            const int c = pleaf[poff[g] + r];
            dst[r] = make_int4(crange_h[c].x, crange_h[c].y, anchor_of[c], 0);
        }
        // the traversal emits a group's leaves in Morton order, i.e. by ascending panel range: sort only if not
        auto by_pos = [](const int4 &a, const int4 &b) { return a.x < b.x; };
        if (!std::is_sorted(dst, dst + nl, by_pos)) std::sort(dst, dst + nl, by_pos);
        int n = 0;
        for (int r = 0; r < nl; r++) {
            if (n > 0 && dst[n - 1].y == dst[r].x && dst[n - 1].z == dst[r].z) dst[n - 1].y = dst[r].y;
            else dst[n++] = dst[r];
        }
        rcnt[g] = n;
        const long ntg = std::min(PYGBE_TG, R.np - g * PYGBE_TG);
        long src = 0;
        for (int r = 0; r < n; r++) src += dst[r].y - dst[r].x;
        total_src_panels += src;
        p2p_pairs += ntg * src * K;
        m2p_evals += ntg * mcnt[g];
    }
    R.p2p_pairs = p2p_pairs; R.m2p_evals = m2p_evals;
    std::vector<int> poff2(ng + 1, 0);
    for (int g = 0; g < ng; g++) poff2[g + 1] = poff2[g] + rcnt[g];
    std::vector<int4> prng((size_t)poff2[ng]);           // merged ranges, CSR by group
#pragma omp parallel for schedule(static) if (par)
    for (int g = 0; g < ng; g++) std::copy(prng_raw.begin() + poff[g], prng_raw.begin() + poff[g] + rcnt[g], prng.begin() + poff2[g]);
    TRY(upload(h, &R.p2p_off, poff2)); TRY(upload(h, &R.p2p_rng, prng));

    dbg_t("  P2P ranges (host)");
    // ---- work items of bounded size, enough of them to fill 148 SMs several times over
    const long want_items = 148L * 16;
    // M2P CTAs keep only 8-20 warps per SM resident (72-127 registers): finer items even out the tail (config 1:
    // 4 cells per item 0.057 ms, 8 cells 0.060, 16 cells 0.068)
    int m2p_item = (int)std::min(64L, std::max(4L, (long)moff[ng] / (6 * want_items)));
    if (R.lap) m2p_item = std::max(m2p_item, 12);            // k_m2p_lap stages up to 12 cells at a time
    m2p_item = (m2p_item + 3) / 4 * 4;
    if (const char *e = tune_env("PYGBE_M2P_ITEM")) m2p_item = std::max(1, atoi(e));                 // tuning
    // P2P tiles gather up to P2P_TILE source points from several panel ranges of one anchor cell: a group's near
    // field is ~30 short runs of Morton-consecutive panels (one or two leaves each), and tiles cut range by range
    // were 62 % full with a third of them under a quarter (config 1).  tile = (first segment, last segment + 1,
    // anchor cell, 2 * points + self flag), segment = (first point, points), whole panels only; self flag = the
    // tile holds panels of the group's own targets, the only place where a pair at zero distance can occur
    // (reading A5).
    const int tile_panels = std::max(1, P2P_TILE / K);
    // pass 1 (parallel): tiles and segments of every group with group-local segment indices
    std::vector<std::vector<int4>> gsub(ng);
    std::vector<std::vector<int2>> gseg(ng);
#pragma omp parallel if (par)
    {
        std::vector<int4> grng;
#pragma omp for schedule(dynamic, 64)
        for (int g = 0; g < ng; g++) {
            grng.assign(prng.begin() + poff2[g], prng.begin() + poff2[g + 1]);
            std::stable_sort(grng.begin(), grng.end(), [](const int4 &a, const int4 &b) { return a.z < b.z; });
            const int own_lo = g * PYGBE_TG, own_hi = std::min(R.np, own_lo + PYGBE_TG);
            std::vector<int4> &sub = gsub[g];
            std::vector<int2> &segs = gseg[g];
            int fill = 0;                                              // panels in the open tile (sub.back())
            for (size_t r = 0; r < grng.size(); r++) {
                if (r > 0 && grng[r].z != grng[r - 1].z) fill = 0;     // another anchor: close the tile
                int a = grng[r].x;
                while (a < grng[r].y) {
                    if (fill == 0 || fill == tile_panels) {
                        sub.push_back(make_int4((int)segs.size(), (int)segs.size(), grng[r].z, 0));
                        fill = 0;
                    }
                    const int take = std::min(grng[r].y - a, tile_panels - fill);
                    segs.push_back(make_int2(a * K, take * K));
                    int4 &t = sub.back();
                    t.y = (int)segs.size();
                    t.w += 2 * take * K;
                    if (a < own_hi && a + take > own_lo) t.w |= 1;
                    a += take; fill += take;
                }
            }
        }
    }
    std::vector<int> gtile(ng + 1, 0), gsegoff(ng + 1, 0), gmit(ng + 1, 0);   // first tile / segment / M2P item of each group
    for (int g = 0; g < ng; g++) {
        gtile[g + 1] = gtile[g] + (int)gsub[g].size();
        gsegoff[g + 1] = gsegoff[g] + (int)gseg[g].size();
        gmit[g + 1] = gmit[g] + (moff[g + 1] - moff[g] + m2p_item - 1) / m2p_item;
    }
    // items = short runs of a group's tiles.  An SM holds ~12 of these CTAs, which share its pipes, so an item of n
    // tiles lasts about n / 1100 of the whole launch at config 1 (13 k tiles): equal items of 5 tiles left a tail
    // of a fifth of the kernel, single tiles none (the double buffer then only hides the first tile's latency
    // behind other CTAs).  Large problems take longer runs to save the per-item target loads and atomics.
    const long slots = 148L * 12;
    int per_item = (int)std::min(8L, std::max(1L, (long)gtile[ng] / (slots * 24)));
    if (const char *e = tune_env("PYGBE_P2P_ITEM_TILES")) per_item = std::max(1, atoi(e));      // tuning
    std::vector<int> gpit(ng + 1, 0);
    for (int g = 0; g < ng; g++) gpit[g + 1] = gpit[g] + ((int)gsub[g].size() + per_item - 1) / per_item;
    // pass 2 (parallel): concatenate with global indices
    std::vector<int4> sub((size_t)gtile[ng]), pitems((size_t)gpit[ng]), mitems((size_t)gmit[ng]);
    std::vector<int2> segs((size_t)gsegoff[ng]);
#pragma omp parallel for schedule(static) if (par)
    for (int g = 0; g < ng; g++) {
        const int nt = (int)gsub[g].size();
        for (int t = 0; t < nt; t++) {
            int4 v = gsub[g][t];
            v.x += gsegoff[g]; v.y += gsegoff[g];
            sub[gtile[g] + t] = v;
        }
        std::copy(gseg[g].begin(), gseg[g].end(), segs.begin() + gsegoff[g]);
        int at = gpit[g];
        for (int t = 0; t < nt; t += per_item) {
            const int n = std::min(per_item, nt - t);
            int acc = 0;
            for (int u = 0; u < n; u++) acc += (gsub[g][t + u].w >> 1) / K;
            pitems[at++] = make_int4(g, gtile[g] + t, gtile[g] + t + n, acc);
        }
        at = gmit[g];
        for (int q = moff[g]; q < moff[g + 1]; q += m2p_item) mitems[at++] = make_int4(g, q, std::min(q + m2p_item, moff[g + 1]), 0);
    }
    if (tune_env("PYGBE_DEBUG")) {
        long pts = 0, selft = 0; int hist[9] = {0};
        for (auto &t : sub) { pts += t.w >> 1; selft += t.w & 1; hist[std::min(8, (t.w >> 1) * 8 / P2P_TILE)]++; }
        fprintf(stderr, "[pygbe] region: groups %d ranges %zu items %zu tiles %zu fill %.3f self tiles %ld; tile fill hist:",
                R.ng, prng.size(), pitems.size(), sub.size(), (double)pts / (sub.size() * (double)P2P_TILE), selft);
        for (int i = 0; i < 9; i++) fprintf(stderr, " %d", hist[i]);
        fprintf(stderr, "\n");
    }
    dbg_t("  tiles + items (host)");
    R.n_p2p_items = (int)pitems.size(); R.n_m2p_items = (int)mitems.size();
    TRY(upload(h, &R.p2p_sub, sub)); TRY(upload(h, &R.p2p_seg, segs)); TRY(upload(h, &R.p2p_items, pitems)); TRY(upload(h, &R.m2p_items, mitems));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return PYGBE_OK;
}
