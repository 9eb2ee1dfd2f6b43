// pygbe.cu -- the C ABI of include/pygbe.h: orchestration of the kernels in tree.cuh, nearfield.cuh,
// farfield.cuh and gmres.cuh.  The host code here only parses inputs, sizes buffers, turns traversal
// output into work items and launches kernels; every arithmetic step of the path runs on the device.
#include "common.cuh"
#include "tables.cuh"
#include "tree.cuh"
#include "nearfield.cuh"
#include "farfield.cuh"
#include "m2p.cuh"
#include "mixed.cuh"
#include "gmres.cuh"

static thread_local char g_err[1024] = "";

void pygbe_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *pygbe_last_error(void) { return g_err; }
extern "C" const char *pygbe_version(void) { return "pygbe-b200 0.1 sm_100a"; }

static double now_ms()
{
    using namespace std::chrono;
    return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

template <class T> static int upload(pygbe_handle *h, T **dst, const std::vector<T> &src)
{
    TRY(h->mem.alloc(dst, src.size()));
    if (!src.empty())
        CUDA_TRY(cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, h->stream));
    return PYGBE_OK;
}
template <class T> static int download(pygbe_handle *h, std::vector<T> &dst, const T *src, size_t n)
{
    dst.resize(n);
    if (n) CUDA_TRY(cudaMemcpyAsync(dst.data(), src, n * sizeof(T), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return PYGBE_OK;
}

// ------------------------------------------------------------------------------------- mesh checking
// Closed, consistently oriented surface: every directed edge occurs once and its reverse once.
static int check_closed(const pygbe_surface &S, int s)
{
    std::vector<unsigned long long> e;
    e.reserve(3 * (size_t)S.n_triangles);
    for (int64_t t = 0; t < S.n_triangles; t++)
        for (int k = 0; k < 3; k++) {
            unsigned long long a = (unsigned)S.triangles[3 * t + k], b = (unsigned)S.triangles[3 * t + (k + 1) % 3];
            if (a == b) { pygbe_set_error("surface %d: triangle %ld repeats a vertex", s, (long)t); return PYGBE_EINVAL; }
            e.push_back((a << 32) | b);
        }
    std::sort(e.begin(), e.end());
    for (size_t i = 1; i < e.size(); i++)
        if (e[i] == e[i - 1]) {
            pygbe_set_error("surface %d: directed edge (%u,%u) occurs twice (inconsistent orientation or non-manifold)",
                            s, (unsigned)(e[i] >> 32), (unsigned)(e[i] & 0xffffffffu));
            return PYGBE_EINVAL;
        }
    for (size_t i = 0; i < e.size(); i++) {
        unsigned long long rev = (e[i] << 32) | (e[i] >> 32);
        if (!std::binary_search(e.begin(), e.end(), rev)) {
            pygbe_set_error("surface %d is open: edge (%u,%u) has no opposite", s, (unsigned)(e[i] >> 32),
                            (unsigned)(e[i] & 0xffffffffu));
            return PYGBE_EINVAL;
        }
    }
    return PYGBE_OK;
}

// ------------------------------------------------------------------------------------- region build
static int build_region(pygbe_handle *h, Region &R, const std::vector<double> &tri_host, const QuadTables &qt)
{
    const int K = h->K;
    // boundary panels of the region with sigma_S c_S, sigma_S (reading A4) and their slots in x / y
    std::vector<int> gid_u, phi_u, dphi_u, row_u;
    std::vector<double> cV_u, cK_u;
    for (int s = 0; s < h->nsurf; s++) {
        double sigma, c;
        int half;
        if (h->rin[s] == R.id) { sigma = 1.0; c = 1.0; half = 0; }
        else if (h->rout[s] == R.id) { sigma = -1.0; c = h->eps[h->rin[s]] / h->eps[h->rout[s]]; half = 1; }
        else continue;
        long o = h->surf_first[s], N = h->surf_count[s];
        for (long j = 0; j < N; j++) {
            gid_u.push_back((int)(o + j));
            phi_u.push_back((int)(2 * o + j));
            dphi_u.push_back((int)(2 * o + N + j));
            row_u.push_back((int)(2 * o + half * N + j));
            cV_u.push_back(sigma * c);
            cK_u.push_back(sigma);
        }
    }
    R.np = (int)gid_u.size();
    R.npts = R.np * K;
    if (R.np == 0) return PYGBE_OK;
    // root cube around the centroids; longest panel (for the near-field guard of the traversal)
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    double Lmax = 0.0;
    for (int p = 0; p < R.np; p++) {
        const double *t = tri_host.data() + 9 * (size_t)gid_u[p];
        double ux = t[3] - t[0], uy = t[4] - t[1], uz = t[5] - t[2];
        double vx = t[6] - t[0], vy = t[7] - t[1], vz = t[8] - t[2];
        double cx = uy * vz - uz * vy, cy = uz * vx - ux * vz, cz = ux * vy - uy * vx;
        Lmax = std::max(Lmax, std::sqrt(std::sqrt(cx * cx + cy * cy + cz * cz)));   // sqrt(2A), 2A = |cross|
        for (int a = 0; a < 3; a++) {
            double c = (t[a] + t[3 + a] + t[6 + a]) / 3.0;
            lo[a] = std::min(lo[a], c); hi[a] = std::max(hi[a], c);
        }
    }
    R.Lmax = Lmax;
    double edge = std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]}) * (1.0 + 1e-6) + 1e-9;
    for (int a = 0; a < 3; a++) R.root_c[a] = 0.5 * (lo[a] + hi[a]);
    R.root_edge = edge;

    int *d_gid_u, *d_phi_u, *d_dphi_u, *d_row_u, *d_iota, *d_perm;
    double *d_cV_u, *d_cK_u;
    unsigned long long *d_keys_u;
    TRY(upload(h, &d_gid_u, gid_u)); TRY(upload(h, &d_phi_u, phi_u)); TRY(upload(h, &d_dphi_u, dphi_u));
    TRY(upload(h, &d_row_u, row_u)); TRY(upload(h, &d_cV_u, cV_u)); TRY(upload(h, &d_cK_u, cK_u));
    TRY(h->mem.alloc(&d_iota, R.np)); TRY(h->mem.alloc(&d_perm, R.np));
    TRY(h->mem.alloc(&d_keys_u, R.np)); TRY(h->mem.alloc(&R.keys, R.np));
    LAUNCH(h, k_region_keys, cdiv(R.np, 256), 256, 0, h->gcen, d_gid_u, R.np, R.root_c[0] - 0.5 * edge,
           R.root_c[1] - 0.5 * edge, R.root_c[2] - 0.5 * edge, 2097152.0 / edge, d_keys_u, d_iota);
    {
        size_t tmp_bytes = 0;
        cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, d_keys_u, R.keys, d_iota, d_perm, R.np, 0, 63, h->stream);
        char *tmp;
        TRY(h->mem.alloc(&tmp, tmp_bytes));
        CUDA_TRY(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, d_keys_u, R.keys, d_iota, d_perm, R.np, 0, 63, h->stream));
        h->launches += 4;
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        h->mem.release_one(tmp);
    }
    TRY(h->mem.alloc(&R.gid, R.np)); TRY(h->mem.alloc(&R.phi_idx, R.np)); TRY(h->mem.alloc(&R.dphi_idx, R.np));
    TRY(h->mem.alloc(&R.row_idx, R.np)); TRY(h->mem.alloc(&R.cV, R.np)); TRY(h->mem.alloc(&R.cK, R.np));
    TRY(h->mem.alloc(&R.tpos, R.np)); TRY(h->mem.alloc(&R.pnrm, R.np));
    TRY(h->mem.alloc(&R.spos, R.npts)); TRY(h->mem.alloc(&R.schg, R.npts));
    TRY(h->mem.alloc(&R.pphi, R.np)); TRY(h->mem.alloc(&R.pdphi, R.np)); TRY(h->mem.alloc(&R.out, R.np));
    LAUNCH(h, k_region_gather, cdiv(R.np, 128), 128, 0, R.np, K, qt, d_perm, d_gid_u, d_phi_u, d_dphi_u, d_row_u,
           d_cV_u, d_cK_u, h->tri, h->gcen, h->gnrm, R.gid, R.phi_idx, R.dphi_idx, R.row_idx, R.cV, R.cK, R.tpos,
           R.pnrm, R.spos);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (void *q : {(void *)d_gid_u, (void *)d_phi_u, (void *)d_dphi_u, (void *)d_row_u, (void *)d_iota,
                    (void *)d_perm, (void *)d_cV_u, (void *)d_cK_u, (void *)d_keys_u})
        h->mem.release_one(q);

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
    TRY(download(h, crange_h, R.crange, (size_t)ncells));
    TRY(download(h, cchild_h, R.cchild, (size_t)ncells));
    std::vector<int> leaves;
    for (int c = 0; c < ncells; c++)
        if (cchild_h[c].y == 0) leaves.push_back(c);
    std::sort(leaves.begin(), leaves.end(), [&](int a, int b) { return crange_h[a].x < crange_h[b].x; });
    R.nleaves = (int)leaves.size();
    TRY(upload(h, &R.leaf_cell, leaves));

    // ---- target groups + traversal (count, offsets, fill)
    R.ng = cdiv(R.np, PYGBE_TG);
    TRY(h->mem.alloc(&R.ggeo, R.ng));
    LAUNCH(h, k_group_geometry, R.ng, PYGBE_TG, 0, R.tpos, R.np, R.ggeo);
    int *d_mcnt, *d_pcnt, *d_over;
    TRY(h->mem.alloc(&d_mcnt, R.ng)); TRY(h->mem.alloc(&d_pcnt, R.ng)); TRY(h->mem.alloc(&d_over, 1));
    CUDA_TRY(cudaMemsetAsync(d_over, 0, sizeof(int), h->stream));
    const double near_dist = h->thres > 0 ? h->thres * R.Lmax : 0.0;
    LAUNCH(h, k_traverse, cdiv(R.ng, TRAV_WARPS), TRAV_WARPS * 32, 0, R.ng, R.ggeo, R.cgeo, R.crange, R.cchild,
           h->theta, near_dist, 0, d_mcnt, d_pcnt, nullptr, nullptr, nullptr, nullptr, d_over);
    std::vector<int> mcnt, pcnt;
    TRY(download(h, mcnt, d_mcnt, (size_t)R.ng));
    TRY(download(h, pcnt, d_pcnt, (size_t)R.ng));
    std::vector<int> moff(R.ng + 1, 0), poff(R.ng + 1, 0);
    for (int g = 0; g < R.ng; g++) { moff[g + 1] = moff[g] + mcnt[g]; poff[g + 1] = poff[g] + pcnt[g]; }
    int *d_poff_raw;
    int2 *d_prng_raw;
    TRY(upload(h, &R.m2p_off, moff)); TRY(upload(h, &d_poff_raw, poff));
    TRY(h->mem.alloc(&R.m2p_cell, moff[R.ng])); TRY(h->mem.alloc(&d_prng_raw, poff[R.ng]));
    LAUNCH(h, k_traverse, cdiv(R.ng, TRAV_WARPS), TRAV_WARPS * 32, 0, R.ng, R.ggeo, R.cgeo, R.crange, R.cchild,
           h->theta, near_dist, 1, d_mcnt, d_pcnt, R.m2p_off, d_poff_raw, R.m2p_cell, d_prng_raw, d_over);
    std::vector<int2> prng_raw;
    TRY(download(h, prng_raw, d_prng_raw, (size_t)poff[R.ng]));
    int over = 0;
    CUDA_TRY(cudaMemcpy(&over, d_over, sizeof(int), cudaMemcpyDeviceToHost));
    if (over) { pygbe_set_error("traversal stack overflow"); return PYGBE_ECUDA; }
    for (void *q : {(void *)d_mcnt, (void *)d_pcnt, (void *)d_over, (void *)d_poff_raw, (void *)d_prng_raw})
        h->mem.release_one(q);

    // ---- P2P lists: sort each group's leaf ranges, merge adjacent ones; work items of bounded size
    std::vector<int2> prng;               // merged ranges, CSR by group
    std::vector<int> poff2(R.ng + 1, 0);
    long total_src_panels = 0;
    R.p2p_pairs = 0;
    for (int g = 0; g < R.ng; g++) {
        std::sort(prng_raw.begin() + poff[g], prng_raw.begin() + poff[g + 1],
                  [](const int2 &a, const int2 &b) { return a.x < b.x; });
        size_t start = prng.size();
        for (int r = poff[g]; r < poff[g + 1]; r++) {
            if (prng.size() > start && prng.back().y == prng_raw[r].x) prng.back().y = prng_raw[r].y;
            else prng.push_back(prng_raw[r]);
        }
        poff2[g + 1] = (int)prng.size();
        long ntg = std::min(PYGBE_TG, R.np - g * PYGBE_TG), src = 0;
        for (size_t r = start; r < prng.size(); r++) src += prng[r].y - prng[r].x;
        total_src_panels += src;
        R.p2p_pairs += ntg * src * K;
    }
    R.m2p_evals = 0;
    for (int g = 0; g < R.ng; g++) R.m2p_evals += (long)std::min(PYGBE_TG, R.np - g * PYGBE_TG) * mcnt[g];
    TRY(upload(h, &R.p2p_off, poff2)); TRY(upload(h, &R.p2p_rng, prng));
    const long want_items = 148L * 16;
    int p2p_item = (int)std::min(512L, std::max(32L, total_src_panels / want_items));
    int m2p_item = (int)std::min(64L, std::max(4L, (long)moff[R.ng] / want_items));
    m2p_item = (m2p_item + M2P_CB - 1) / M2P_CB * M2P_CB;
    std::vector<int2> sub;
    std::vector<int4> pitems, mitems;
    for (int g = 0; g < R.ng; g++) {
        int first = (int)sub.size(), acc = 0;
        for (int r = poff2[g]; r < poff2[g + 1]; r++) {
            int a = prng[r].x;
            while (a < prng[r].y) {
                int take = std::min(prng[r].y - a, p2p_item - acc);
                sub.push_back(make_int2(a, a + take));
                a += take; acc += take;
                if (acc == p2p_item) { pitems.push_back(make_int4(g, first, (int)sub.size(), 0)); first = (int)sub.size(); acc = 0; }
            }
        }
        if (acc > 0) pitems.push_back(make_int4(g, first, (int)sub.size(), 0));
        for (int s = moff[g]; s < moff[g + 1]; s += m2p_item)
            mitems.push_back(make_int4(g, s, std::min(s + m2p_item, moff[g + 1]), 0));
    }
    R.n_p2p_items = (int)pitems.size(); R.n_m2p_items = (int)mitems.size();
    TRY(upload(h, &R.p2p_sub, sub)); TRY(upload(h, &R.p2p_items, pitems)); TRY(upload(h, &R.m2p_items, mitems));

    // ---- singular / near-singular corrections (a8)
    {
        int *d_cnt;
        TRY(h->mem.alloc(&d_cnt, R.np));
        const double thres2 = h->thres > 0 ? h->thres * h->thres : 0.0;
        LAUNCH(h, k_near_find, R.ng, PYGBE_TG, 0, R.np, R.tpos, R.pnrm, R.p2p_off, R.p2p_rng, thres2, 0, d_cnt, nullptr, nullptr);
        std::vector<int> cnt;
        TRY(download(h, cnt, d_cnt, (size_t)R.np));
        std::vector<int> off(R.np + 1, 0);
        long nself = 0;
        for (int t = 0; t < R.np; t++) { off[t + 1] = off[t] + cnt[t]; nself += cnt[t] > 0; }
        R.corr_nnz = off[R.np];
        if (nself != R.np) { pygbe_set_error("internal: a target's own panel is missing from its P2P list"); return PYGBE_ECUDA; }
        TRY(upload(h, &R.corr_off, off));
        TRY(h->mem.alloc(&R.corr_col, R.corr_nnz)); TRY(h->mem.alloc(&R.corr_val, R.corr_nnz));
        LAUNCH(h, k_near_find, R.ng, PYGBE_TG, 0, R.np, R.tpos, R.pnrm, R.p2p_off, R.p2p_rng, thres2, 1, d_cnt, R.corr_off, R.corr_col);
        LAUNCH(h, k_near_values, cdiv(R.np, 64), 64, 0, R.np, qt, R.yukawa, R.kappa, R.corr_off, R.corr_col, R.gid, h->tri,
               R.tpos, R.pnrm, R.spos, R.cV, R.cK, R.corr_val);
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        h->mem.release_one(d_cnt);
    }
    if (R.n_m2p_items > 0) TRY(h->mem.alloc(&R.mom, (size_t)R.ncells * h->Nc));
    if (h->precision == PYGBE_PRECISION_MIXED) TRY(mixed_build_region(h, R));
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}

// ------------------------------------------------------------------------------------------- create
extern "C" int pygbe_create(const pygbe_surface *surfaces, int32_t n_surfaces, const pygbe_charges *charges,
                            const double *eps, const double *kappa, int32_t n_regions, int32_t K, int32_t P,
                            double theta, const pygbe_options *opt, pygbe_handle **out)
{
    g_err[0] = 0;
    if (!out) { pygbe_set_error("out is NULL"); return PYGBE_EINVAL; }
    *out = nullptr;
    if (!surfaces || n_surfaces <= 0 || !eps || !kappa || n_regions <= 0) {
        pygbe_set_error("surfaces / eps / kappa missing or empty");
        return PYGBE_EINVAL;
    }
    if (P < 1 || P > PYGBE_PMAX) { pygbe_set_error("P = %d outside 1..%d", P, PYGBE_PMAX); return PYGBE_EINVAL; }
    if (!(theta >= 0.0) || theta >= 1.0) { pygbe_set_error("theta = %g outside [0,1)", theta); return PYGBE_EINVAL; }
    pygbe_options o;
    memset(&o, 0, sizeof(o));
    if (opt) o = *opt;
    QuadTables qt;
    TRY(make_quad_tables(K, o.K_fine ? o.K_fine : 19, o.N_k ? o.N_k : 5, &qt));
    if (o.precision != PYGBE_PRECISION_FP64 && o.precision != PYGBE_PRECISION_MIXED) {
        pygbe_set_error("unknown precision %d", o.precision);
        return PYGBE_EINVAL;
    }
    for (int r = 0; r < n_regions; r++)
        if (!(eps[r] > 0.0) || !(kappa[r] >= 0.0)) { pygbe_set_error("region %d: eps must be > 0 and kappa >= 0", r); return PYGBE_EINVAL; }
    long npan = 0;
    for (int s = 0; s < n_surfaces; s++) {
        const pygbe_surface &S = surfaces[s];
        if (!S.vertices || !S.triangles || S.n_vertices < 4 || S.n_triangles < 4) {
            pygbe_set_error("surface %d: missing or too small", s);
            return PYGBE_EINVAL;
        }
        if (S.region_in < 0 || S.region_in >= n_regions || S.region_out < 0 || S.region_out >= n_regions ||
            S.region_in == S.region_out) {
            pygbe_set_error("surface %d: bad region ids (%d, %d)", s, S.region_in, S.region_out);
            return PYGBE_EINVAL;
        }
        for (int64_t t = 0; t < 3 * S.n_triangles; t++)
            if (S.triangles[t] < 0 || S.triangles[t] >= S.n_vertices) {
                pygbe_set_error("surface %d: vertex index out of range in triangle %ld", s, (long)(t / 3));
                return PYGBE_EINVAL;
            }
        if (o.check_mesh) TRY(check_closed(S, s));
        npan += S.n_triangles;
    }
    if (2 * npan * (long)std::max(K, 1) > 2000000000L) { pygbe_set_error("problem too large for 32-bit indices"); return PYGBE_EINVAL; }
    long nq = charges ? charges->n : 0;
    if (nq < 0 || (nq > 0 && (!charges->xyz || !charges->q))) { pygbe_set_error("charges: null arrays"); return PYGBE_EINVAL; }
    for (long k = 0; k < nq; k++) {
        int r = charges->region ? charges->region[k] : 0;
        if (r < 0 || r >= n_regions) { pygbe_set_error("charge %ld: region %d out of range", k, r); return PYGBE_EINVAL; }
    }

    double t0 = now_ms();
    cudaError_t ce = cudaSetDevice(o.device);
    if (ce != cudaSuccess) { pygbe_set_error("cudaSetDevice(%d): %s", o.device, cudaGetErrorString(ce)); return PYGBE_ECUDA; }
    pygbe_handle *h = new (std::nothrow) pygbe_handle();
    if (!h) return PYGBE_ENOMEM;
    h->device = o.device; h->stream = (cudaStream_t)o.stream;
    h->K = K; h->P = P; h->Nc = nc_of(P); h->Kfine = qt.Kfine; h->Nk = qt.Nk;
    h->theta = theta; h->thres = o.thres == 0.0 ? 2.0 : o.thres;
    h->ncrit = o.ncrit > 0 ? o.ncrit : 96;
    h->precision = o.precision;
    h->npan = npan; h->nsurf = n_surfaces; h->nreg = n_regions; h->nq = nq;
    h->eps.assign(eps, eps + n_regions); h->kappa.assign(kappa, kappa + n_regions);
    auto fail = [&](int rc) { h->mem.release(); if (h->pinned_flags) cudaFreeHost(h->pinned_flags);
                              if (h->pinned_scal) cudaFreeHost(h->pinned_scal); delete h; return rc; };
#define TRYF(expr) do { int rc__ = (expr); if (rc__ != PYGBE_OK) return fail(rc__); } while (0)
#define CUDAF(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { pygbe_set_error("%s: %s", #expr, cudaGetErrorString(e__)); return fail(PYGBE_ECUDA); } } while (0)
    TRYF(upload_index_tables());
    CUDAF(cudaMallocHost(&h->pinned_flags, 4 * sizeof(int)));
    CUDAF(cudaMallocHost(&h->pinned_scal, 8 * sizeof(double)));

    std::vector<double> tri_host((size_t)npan * 9);
    long at = 0;
    for (int s = 0; s < n_surfaces; s++) {
        const pygbe_surface &S = surfaces[s];
        h->surf_first.push_back(at); h->surf_count.push_back(S.n_triangles);
        h->rin.push_back(S.region_in); h->rout.push_back(S.region_out);
        for (int64_t t = 0; t < S.n_triangles; t++, at++)
            for (int k = 0; k < 3; k++) {
                const double *v = S.vertices + 3 * (size_t)S.triangles[3 * t + k];
                tri_host[9 * at + 3 * k] = v[0]; tri_host[9 * at + 3 * k + 1] = v[1]; tri_host[9 * at + 3 * k + 2] = v[2];
            }
    }
    TRYF(upload(h, &h->tri, tri_host));
    TRYF(h->mem.alloc(&h->gcen, npan)); TRYF(h->mem.alloc(&h->gnrm, npan)); TRYF(h->mem.alloc(&h->scratch, 16));
    int *d_flag;
    TRYF(h->mem.alloc(&d_flag, 1));
    CUDAF(cudaMemsetAsync(d_flag, 0, sizeof(int), h->stream));
    LAUNCH(h, k_panel_geometry, cdiv(npan, 256), 256, 0, h->tri, npan, h->gcen, h->gnrm, d_flag);
    int flag = 0;
    CUDAF(cudaMemcpyAsync(&flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CUDAF(cudaStreamSynchronize(h->stream));
    h->mem.release_one(d_flag);
    if (flag) { pygbe_set_error("degenerate (zero-area or non-finite) triangle"); return fail(PYGBE_EINVAL); }

    h->regions.resize(n_regions);
    for (int r = 0; r < n_regions; r++) {
        Region &R = h->regions[r];
        R.id = r; R.eps = eps[r]; R.kappa = kappa[r]; R.yukawa = kappa[r] > 0.0;
        TRYF(build_region(h, R, tri_host, qt));
        // charges of this region
        std::vector<double4> qp;
        std::vector<int> qi;
        for (long k = 0; k < nq; k++)
            if ((charges->region ? charges->region[k] : 0) == r) {
                qp.push_back(make_double4(charges->xyz[3 * k], charges->xyz[3 * k + 1], charges->xyz[3 * k + 2], charges->q[k]));
                qi.push_back((int)k);
            }
        R.nq = (int)qp.size();
        if (R.nq > 0 && R.np == 0) { pygbe_set_error("charges in region %d, which has no boundary", r); return fail(PYGBE_EINVAL); }
        TRYF(upload(h, &R.qpos, qp)); TRYF(upload(h, &R.qid, qi));
    }
    if (nq > 0) {
        h->qxyz.assign(charges->xyz, charges->xyz + 3 * nq);
        h->qq.assign(charges->q, charges->q + nq);
        TRYF(h->mem.alloc(&h->phi_reac, nq + 1));
    }
    CUDAF(cudaStreamSynchronize(h->stream));
    CUDAF(cudaGetLastError());
    h->create_ms = now_ms() - t0;
    *out = h;
    return PYGBE_OK;
}

extern "C" void pygbe_destroy(pygbe_handle *h)
{
    if (!h) return;
    cudaSetDevice(h->device);
    cudaStreamSynchronize(h->stream);
    h->mem.release();
    if (h->pinned_flags) cudaFreeHost(h->pinned_flags);
    if (h->pinned_scal) cudaFreeHost(h->pinned_scal);
    for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
    delete h;
}

extern "C" int64_t pygbe_num_unknowns(const pygbe_handle *h) { return h ? 2 * h->npan : -1; }

// ------------------------------------------------------------------------------------------- matvec
#define M2P_DECL(PP) int pygbe_m2p_f64_launch_##PP(const M2PArgs &);
M2P_DECL(1) M2P_DECL(2) M2P_DECL(3) M2P_DECL(4) M2P_DECL(5) M2P_DECL(6)
M2P_DECL(7) M2P_DECL(8) M2P_DECL(9) M2P_DECL(10) M2P_DECL(11) M2P_DECL(12)
#undef M2P_DECL

static int launch_m2p(pygbe_handle *h, Region &R, const int *skip)
{
    M2PArgs a;
    memset(&a, 0, sizeof(a));
    a.skip = skip; a.items = R.m2p_items; a.m2p_cell = R.m2p_cell; a.n_items = R.n_m2p_items; a.np = R.np;
    a.tpos = R.tpos; a.cgeo = R.cgeo; a.mom = R.mom; a.kappa = R.kappa; a.out = R.out; a.yukawa = R.yukawa;
    a.stream = h->stream;
    typedef int (*fn_t)(const M2PArgs &);
    static const fn_t table[PYGBE_PMAX + 1] = {nullptr, pygbe_m2p_f64_launch_1, pygbe_m2p_f64_launch_2,
        pygbe_m2p_f64_launch_3, pygbe_m2p_f64_launch_4, pygbe_m2p_f64_launch_5, pygbe_m2p_f64_launch_6,
        pygbe_m2p_f64_launch_7, pygbe_m2p_f64_launch_8, pygbe_m2p_f64_launch_9, pygbe_m2p_f64_launch_10,
        pygbe_m2p_f64_launch_11, pygbe_m2p_f64_launch_12};
    if (h->P < 1 || h->P > PYGBE_PMAX) { pygbe_set_error("P = %d not instantiated", h->P); return PYGBE_EINVAL; }
    table[h->P](a);
    h->launches++;
    return PYGBE_OK;
}

// Stage timers: an event is recorded where a stage starts; the time to the next event belongs to it.
static void stage_mark(pygbe_handle *h, int stage)
{
    if (!h->profile) return;
    if (h->ev_used == h->ev_pool.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return;
        h->ev_pool.push_back(e);
        h->ev_stage.push_back(-1);
    }
    h->ev_stage[h->ev_used] = stage;
    cudaEventRecord(h->ev_pool[h->ev_used], h->stream);
    h->ev_used++;
}

extern "C" int pygbe_profile(pygbe_handle *h, int enable)
{
    if (!h) { pygbe_set_error("profile: null handle"); return PYGBE_EINVAL; }
    h->profile = enable != 0;
    h->ev_used = 0;
    for (int i = 0; i < PYGBE_N_STAGES; i++) { h->stage_ms[i] = 0; h->stage_launches[i] = 0; }
    return PYGBE_OK;
}

extern "C" int pygbe_stage_times(pygbe_handle *h, double *ms, int64_t *launches)
{
    if (!h || !ms) { pygbe_set_error("stage_times: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (size_t i = 0; i + 1 < h->ev_used; i++) {
        int st = h->ev_stage[i];
        if (st < 0 || st >= PYGBE_N_STAGES) continue;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, h->ev_pool[i], h->ev_pool[i + 1]) == cudaSuccess) h->stage_ms[st] += t;
    }
    h->ev_used = 0;
    for (int i = 0; i < PYGBE_N_STAGES; i++) { ms[i] = h->stage_ms[i]; if (launches) launches[i] = h->stage_launches[i]; }
    return PYGBE_OK;
}
#define STAGE(h, st) do { stage_mark(h, st); if ((h)->profile) (h)->stage_launches[st] -= (h)->launches; } while (0)
#define STAGE_END(h, st) do { if ((h)->profile) (h)->stage_launches[st] += (h)->launches; } while (0)

// weights -> (P2M -> M2M -> M2P) + P2P -> corrections; leaves sum_S sigma[c V dphi - K phi] in R.out
static int region_sum(pygbe_handle *h, Region &R, const double *x, const int *skip)
{
    if (R.np == 0) return PYGBE_OK;
    const bool mixed = h->precision == PYGBE_PRECISION_MIXED;
    STAGE(h, PYGBE_STAGE_PREP);
    LAUNCH(h, k_prep, cdiv(R.np, 128), 128, 0, skip, R.np, h->K, x, R.phi_idx, R.dphi_idx, R.cV, R.cK, R.pnrm, R.spos,
           R.schg, R.schgf, R.pphi, R.pdphi, R.out);
    STAGE_END(h, PYGBE_STAGE_PREP);
    if (mixed) {
        TRY(mixed_region_sum(h, R, skip));
    } else {
        if (R.n_m2p_items > 0) {
            STAGE(h, PYGBE_STAGE_P2M);
            LAUNCH(h, k_p2m, R.nleaves, P2M_THREADS, 0, skip, h->P, h->Nc, h->K, R.leaf_cell, R.cgeo, R.crange, R.spos,
                   R.schg, R.mom);
            STAGE_END(h, PYGBE_STAGE_P2M);
            STAGE(h, PYGBE_STAGE_M2M);
            for (int l = R.depth - 2; l >= 0; l--) {
                int b = R.level_begin[l], e = R.level_begin[l + 1];
                LAUNCH(h, k_m2m, e - b, M2M_THREADS, 0, skip, h->P, h->Nc, b, e, R.cgeo, R.cchild, R.mom);
            }
            STAGE_END(h, PYGBE_STAGE_M2M);
            STAGE(h, PYGBE_STAGE_M2P);
            TRY(launch_m2p(h, R, skip));
            STAGE_END(h, PYGBE_STAGE_M2P);
        }
        if (R.n_p2p_items > 0) {
            STAGE(h, PYGBE_STAGE_P2P);
            if (R.yukawa)
                LAUNCH(h, k_p2p_f64<true>, R.n_p2p_items, PYGBE_TG, 0, skip, R.p2p_items, R.p2p_sub, h->K, R.np, R.tpos,
                       R.spos, R.schg, R.kappa, R.out);
            else
                LAUNCH(h, k_p2p_f64<false>, R.n_p2p_items, PYGBE_TG, 0, skip, R.p2p_items, R.p2p_sub, h->K, R.np, R.tpos,
                       R.spos, R.schg, R.kappa, R.out);
            STAGE_END(h, PYGBE_STAGE_P2P);
        }
    }
    STAGE(h, PYGBE_STAGE_NEAR);
    LAUNCH(h, k_near_apply, cdiv(R.np, 128), 128, 0, skip, R.np, R.corr_off, R.corr_col, R.corr_val, R.pphi, R.pdphi, R.out);
    STAGE_END(h, PYGBE_STAGE_NEAR);
    return PYGBE_OK;
}

static int matvec_impl(pygbe_handle *h, const double *x, double *y, const int *skip)
{
    long before = h->launches;
    for (Region &R : h->regions) {
        if (R.np == 0) continue;
        TRY(region_sum(h, R, x, skip));
        STAGE(h, PYGBE_STAGE_COMBINE);
        LAUNCH(h, k_combine, cdiv(R.np, 256), 256, 0, skip, R.np, R.row_idx, R.pphi, R.out, y);
        STAGE_END(h, PYGBE_STAGE_COMBINE);
    }
    stage_mark(h, -1);
    h->kernels_per_matvec = h->launches - before;
    h->n_matvec++;
    return PYGBE_OK;
}

extern "C" int pygbe_matvec(pygbe_handle *h, const double *x_dev, double *y_dev)
{
    if (!h || !x_dev || !y_dev || x_dev == y_dev) { pygbe_set_error("matvec: null or aliased pointers"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    TRY(matvec_impl(h, x_dev, y_dev, nullptr));
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}

static int ensure_host_staging(pygbe_handle *h)
{
    if (!h->xh) { TRY(h->mem.alloc(&h->xh, 2 * h->npan)); TRY(h->mem.alloc(&h->yh, 2 * h->npan)); }
    return PYGBE_OK;
}

extern "C" int pygbe_matvec_host(pygbe_handle *h, const double *x_host, double *y_host)
{
    if (!h || !x_host || !y_host) { pygbe_set_error("matvec_host: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    TRY(ensure_host_staging(h));
    size_t bytes = 2 * h->npan * sizeof(double);
    CUDA_TRY(cudaMemcpyAsync(h->xh, x_host, bytes, cudaMemcpyHostToDevice, h->stream));
    TRY(matvec_impl(h, h->xh, h->yh, nullptr));
    CUDA_TRY(cudaMemcpyAsync(y_host, h->yh, bytes, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
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
    TRY(h->mem.alloc(&G.V, (size_t)(m + 1) * n));
    TRY(h->mem.alloc(&G.H, (size_t)(m + 1) * m));
    TRY(h->mem.alloc(&G.h1, m + 2)); TRY(h->mem.alloc(&G.h2, m + 2)); TRY(h->mem.alloc(&G.cs, m + 1));
    TRY(h->mem.alloc(&G.sn, m + 1)); TRY(h->mem.alloc(&G.g, m + 2)); TRY(h->mem.alloc(&G.yk, m + 1));
    if (!G.w) {
        TRY(h->mem.alloc(&G.w, n)); TRY(h->mem.alloc(&G.b, n)); TRY(h->mem.alloc(&G.scal, 8)); TRY(h->mem.alloc(&G.flags, 4));
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
    int total = 0, done = 0;
    bool first = true;
    while (total < max_iter && !done) {
        const int mc = std::min(m, max_iter - total);
        if (!first) TRY(matvec_impl(h, x_dev, G.w, G.flags));
        LAUNCH(h, k_gm_residual, gridn, GM_THREADS, 0, G.flags, n, G.b, G.w, first ? 0 : 1, G.V, G.scal);
        LAUNCH(h, k_gm_begin, 1, 1, 0, G.flags, G.scal, G.g, G.m, first ? 1 : 0, tol);
        LAUNCH(h, k_gm_scale, gridn, GM_THREADS, 0, G.flags, n, G.V, G.scal + 1, 0, G.V);
        first = false;
        int j = 0;
        for (; j < mc; j++) {
            double *vj = G.V + (size_t)j * n, *vn = G.V + (size_t)(j + 1) * n;
            TRY(matvec_impl(h, vj, G.w, G.flags));
            LAUNCH(h, k_gm_zero, cdiv(j + 2, 128), 128, 0, G.flags, G.h1, j + 1, G.h2, j + 1, G.scal + 3, 1);
            LAUNCH(h, k_gm_dots, gridd, GM_THREADS, 0, G.flags, G.V, n, j + 1, G.w, G.h1);
            LAUNCH(h, k_gm_axpys, gridn, GM_THREADS, 0, G.flags, G.V, n, j + 1, G.h1, G.w);
            LAUNCH(h, k_gm_dots, gridd, GM_THREADS, 0, G.flags, G.V, n, j + 1, G.w, G.h2);
            LAUNCH(h, k_gm_axpys, gridn, GM_THREADS, 0, G.flags, G.V, n, j + 1, G.h2, G.w);
            LAUNCH(h, k_gm_dots, gridd, GM_THREADS, 0, G.flags, G.w, n, 1, G.w, G.scal + 3);
            LAUNCH(h, k_gm_scale, gridn, GM_THREADS, 0, G.flags, n, G.w, G.scal + 3, 1, vn);
            LAUNCH(h, k_gm_givens, 1, 1, 0, G.flags, j, G.m, G.h1, G.h2, G.scal + 3, G.H, G.cs, G.sn, G.g, G.scal, tol);
            if ((j + 1) % poll == 0 || j + 1 == mc) {
                CUDA_TRY(cudaMemcpyAsync(h->pinned_flags, G.flags, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
                CUDA_TRY(cudaStreamSynchronize(st));
                if (h->pinned_flags[0]) { done = 1; break; }
            }
        }
        LAUNCH(h, k_gm_solve_small, 1, 1, 0, G.flags, G.m, G.H, G.g, G.yk);
        LAUNCH(h, k_gm_update, gridn, GM_THREADS, 0, G.flags, n, G.V, G.yk, x_dev);
        CUDA_TRY(cudaMemcpyAsync(h->pinned_flags, G.flags, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaMemcpyAsync(h->pinned_scal, G.scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        done = h->pinned_flags[0];
        total = h->pinned_flags[2];
        if (!done) {
            // new cycle: rotations and g restart; flags[1] is rewritten by the next givens
            CUDA_TRY(cudaMemsetAsync(G.scal + 3, 0, sizeof(double), st));
        }
    }
    CUDA_TRY(cudaGetLastError());
    h->last_iters = total;
    h->last_solve_ms = now_ms() - t0;
    if (iters) *iters = total;
    if (rel_resid) *rel_resid = h->pinned_scal[2];
    if (!done) { pygbe_set_error("GMRES: %d iterations, relative residual %.3e > tol %.3e", total, h->pinned_scal[2], tol); return PYGBE_ENOCONV; }
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
        LAUNCH(h, k_prep, cdiv(R.np, 128), 128, 0, nullptr, R.np, h->K, x_dev, R.phi_idx, R.dphi_idx, R.cV, R.cK, R.pnrm,
               R.spos, R.schg, (float4 *)nullptr, R.pphi, R.pdphi, R.out);
        dim3 grid(cdiv(R.npts, EN_CHUNK), R.nq);
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
        double *d_q;
        TRY(h->mem.alloc(&d_q, h->nq));
        CUDA_TRY(cudaMemcpyAsync(d_q, h->qq.data(), h->nq * sizeof(double), cudaMemcpyHostToDevice, h->stream));
        LAUNCH(h, k_dot_q, 1, 256, 0, (int)h->nq, d_q, h->phi_reac, h->scratch);
        CUDA_TRY(cudaMemcpyAsync(h->pinned_scal, h->scratch, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        h->mem.release_one(d_q);
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

extern "C" int pygbe_stats(const pygbe_handle *h, pygbe_stats_t *s)
{
    if (!h || !s) { pygbe_set_error("stats: null pointer"); return PYGBE_EINVAL; }
    memset(s, 0, sizeof(*s));
    s->n_panels = h->npan; s->n_unknowns = 2 * h->npan; s->n_regions = h->nreg; s->n_surfaces = h->nsurf;
    s->n_charges = h->nq;
    for (const Region &R : h->regions) {
        s->n_points += R.npts; s->n_cells += R.ncells; s->n_leaves += R.nleaves; s->n_groups += R.ng;
        s->tree_depth = std::max<int64_t>(s->tree_depth, R.depth);
        s->p2p_pairs += R.p2p_pairs; s->m2p_evals += R.m2p_evals;
        s->direct_equiv += (int64_t)R.np * R.npts;
        s->near_nnz += R.corr_nnz;
    }
    s->device_bytes = (int64_t)h->mem.bytes;
    s->n_matvec = h->n_matvec; s->kernels_per_matvec = h->kernels_per_matvec; s->kernel_launches = h->launches;
    s->create_ms = h->create_ms; s->last_solve_ms = h->last_solve_ms; s->last_iters = h->last_iters;
    s->P = h->P; s->K = h->K; s->precision = h->precision; s->theta = h->theta;
    return PYGBE_OK;
}

// ------------------------------------------------------------------------------------ ALU peak probes
#include "microbench.cuh"
extern "C" int pygbe_alu_peaks(int32_t device, double *out3)
{
    if (!out3) { pygbe_set_error("alu_peaks: null pointer"); return PYGBE_EINVAL; }
    return run_alu_peaks(device, out3);
}
