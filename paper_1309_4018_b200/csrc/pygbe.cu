// pygbe.cu -- the C ABI of include/pygbe.h.  Orchestration only: the host code parses inputs, sizes buffers,
// turns traversal output into work items and launches kernels (build_*.cuh, matvec.cuh, solve.cuh); every
// arithmetic step of the path runs on the device.
#include <mutex>
#include "common.cuh"
#include "host_util.cuh"
#include "tables.cuh"
#include "build_primary.cuh"
#include "matvec.cuh"
#include "solve.cuh"
#include "microbench.cuh"
#include "mma_probe.cuh"

static thread_local char g_err[1024] = "";

void pygbe_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *pygbe_last_error(void) { return g_err; }
extern "C" const char *pygbe_version(void) { return "pygbe-b200 0.3 sm_100a"; }

// Pinned host blocks (128 B: GMRES flags and scalars read back each poll) are kept for the life of the
// process and handed from handle to handle: cudaMallocHost costs 2-3 ms, a third of create at config 1.
static std::mutex g_pinned_mu;
static std::vector<void *> g_pinned_free;
static void *pinned_block_get()
{
    {
        std::lock_guard<std::mutex> lk(g_pinned_mu);
        if (!g_pinned_free.empty()) { void *p = g_pinned_free.back(); g_pinned_free.pop_back(); return p; }
    }
    void *p = nullptr;
    return cudaMallocHost(&p, 128) == cudaSuccess ? p : nullptr;
}
static void pinned_block_put(void *p)
{
    std::lock_guard<std::mutex> lk(g_pinned_mu);
    g_pinned_free.push_back(p);
}

static void free_handle(pygbe_handle *h)
{
    h->mem.release();
    if (h->pinned_scal) pinned_block_put(h->pinned_scal);
    for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    if (h->ev_join2) cudaEventDestroy(h->ev_join2);
    if (h->g_matvec.exec) cudaGraphExecDestroy(h->g_matvec.exec);
    if (h->g_iter.exec) cudaGraphExecDestroy(h->g_iter.exec);
    if (h->capst) cudaStreamDestroy(h->capst);
    if (h->side) cudaStreamDestroy(h->side);
    if (h->side2) cudaStreamDestroy(h->side2);
    delete h;
}

#include "create.inc"

extern "C" void pygbe_destroy(pygbe_handle *h)
{
    if (!h) return;
    cudaSetDevice(h->device);
    cudaStreamSynchronize(h->stream);
    if (h->side) cudaStreamSynchronize(h->side);
    if (h->side2) cudaStreamSynchronize(h->side2);
    free_handle(h);
}

extern "C" int64_t pygbe_num_unknowns(const pygbe_handle *h) { return h ? 2 * h->npan : -1; }

extern "C" int pygbe_matvec(pygbe_handle *h, const double *x_dev, double *y_dev)
{
    if (!h || !x_dev || !y_dev || x_dev == y_dev) { pygbe_set_error("matvec: null or aliased pointers"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    TRY(matvec_run(h, x_dev, y_dev));
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}

extern "C" int pygbe_matvec_host(pygbe_handle *h, const double *x_host, double *y_host)
{
    if (!h || !x_host || !y_host) { pygbe_set_error("matvec_host: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    TRY(ensure_host_staging(h));
    size_t bytes = 2 * h->npan * sizeof(double);
    CUDA_TRY(cudaMemcpyAsync(h->xh, x_host, bytes, cudaMemcpyHostToDevice, h->stream));
    TRY(matvec_run(h, h->xh, h->yh));
    CUDA_TRY(cudaMemcpyAsync(y_host, h->yh, bytes, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return PYGBE_OK;
}

extern "C" int pygbe_profile(pygbe_handle *h, int enable)
{
    if (!h) { pygbe_set_error("profile: null handle"); return PYGBE_EINVAL; }
    h->profile = enable != 0;
    h->ev_used = 0;
    h->launch_acc.clear();
    for (int i = 0; i < PYGBE_N_STAGES; i++) { h->stage_ms[i] = 0; h->stage_launches[i] = 0; }
    return PYGBE_OK;
}

extern "C" int pygbe_stage_times(pygbe_handle *h, double *ms, int64_t *launches)
{
    if (!h || !ms) { pygbe_set_error("stage_times: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    stage_collect(h);
    for (int i = 0; i < PYGBE_N_STAGES; i++) { ms[i] = h->stage_ms[i]; if (launches) launches[i] = h->stage_launches[i]; }
    return PYGBE_OK;
}

// What one launch of (stage, tree owner A) does: kernel name, work units, algorithmic bytes.
static void describe_launch(const pygbe_handle *h, int stage, const Region &A, pygbe_launch_info *o)
{
    const Region *B = A.twin >= 0 ? &h->regions[A.twin] : nullptr;
    const bool mixed = h->precision == PYGBE_PRECISION_MIXED;
    const int64_t np = A.np, npts = A.npts, Nc = h->Nc, nreg = B ? 2 : 1;
    const int64_t wrow = (int64_t)m2p_row_elems(h->P, A) * (mixed ? 4 : 8);
    o->twin_region = B ? B->id : -1;
    const char *name = "";
    switch (stage) {
    case PYGBE_STAGE_PREP:
        name = "k_prep"; o->units = npts;
        // per panel: x (2 x 8) through two indices (2 x 4), cV, cK, normal + area; writes phi, dphi, (cV dphi, cK phi), zeroed out
        // per point: weight (8 of the 32-byte record), writes the charge record (16 B fp32 / 32 B fp64)
        o->bytes = np * (16 + 8 + 16 + 32 + 8 + 8 + 16 + 8 * nreg) + npts * (8 + (mixed ? 16 : 32));
        break;
    case PYGBE_STAGE_P2M: {
        name = mixed ? "k_p2m<float>" : "k_p2m<double>"; o->units = A.p2m_panels;
        // per panel of a needed leaf: its two moment sets (pmom) and its two weights; per leaf: mom and the wc row written
        o->bytes = A.p2m_panels * (2 * Nc * (mixed ? 4 : 8) + 16) + (int64_t)A.n_p2m * (2 * Nc * 8 + wrow);
        break; }
    case PYGBE_STAGE_M2M:
        name = "k_m2m"; o->units = A.n_m2m;
        o->bytes = A.m2m_children * (2 * Nc * 8) + (int64_t)A.n_m2m * (2 * Nc * 8 + wrow + 32);
        break;
    case PYGBE_STAGE_M2P: name = m2p_kernel_name(h, A, B); o->units = A.m2p_evals; o->bytes = 0; break;
    case PYGBE_STAGE_P2P: name = p2p_kernel_name(h, A, B); o->units = A.p2p_pairs; o->bytes = 0; break;
    case PYGBE_STAGE_NEAR:
        name = "k_near"; o->units = np;
        o->bytes = A.corr_nnz * (4 + 16 * nreg) + np * (4 + 16 + 8 * nreg);
        break;
    case PYGBE_STAGE_COMBINE:
        name = "k_combine"; o->units = np;
        o->bytes = np * (8 + nreg * (8 + 8 + 4 + 8));
        break;
    default: break;
    }
    snprintf(o->kernel, sizeof(o->kernel), "%s", name);
}

extern "C" int pygbe_launch_times(pygbe_handle *h, pygbe_launch_info *out, int32_t max_out, int32_t *n_out)
{
    if (!h || !out || !n_out || max_out < 0) { pygbe_set_error("launch_times: null pointer"); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(h->device));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    stage_collect(h);
    int n = 0;
    for (const auto &a : h->launch_acc) {
        if (n >= max_out) break;
        if (a.region < 0 || a.region >= h->nreg) continue;
        pygbe_launch_info *o = out + n++;
        memset(o, 0, sizeof(*o));
        o->stage = a.stage; o->region = a.region; o->launches = a.launches; o->ms = a.ms;
        describe_launch(h, a.stage, h->regions[a.region], o);
    }
    *n_out = n;
    return PYGBE_OK;
}

extern "C" int pygbe_stats(const pygbe_handle *h, pygbe_stats_t *s)
{
    if (!h || !s) { pygbe_set_error("stats: null pointer"); return PYGBE_EINVAL; }
    memset(s, 0, sizeof(*s));
    s->n_panels = h->npan; s->n_unknowns = 2 * h->npan; s->n_regions = h->nreg; s->n_surfaces = h->nsurf;
    s->n_charges = h->nq;
    for (const Region &R : h->regions) {
        s->n_points += R.npts;
        if (R.twin_of < 0) { s->n_cells += R.ncells; s->n_leaves += R.nleaves; s->n_groups += R.ng; }
        s->tree_depth = std::max<int64_t>(s->tree_depth, R.depth);
        s->p2p_pairs += R.p2p_pairs; s->m2p_evals += R.m2p_evals;
        s->direct_equiv += (int64_t)R.np * R.npts;
        s->near_nnz += R.corr_nnz;
    }
    s->device_bytes = (int64_t)h->mem.bytes;
    s->workspace_high_water = (int64_t)h->mem.high_water;
    s->graph_launches = h->graph_launches;
    s->n_matvec = h->n_matvec; s->kernels_per_matvec = h->kernels_per_matvec; s->kernel_launches = h->launches;
    s->create_ms = h->create_ms; s->last_solve_ms = h->last_solve_ms; s->last_iters = h->last_iters;
    s->P = h->P; s->K = h->K; s->precision = h->precision; s->theta = h->theta;
    return PYGBE_OK;
}

extern "C" int pygbe_alu_peaks(int32_t device, double *out5)
{
    if (!out5) { pygbe_set_error("alu_peaks: null pointer"); return PYGBE_EINVAL; }
    return run_alu_peaks(device, out5);
}

extern "C" int pygbe_mma_probe(int32_t device, int32_t P, double *out12)
{
    if (!out12) { pygbe_set_error("mma_probe: null pointer"); return PYGBE_EINVAL; }
    if (P == 6) return run_mma_probe_p<6>(device, out12);
    if (P == 8) return run_mma_probe_p<8>(device, out12);
    pygbe_set_error("mma_probe: P = %d (instantiated for 6 and 8)", P);
    return PYGBE_EINVAL;
}

// Host-only: the coefficient tables of the M2P (tables.cuh), for CPU-side checks of the host logic.
extern "C" int pygbe_host_table(int32_t which, int32_t P, double kappa, int32_t cap_entries, int32_t cap_nnz, int32_t *n_entries,
                                int32_t *n_nnz, int32_t *off, int16_t *k, double *c, int16_t *deg)
{
    if (P < 0 || P > PYGBE_PMAX || !n_entries || !n_nnz || (which != 0 && which != 1)) { pygbe_set_error("host_table: bad arguments"); return PYGBE_EINVAL; }
    IndexTables *it = new IndexTables;
    fill_index_tables(it);
    WTable w;
    if (which == 0) build_w_table(P, kappa, *it, &w); else build_lap_table(P, *it, &w);
    delete it;
    *n_entries = (int)w.off.size() - 1; *n_nnz = (int)w.k.size();
    if (!off || !k || !c) return PYGBE_OK;                              // size query
    if (cap_entries < *n_entries || cap_nnz < *n_nnz) { pygbe_set_error("host_table: buffers too small"); return PYGBE_EINVAL; }
    for (size_t i = 0; i < w.off.size(); i++) off[i] = w.off[i];
    for (size_t i = 0; i < w.k.size(); i++) { k[i] = w.k[i]; c[i] = w.c[i]; }
    if (deg && which == 1) for (size_t i = 0; i < w.deg.size(); i++) deg[i] = w.deg[i];
    return PYGBE_OK;
}
