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

static thread_local char g_err[1024] = "";

void pygbe_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *pygbe_last_error(void) { return g_err; }
extern "C" const char *pygbe_version(void) { return "pygbe-b200 0.2 sm_100a"; }

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
    TRY(matvec_impl(h, x_dev, y_dev, nullptr));
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
    TRY(matvec_impl(h, h->xh, h->yh, nullptr));
    CUDA_TRY(cudaMemcpyAsync(y_host, h->yh, bytes, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return PYGBE_OK;
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
    s->n_matvec = h->n_matvec; s->kernels_per_matvec = h->kernels_per_matvec; s->kernel_launches = h->launches;
    s->create_ms = h->create_ms; s->last_solve_ms = h->last_solve_ms; s->last_iters = h->last_iters;
    s->P = h->P; s->K = h->K; s->precision = h->precision; s->theta = h->theta;
    return PYGBE_OK;
}

extern "C" int pygbe_alu_peaks(int32_t device, double *out4)
{
    if (!out4) { pygbe_set_error("alu_peaks: null pointer"); return PYGBE_EINVAL; }
    return run_alu_peaks(device, out4);
}
