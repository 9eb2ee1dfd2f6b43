// host_util.cuh -- small host helpers shared by the orchestration files.
#pragma once
#include "common.cuh"

static inline double now_ms()
{
    using namespace std::chrono;
    return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

// PYGBE_DEBUG=1: host milliseconds since the previous checkpoint (create-time diagnostics on stderr)
static inline void dbg_t(const char *what)
{
    static const bool on = tune_env("PYGBE_DEBUG") != nullptr;
    static double last = 0.0;
    if (!on) return;
    const double t = now_ms();
    if (what) fprintf(stderr, "[pygbe] %-28s %8.3f ms\n", what, t - last);
    last = t;
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
