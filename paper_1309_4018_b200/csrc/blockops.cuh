// blockops.cuh -- the library's own block-level reductions / scan and its radix sort (no CUB, no Thrust).
//   block_reduce<THREADS>(v, op)   result valid in thread 0; ends with a CTA barrier, so calls may follow one another
//   block_exclusive_sum<THREADS>   exclusive prefix sum of one int per thread + the CTA total (every thread)
//   radix_sort_pairs               stable LSD radix sort of (u64 key, int value) pairs: the Morton sort of a2
#pragma once
#include "common.cuh"

struct OpSum { __device__ __forceinline__ double operator()(double a, double b) const { return a + b; } };
struct OpMin { __device__ __forceinline__ double operator()(double a, double b) const { return fmin(a, b); } };
struct OpMax { __device__ __forceinline__ double operator()(double a, double b) const { return fmax(a, b); } };

template <int THREADS, class Op>
__device__ __forceinline__ double block_reduce(double v, Op op)
{
    static_assert(THREADS % 32 == 0 && THREADS <= 1024, "whole warps");
    __shared__ double s_w[THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = op(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) s_w[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {                                          // at most 32 partials: a serial loop in a fixed order
        double x = s_w[0];
        for (int w = 1; w < THREADS / 32; w++) x = op(x, s_w[w]);
        v = x;
    }
    __syncthreads();                                                 // s_w may be rewritten by a following call
    return v;
}
template <int THREADS> __device__ __forceinline__ double block_sum(double v) { return block_reduce<THREADS>(v, OpSum()); }

template <int THREADS>
__device__ __forceinline__ void block_exclusive_sum(int v, int &excl, int &total)
{
    static_assert(THREADS % 32 == 0 && THREADS <= 1024, "whole warps");
    __shared__ int s_w[THREADS / 32 + 1];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += y;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        constexpr int NW = THREADS / 32;
        const int w = lane < NW ? s_w[lane] : 0;
        int winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += y;
        }
        if (lane < NW) s_w[lane] = winc - w;                         // exclusive prefix of the warp totals
        if (lane == 31) s_w[NW] = winc;                              // CTA total
    }
    __syncthreads();
    excl = s_w[warp] + inc - v;
    total = s_w[THREADS / 32];
    __syncthreads();                                                 // s_w may be rewritten by a following call
}

// ---------------------------------------------------------------------------------------------- radix sort
// Stable least-significant-digit radix sort, 8-bit digits.  Per pass: (1) every CTA counts the digits of its tile
// (RS_ROUNDS x 256 keys) into hist[digit][cta]; (2) one CTA turns hist into exclusive offsets in (digit, cta) order;
// (3) every CTA scatters its tile: a key's position = offset of its (digit, cta) + keys with the same digit earlier in
// the tile -- counted round by round (running per-digit base), inside a round warp by warp (per-warp digit counts in
// shared memory), inside a warp with match_any + popc of the lower lanes.  Equal keys keep their order.
#define RS_THREADS 256
#define RS_ROUNDS 4
#define RS_TILE (RS_THREADS * RS_ROUNDS)

__global__ void __launch_bounds__(RS_THREADS)
k_rs_hist(const unsigned long long *__restrict__ keys, int n, int shift, int ncta, int *__restrict__ hist)
{
    __shared__ int s_cnt[256];
    s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const long base = (long)blockIdx.x * RS_TILE;
#pragma unroll
    for (int r = 0; r < RS_ROUNDS; r++) {
        const long i = base + r * RS_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&s_cnt[(int)((keys[i] >> shift) & 255ull)], 1);
    }
    __syncthreads();
    hist[(long)threadIdx.x * ncta + blockIdx.x] = s_cnt[threadIdx.x];
}

// exclusive scan of hist[256 * ncta] in place, one CTA
__global__ void __launch_bounds__(1024)
k_rs_scan(int *hist, long m)
{
    __shared__ int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (long i0 = 0; i0 < m; i0 += 1024) {
        const long i = i0 + threadIdx.x;
        const int v = i < m ? hist[i] : 0;
        int excl, total;
        block_exclusive_sum<1024>(v, excl, total);
        const int carry = s_carry;
        if (i < m) hist[i] = carry + excl;
        __syncthreads();
        if (threadIdx.x == 0) s_carry = carry + total;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(RS_THREADS)
k_rs_scatter(const unsigned long long *__restrict__ keys, const int *__restrict__ vals, int n, int shift, int ncta,
             const int *__restrict__ offs, unsigned long long *__restrict__ keys_out, int *__restrict__ vals_out)
{
    __shared__ int s_base[256];                                      // position of the next key with this digit
    __shared__ int s_wcnt[RS_THREADS / 32][256];                     // per-warp digit counts of the round
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    s_base[threadIdx.x] = offs[(long)threadIdx.x * ncta + blockIdx.x];
    const long base = (long)blockIdx.x * RS_TILE;
    for (int r = 0; r < RS_ROUNDS; r++) {
        for (int w = 0; w < RS_THREADS / 32; w++) s_wcnt[w][threadIdx.x] = 0;
        __syncthreads();
        const long i = base + r * RS_THREADS + threadIdx.x;
        const bool ok = i < n;
        const unsigned long long key = ok ? keys[i] : ~0ull;
        const int d = (int)((key >> shift) & 255ull);
        // lanes of this warp with the same digit (inactive lanes take digit 256 + lane: never equal)
        const unsigned peers = __match_any_sync(0xffffffffu, ok ? d : 256 + lane);
        const int rank = __popc(peers & ((1u << lane) - 1u));
        if (ok && rank == 0) s_wcnt[warp][d] = __popc(peers);
        __syncthreads();
        int before = 0;
        for (int w = 0; w < warp; w++) before += s_wcnt[w][d];
        if (ok) {
            const int pos = s_base[d] + before + rank;
            keys_out[pos] = key;
            vals_out[pos] = vals[i];
        }
        __syncthreads();
        int tot = 0;                                                 // thread = digit: advance its base by the round's count
        for (int w = 0; w < RS_THREADS / 32; w++) tot += s_wcnt[w][threadIdx.x];
        s_base[threadIdx.x] += tot;
        __syncthreads();
    }
}

// Sorts (keys_a, vals_a) by bits [0, nbits) of the key into (keys_b, vals_b); keys_a / vals_a are overwritten (they
// serve as the other half of the ping-pong).  hist: int[256 * radix_sort_ctas(n)] scratch.  Asynchronous on stream.
static inline int radix_sort_ctas(int n) { return (n + RS_TILE - 1) / RS_TILE; }
static int radix_sort_pairs(unsigned long long *keys_a, int *vals_a, unsigned long long *keys_b, int *vals_b, int n, int nbits,
                            int *hist, cudaStream_t st, long *launches)
{
    if (n <= 0) return PYGBE_OK;
    const int ncta = radix_sort_ctas(n), passes = (nbits + 7) / 8;
    unsigned long long *ki = keys_a, *ko = keys_b;
    int *vi = vals_a, *vo = vals_b;
    for (int p = 0; p < passes; p++) {
        k_rs_hist<<<ncta, RS_THREADS, 0, st>>>(ki, n, 8 * p, ncta, hist);
        k_rs_scan<<<1, 1024, 0, st>>>(hist, 256L * ncta);
        k_rs_scatter<<<ncta, RS_THREADS, 0, st>>>(ki, vi, n, 8 * p, ncta, hist, ko, vo);
        if (launches) *launches += 3;
        std::swap(ki, ko); std::swap(vi, vo);
    }
    if (ki != keys_b) {                                              // an even number of passes ended in (keys_a, vals_a)
        CUDA_TRY(cudaMemcpyAsync(keys_b, keys_a, (size_t)n * sizeof(unsigned long long), cudaMemcpyDeviceToDevice, st));
        CUDA_TRY(cudaMemcpyAsync(vals_b, vals_a, (size_t)n * sizeof(int), cudaMemcpyDeviceToDevice, st));
    }
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}
