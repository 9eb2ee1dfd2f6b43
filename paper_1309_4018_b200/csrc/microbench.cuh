// microbench.cuh -- ALU peak probes used as roofline denominators for the P2P / M2P stages, whose bound
// is the CUDA-core pipes and not HBM or the tensor cores (MEASURED_PEAKS.json holds only the latter two).
// Dependent FMA chains, 8 per thread, enough warps to fill every SM; one MUFU.RSQ chain set for the SFU.
#pragma once
#include "common.cuh"
#include "m2p.cuh"

template <typename T>
__global__ void __launch_bounds__(256) k_fma_peak(int iters, T a, T b, T *out)
{
    T x0 = T(threadIdx.x), x1 = x0 + T(1), x2 = x0 + T(2), x3 = x0 + T(3);
    T x4 = x0 + T(4), x5 = x0 + T(5), x6 = x0 + T(6), x7 = x0 + T(7);
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b;
            x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
        }
    }
    T s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == T(-12345)) out[0] = s;          // never true; keeps the chains alive
}

__global__ void __launch_bounds__(256) k_mufu_peak(int iters, float *out)
{
    float x0 = 1.0f + threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            x0 = rsqrtf(x0); x1 = rsqrtf(x1); x2 = rsqrtf(x2); x3 = rsqrtf(x3);
        }
    }
    float s = x0 + x1 + x2 + x3;
    if (s == -12345.f) out[0] = s;
}

// A register-resident mix that looks like the Taylor recurrences: per element one FMUL and one three-register
// FFMA over 24 live values with scattered operand indices (3 flops per 2 instructions).  It measures what the
// FP32 pipe delivers once operands come from three different registers (bank conflicts in the operand
// collector), i.e. the practical ceiling of the M2P / P2P instruction mix, below the pure-FMA peak.
__global__ void __launch_bounds__(128) k_mix_peak(int iters, float *out)
{
    float v[24];
#pragma unroll
    for (int i = 0; i < 24; i++) v[i] = 1.0f + 1e-3f * (threadIdx.x + i);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 24; i++) v[i] = v[(i + 7) % 24] * v[(i + 13) % 24] + v[i] * 0.5f;
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 24; i++) s += v[i];
    if (s == -12345.f) out[0] = s;
}

// The instruction stream of the Laplace-form M2P with nothing around it: lap_poly<8, float> (164 Horner steps on four
// targets = 328 FFMA2 with a scalar coefficient operand read from shared memory by broadcast LDS.128) on register-
// resident arguments, no staging, no offsets, no accumulation.  What it reaches is the ceiling of that pattern on this
// machine (0.74-0.75 of the nominal FMA peak on B200, with 4 or 8 targets per thread alike), against which k_m2p_lap's
// fraction is to be read.
__global__ void __launch_bounds__(32) k_horner_peak(int ncell, const float *__restrict__ wg, float *out)
{
    __shared__ __align__(16) float s_w[8][m2p_lap_stride(8)];
    for (int i = threadIdx.x; i < 8 * m2p_lap_stride(8); i += 32) s_w[i / m2p_lap_stride(8)][i % m2p_lap_stride(8)] = wg[i];
    __syncwarp();
    const int sub = threadIdx.x >> 4;
    float a = 1e-3f * threadIdx.x, acc = 0.f;
    for (int c = 0; c < ncell; c++) {
        typedef LapVec<float> V;
        const V p = lap_poly<8, float>(V::make(a, a + .1f, a + .2f, a + .3f), V::make(a + .01f, a + .11f, a + .21f, a + .31f),
                                       V::make(a + .02f, a + .12f, a + .22f, a + .32f), s_w[(2 * c + sub) & 7]);
        float o[4];
        p.get(o);
        acc += (o[0] + o[1]) + (o[2] + o[3]);
        a += 1e-4f;
    }
    if (acc == -12345.f) out[0] = acc;
}

// out[0] = fp32 FMA TFLOP/s, out[1] = fp64 FMA TFLOP/s, out[2] = MUFU.RSQ Gop/s, out[3] = fp32 FMUL + 3-register
// FFMA mix TFLOP/s (FMA = 2 flops, MUL = 1); best of 5 launches each
static int run_alu_peaks(int device, double *out)
{
    CUDA_TRY(cudaSetDevice(device));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, device));
    const int grid = prop.multiProcessorCount * 8, block = 256;
    void *buf;
    CUDA_TRY(cudaMalloc(&buf, 64));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0)); CUDA_TRY(cudaEventCreate(&e1));
    for (int which = 0; which < 3; which++) {
        const int iters = which == 1 ? 2048 : 4096;
        double best = 0.0;
        for (int rep = 0; rep < 6; rep++) {
            CUDA_TRY(cudaEventRecord(e0));
            if (which == 0) k_fma_peak<float><<<grid, block>>>(iters, 1.0000001f, 1e-7f, (float *)buf);
            else if (which == 1) k_fma_peak<double><<<grid, block>>>(iters, 1.0000001, 1e-7, (double *)buf);
            else k_mufu_peak<<<grid, block>>>(iters, (float *)buf);
            CUDA_TRY(cudaEventRecord(e1));
            CUDA_TRY(cudaEventSynchronize(e1));
            float ms = 0;
            CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
            double ops = (double)grid * block * iters * 8.0 * (which == 2 ? 4.0 : 8.0 * 2.0);
            if (rep > 0) best = std::max(best, ops / (ms * 1e-3));
        }
        out[which] = which == 2 ? best * 1e-9 : best * 1e-12;
    }
    {
        const int g2 = prop.multiProcessorCount * 16, iters = 4096;
        double best = 0.0;
        for (int rep = 0; rep < 6; rep++) {
            CUDA_TRY(cudaEventRecord(e0));
            k_mix_peak<<<g2, 128>>>(iters, (float *)buf);
            CUDA_TRY(cudaEventRecord(e1));
            CUDA_TRY(cudaEventSynchronize(e1));
            float ms = 0;
            CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0) best = std::max(best, (double)g2 * 128 * iters * 24.0 * 3.0 / (ms * 1e-3));
        }
        out[3] = best * 1e-12;
    }
    {   // out[4] = TFLOP/s of the bare Horner stream of k_m2p_lap<8, float> (2 flops per step and target)
        const int g3 = prop.multiProcessorCount * 16, ncell = 400;
        float *wg;
        CUDA_TRY(cudaMalloc(&wg, 8 * m2p_lap_stride(8) * sizeof(float)));
        CUDA_TRY(cudaMemset(wg, 0, 8 * m2p_lap_stride(8) * sizeof(float)));
        double best = 0.0;
        for (int rep = 0; rep < 6; rep++) {
            CUDA_TRY(cudaEventRecord(e0));
            k_horner_peak<<<g3, 32>>>(ncell, wg, (float *)buf);
            CUDA_TRY(cudaEventRecord(e1));
            CUDA_TRY(cudaEventSynchronize(e1));
            float ms = 0;
            CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0) best = std::max(best, (double)g3 * 32 * ncell * 4.0 * 164.0 * 2.0 / (ms * 1e-3));
        }
        out[4] = best * 1e-12;
        cudaFree(wg);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    return PYGBE_OK;
}
