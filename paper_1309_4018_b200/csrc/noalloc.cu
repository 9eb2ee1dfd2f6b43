// noalloc.cu -- ONE entry point that allocates nothing: pygbe_coulomb_energy_noalloc (include/pygbe.h).
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it).  It is a variant of k_coulomb (nearfield.cuh; eq. 8), the kernel behind pygbe_energy's Coulomb
// term, which needs scratch memory: the charges packed as (x, y, z, q) records and a device accumulator.  The existing
// path takes both from the handle's workspace / pool; this one takes them from a file-scope
//     static __device__ __align__(256) array of PYGBE_NOALLOC_MAX_CHARGES records + one accumulator line (512.25 KB),
// which every GPU that loads the library holds until the process exits.  Inputs and output are the caller's.
//
// In host code the array's NAME is a host-side stand-in, not a device address (a kernel given it would fault or, where
// the GPU can reach host memory, silently use the wrong memory): the address is taken once per device, with that device
// current, by cudaGetSymbolAddress in this same translation unit, and that pointer is what the kernels receive.
//
// Every call shares the array, which keeps the last call's contents: each call overwrites the records it uses and
// clears the accumulator first.  Calls that overlap on the GPU (two streams, two host threads) race on it.
// No existing code path is changed; nothing here is used by pygbe_energy.
#include <mutex>
#include "common.cuh"

#define NA_MAXQ PYGBE_NOALLOC_MAX_CHARGES
#define NA_ACC_OFF (4 * (size_t)NA_MAXQ)                 // doubles: records first, then the accumulator line
static __device__ __align__(256) double g_na_scratch[4 * (size_t)NA_MAXQ + 32];

static std::mutex g_na_mu;
static double *g_na_ptr[64] = {nullptr};                 // device address of g_na_scratch, per device ordinal

// records (x, y, z, q) from the caller's arrays; thread 0 clears the accumulator (stale from the last call)
__global__ void __launch_bounds__(256)
k_na_pack(long n, const double *__restrict__ xyz, const double *__restrict__ q, double *__restrict__ scratch)
{
    const long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k == 0) scratch[NA_ACC_OFF] = 0.0;
    if (k >= n) return;
    reinterpret_cast<double4 *>(scratch)[k] = make_double4(xyz[3 * k], xyz[3 * k + 1], xyz[3 * k + 2], q[k]);
}

// sum_{k != l} q_k q_l / r_kl  (a pair at zero distance contributes nothing, as in k_coulomb): thread = charge k, loop
// over all l through the packed records; warp shuffles, then one atomicAdd per warp into the accumulator
__global__ void __launch_bounds__(128)
k_na_coulomb(long n, double *__restrict__ scratch)
{
    const double4 *__restrict__ rec = reinterpret_cast<const double4 *>(scratch);
    const long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    double acc = 0.0;
    if (k < n) {
        const double4 X = rec[k];
        for (long l = 0; l < n; l++) {
            const double4 a = rec[l];
            const double dx = X.x - a.x, dy = X.y - a.y, dz = X.z - a.z;
            const double r2 = dx * dx + dy * dy + dz * dz;
            acc += r2 > 0.0 ? a.w * rsqrt(r2) : 0.0;
        }
        acc *= X.w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(scratch + NA_ACC_OFF, acc);
}

__global__ void k_na_finish(const double *__restrict__ scratch, double factor, double *__restrict__ E)
{
    E[0] = factor * scratch[NA_ACC_OFF];
}

// once per device, with that device current
static int na_setup(int device)
{
    if (device < 0 || device >= 64) { pygbe_set_error("noalloc: device %d out of range", device); return PYGBE_EINVAL; }
    CUDA_TRY(cudaSetDevice(device));
    std::lock_guard<std::mutex> lk(g_na_mu);
    if (g_na_ptr[device]) return PYGBE_OK;
    double *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_na_scratch);
    if (e != cudaSuccess || !p) {
        pygbe_set_error("noalloc: cudaGetSymbolAddress on device %d failed: %s", device, cudaGetErrorString(e));
        return PYGBE_ECUDA;
    }
    g_na_ptr[device] = p;
    return PYGBE_OK;
}

extern "C" int pygbe_noalloc_setup(int32_t device) { return na_setup(device); }

extern "C" int pygbe_coulomb_energy_noalloc(int32_t device, void *stream, const double *xyz_dev, const double *q_dev, int64_t n,
                                            double eps, double *E_dev)
{
    if (!E_dev || n < 0 || (n > 0 && (!xyz_dev || !q_dev))) { pygbe_set_error("coulomb_energy_noalloc: null pointer or negative size"); return PYGBE_EINVAL; }
    if (!(eps > 0.0)) { pygbe_set_error("coulomb_energy_noalloc: eps must be > 0"); return PYGBE_EINVAL; }
    if (n > NA_MAXQ) {
        pygbe_set_error("coulomb_energy_noalloc: %ld charges exceed the maximum of %d that the static scratch array holds "
                        "(PYGBE_NOALLOC_MAX_CHARGES); use pygbe_energy on a handle instead", (long)n, NA_MAXQ);
        return PYGBE_EINVAL;
    }
    TRY(na_setup(device));                                // sets the device; takes the address on first use
    cudaStream_t st = (cudaStream_t)stream;
    double *scratch = g_na_ptr[device];
    if (n < 2) {                                          // no pair: E = 0 (a memset is not an allocation)
        CUDA_TRY(cudaMemsetAsync(E_dev, 0, sizeof(double), st));
        return PYGBE_OK;
    }
    // reading A17: C0 = qe^2 N_A 1e7 / eps0 kJ A / (mol e^2);  E = 1/2 C0 sum_{k != l} q_k q_l / (4 pi eps r_kl)
    const double qe = 1.60217646e-19, NA = 6.0221415e23, eps0 = 8.854187818e-12;
    const double C0 = qe * qe * NA * 1e7 / eps0;
    const double factor = 0.5 * C0 / (4.0 * 3.14159265358979323846 * eps);
    k_na_pack<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((long)n, xyz_dev, q_dev, scratch);
    k_na_coulomb<<<(unsigned)((n + 127) / 128), 128, 0, st>>>((long)n, scratch);
    k_na_finish<<<1, 1, 0, st>>>(scratch, factor, E_dev);
    CUDA_TRY(cudaGetLastError());
    return PYGBE_OK;
}
