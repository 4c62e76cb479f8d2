// md_noalloc.cu -- md_kinetic_energy_noalloc: the K reduction of row a5 (T(t) is what the thermostat
// needs every step) for callers that cannot allocate device memory -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  Same two-pass reduction as k_energy_partial / k_energy_final of md_kernels.cuh
// (warp shuffle -> block -> fixed-order final sum), but the per-block partial sums live in a file-scope __device__ array
// instead of the caller's workspace.  Self-contained on purpose: it includes none of the other kernel headers (their
// non-template kernels would be defined twice in the library) and changes no existing code path.
//
// The scratch: NA_MAX_BLOCKS doubles = 32 KiB, held by every GPU that loads the library until the process exits.  One
// block of 256 threads reduces NA_PER_BLOCK = 1024 particles, so the entry point serves up to MD_NOALLOC_MAX_PARTICLES
// = 4,194,304 particles and rejects more.  Every call shares the array and finds the previous call's partial sums in
// it: a call overwrites every slot it later reads (slots [0, blocks)), so nothing has to be cleared -- and two calls that
// overlap on the GPU (different streams, or different host threads) race on it: serialise them.
#include "../../include/md.h"

#include <cuda_runtime.h>
#include <cstdio>
#include <mutex>

namespace {

constexpr int NA_THREADS = 256, NA_ITEMS = 4, NA_PER_BLOCK = NA_THREADS * NA_ITEMS;
constexpr int NA_MAX_BLOCKS = MD_NOALLOC_MAX_PARTICLES / NA_PER_BLOCK;
static_assert(NA_MAX_BLOCKS * NA_PER_BLOCK == MD_NOALLOC_MAX_PARTICLES, "maximum must be a whole number of blocks");

// In HOST code this name is a stand-in for the symbol, not a device address: the kernels below are given the address
// cudaGetSymbolAddress returns for the current device (resolved once per device in scratch_for_current_device()).
static __device__ __align__(256) double g_na_partial[NA_MAX_BLOCKS];

__device__ __forceinline__ double na_warp_sum(double v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// partial[b] = sum over particles [b * 1024, (b + 1) * 1024) of 1/2 m |v_i|^2; vel is the caller's device array [n][dim].
__global__ void __launch_bounds__(NA_THREADS) k_na_kinetic_partial(const double* __restrict__ vel, long long n, int dim,
                                                                   double mass, double* __restrict__ partial)
{
    __shared__ double sh[NA_THREADS / 32];
    double k = 0.0;
    const long long base = (long long)blockIdx.x * NA_PER_BLOCK;
#pragma unroll
    for (int u = 0; u < NA_ITEMS; ++u) {
        const long long i = base + u * NA_THREADS + threadIdx.x;          // coalesced over the block
        if (i < n) {
            const double vx = vel[i * dim], vy = vel[i * dim + 1], vz = dim == 3 ? vel[i * dim + 2] : 0.0;
            k += 0.5 * mass * (vx * vx + vy * vy + vz * vz);
        }
    }
    k = na_warp_sum(k);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = k;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < NA_THREADS / 32; ++q) t += sh[q];
        partial[blockIdx.x] = t;                                          // every slot the final pass reads is written here
    }
}

// out[0] = sum of partial[0 .. nblocks) in a fixed order (deterministic for a given input).
__global__ void __launch_bounds__(NA_THREADS) k_na_kinetic_final(const double* __restrict__ partial, int nblocks,
                                                                 double* __restrict__ out)
{
    __shared__ double sh[NA_THREADS / 32];
    double k = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += NA_THREADS) k += partial[b];
    k = na_warp_sum(k);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = k;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < NA_THREADS / 32; ++q) t += sh[q];
        out[0] = t;
    }
}

// Device address of the scratch array on the CURRENT device, resolved once per device (set-up: may load the module).
constexpr int NA_MAX_DEVICES = 64;
double* g_na_ptr[NA_MAX_DEVICES] = {};
std::mutex g_na_mutex;

cudaError_t scratch_for_current_device(double** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_na_partial);
        if (e != cudaSuccess) return e;
        g_na_ptr[dev] = p;
    }
    *out = g_na_ptr[dev];
    return cudaSuccess;
}

int fail(int code, char* errbuf, size_t errbuf_len, const char* what, const char* detail = "")
{
    if (errbuf && errbuf_len) snprintf(errbuf, errbuf_len, "md_kinetic_energy_noalloc: %s%s", what, detail);
    return code;
}

} // namespace

extern "C" int md_kinetic_energy_noalloc(const double* vel_device, long long n, int dim, double mass, double* kinetic_device,
                                         void* cuda_stream, char* errbuf, size_t errbuf_len)
{
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (!vel_device || !kinetic_device) return fail(MD_ERR_INVALID_ARG, errbuf, errbuf_len, "vel_device / kinetic_device is NULL");
    if (dim != 2 && dim != 3) return fail(MD_ERR_INVALID_ARG, errbuf, errbuf_len, "dim must be 2 or 3");
    if (!(mass > 0)) return fail(MD_ERR_INVALID_ARG, errbuf, errbuf_len, "mass must be > 0");
    if (n < 1) return fail(MD_ERR_INVALID_ARG, errbuf, errbuf_len, "n must be >= 1");
    if (n > (long long)MD_NOALLOC_MAX_PARTICLES)
        return fail(MD_ERR_WORKSPACE, errbuf, errbuf_len, "n exceeds MD_NOALLOC_MAX_PARTICLES = 4194304 (the static scratch array holds "
                                                            "one partial sum per 1024 particles); use md_energy with a caller workspace");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(MD_ERR_CUDA, errbuf, errbuf_len, "no CUDA device (there is no CPU fallback)");
    }
    double* partial = nullptr;
    cudaError_t e = scratch_for_current_device(&partial);
    if (e != cudaSuccess) return fail(MD_ERR_CUDA, errbuf, errbuf_len, "cudaGetSymbolAddress: ", cudaGetErrorString(e));
    const int blocks = (int)((n + NA_PER_BLOCK - 1) / NA_PER_BLOCK);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_na_kinetic_partial<<<blocks, NA_THREADS, 0, st>>>(vel_device, n, dim, mass, partial);
    k_na_kinetic_final<<<1, NA_THREADS, 0, st>>>(partial, blocks, kinetic_device);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MD_ERR_CUDA, errbuf, errbuf_len, "kernel launch: ", cudaGetErrorString(e));
    return MD_OK;
}
