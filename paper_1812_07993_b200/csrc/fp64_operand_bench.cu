// fp64_operand_bench.cu -- what bounds the FP64 pipe of sm_100a for the all-pairs distance filter (md_allpairs.cuh)?
// A stand-alone diagnostic, not part of libmd_b200.so:
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 paper_1812_07993_b200/csrc/fp64_operand_bench.cu -o fp64_operand_bench
//     ./fp64_operand_bench
// Every kernel runs the same number of DFMAs per thread (or DMMAs per warp) in a different operand pattern; the rates
// are the ceilings profiles/r02_counters.md section 3 quotes.  The finding: a DFMA whose three source operands are three
// different register pairs issues every 3 cycles, not every 2 (2/3 of the chain peak); sharing one operand between
// consecutive DFMAs (operand-reuse cache) recovers part of it; every integer instruction that consumes a result costs
// about as much as two DFMA slots.
#include <cstdio>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("%s: %s\n", #x, cudaGetErrorString(e_)); return 1; } } while (0)

constexpr int ITER = 4096, THREADS = 128;

enum Mode {
    CHAIN = 0,        // t[k] = fma(t[k], a0, q0): two loop-invariant operands (how md_measure_peaks defines the FP64 peak)
    SHARE4 = 1,       // t[w][b] = fma(q[w], a[b], t[w][b]), b fastest: groups of four DFMAs share q[w]
    DISTINCT = 2,     // three different register pairs in every DFMA
    SHARE4_LDS = 3,   // SHARE4 with the q operands read from shared memory (32-byte entries, as the filter's tile)
    FILTER = 4,       // SHARE4_LDS + running integer maximum of the results' high words: the shape of the filter loop
    DMMA_CHAIN = 5,   // mma.sync m8n8k4 f64: eight accumulating chains per warp
    DMMA_FILTER = 6   // D = A B + C with constant C, integer maximum of the results' high words
};

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b, double c0, double c1)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%4,%5};"
                 : "=d"(d0), "=d"(d1) : "d"(a), "d"(b), "d"(c0), "d"(c1));
}

template <int MODE>
__global__ void __launch_bounds__(THREADS) k(const double* __restrict__ in, double* __restrict__ out, int iters)
{
    __shared__ double4 sj[THREADS];
    double t[16], a[16], q[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        t[i] = in[threadIdx.x + THREADS * i]; a[i] = in[2048 + threadIdx.x + THREADS * i]; q[i] = in[4096 + threadIdx.x + THREADS * i];
    }
    sj[threadIdx.x] = make_double4(in[threadIdx.x], in[threadIdx.x + 1], in[threadIdx.x + 2], in[threadIdx.x + 3]);
    __syncthreads();
    int top[4] = {0, 0, 0, 0};
    for (int it = 0; it < iters; ++it) {
        if (MODE == CHAIN) {
#pragma unroll
            for (int r = 0; r < 12; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) t[i] = fma(t[i], a[0], q[0]);
        } else if (MODE == SHARE4) {
#pragma unroll
            for (int r = 0; r < 12; ++r)
#pragma unroll
                for (int w = 0; w < 4; ++w)
#pragma unroll
                    for (int b = 0; b < 4; ++b) t[w * 4 + b] = fma(q[w + 4 * (r % 3)], a[b + 4 * (r % 3)], t[w * 4 + b]);
        } else if (MODE == DISTINCT) {
#pragma unroll
            for (int r = 0; r < 12; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) t[i] = fma(q[(i + r) & 15], a[(i + 5 * r) & 15], t[i]);
        } else if (MODE == SHARE4_LDS || MODE == FILTER) {
#pragma unroll
            for (int u = 0; u < 16; u += 4) {
                double4 e[4];
                double tt[4][4];
#pragma unroll
                for (int w = 0; w < 4; ++w) e[w] = sj[(it * 16 + u + w) & (THREADS - 1)];
#pragma unroll
                for (int w = 0; w < 4; ++w)
#pragma unroll
                    for (int b = 0; b < 4; ++b) tt[w][b] = fma(e[w].z, a[b], MODE == FILTER ? e[w].w : t[w * 4 + b]);
#pragma unroll
                for (int w = 0; w < 4; ++w)
#pragma unroll
                    for (int b = 0; b < 4; ++b) tt[w][b] = fma(e[w].y, a[4 + b], tt[w][b]);
#pragma unroll
                for (int w = 0; w < 4; ++w)
#pragma unroll
                    for (int b = 0; b < 4; ++b) tt[w][b] = fma(e[w].x, a[8 + b], tt[w][b]);
#pragma unroll
                for (int w = 0; w < 4; ++w)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        if (MODE == FILTER) top[b] = max(top[b], __double2hiint(tt[w][b]));
                        else t[w * 4 + b] = tt[w][b];
                    }
            }
        } else if (MODE == DMMA_CHAIN) {
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) dmma(t[2 * i], t[2 * i + 1], a[i & 3], q[i >> 2], t[2 * i], t[2 * i + 1]);
        } else {
#pragma unroll
            for (int r = 0; r < 3; ++r) {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    dmma(t[2 * i], t[2 * i + 1], a[i & 3], q[i >> 2], a[4 + (i & 3)], a[4 + (i & 3)]);
                    top[i & 3] = max(top[i & 3], max(__double2hiint(t[2 * i]), __double2hiint(t[2 * i + 1])));
                }
                q[0] += 1.0; q[1] += 1.0;                   // stands in for the next B fragment
            }
        }
    }
    double s = top[0] + top[1] + top[2] + top[3];
#pragma unroll
    for (int i = 0; i < 16; ++i) s += t[i];
    out[blockIdx.x * THREADS + threadIdx.x] = s;
}

template <int MODE>
int run(const char* name, const double* in, double* out, int blocks)
{
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    k<MODE><<<blocks, THREADS>>>(in, out, 64);
    CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        CK(cudaEventRecord(e0));
        k<MODE><<<blocks, THREADS>>>(in, out, ITER);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    // flops per thread and iteration: 192 DFMAs; or 24 DMMAs per warp = 24 x 512 flops per 32 threads
    const bool tensor = MODE == DMMA_CHAIN || MODE == DMMA_FILTER;
    const double flops = (tensor ? 24.0 * 512.0 / 32.0 : 2.0 * 192.0) * ITER * (double)THREADS * blocks;
    const double tests = tensor ? flops / 8.0 : flops / 6.0;   // a distance test is 3 DFMAs, or 1/64 of a DMMA (K = 4)
    printf("%-72s %6.2f TFLOP/s   %.3e distance tests/s\n", name, flops / best * 1e-9, tests / best * 1e3);
    return 0;
}

int main()
{
    double *in, *out;
    int sms = 148;
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0));
    CK(cudaMalloc(&in, 8192 * sizeof(double)));
    CK(cudaMalloc(&out, (size_t)sms * 8 * THREADS * sizeof(double)));
    CK(cudaMemset(in, 0, 8192 * sizeof(double)));
    const int blocks = sms * 4;                  // 16 warps per SM; 8 blocks per SM give the same rates to 1 %
    if (run<CHAIN>("DFMA, two loop-invariant operands (chain; the peak's definition)", in, out, blocks)) return 1;
    if (run<SHARE4>("DFMA, 4 x 4 outer-product order: groups of four share one operand", in, out, blocks)) return 1;
    if (run<DISTINCT>("DFMA, three different register pairs per instruction", in, out, blocks)) return 1;
    if (run<SHARE4_LDS>("DFMA, groups of four, shared operand from shared memory", in, out, blocks)) return 1;
    if (run<FILTER>("DFMA, the filter loop: shared memory + integer max of the high words", in, out, blocks)) return 1;
    if (run<DMMA_CHAIN>("DMMA m8n8k4, accumulating chains", in, out, blocks)) return 1;
    if (run<DMMA_FILTER>("DMMA m8n8k4, constant C + integer max of the high words", in, out, blocks)) return 1;
    return 0;
}
