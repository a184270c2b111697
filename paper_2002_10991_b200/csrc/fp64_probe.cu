// fp64_probe.cu -- measures the FP64 ALU roofline denominators that MEASURED_PEAKS.json lacks
// (it has HBM and bf16 only): sustained DFMA throughput, DMMA (mma.sync m8n8k4 f64) throughput,
// and both issued from alternating warps of the same SM (do the pipes overlap?).
// Register-only kernels, all SMs, 8 independent accumulator chains per thread.
#include "../../include/elpa2_bt.h"

#include <cuda_runtime.h>

namespace {

__global__ void __launch_bounds__(512) probe_dfma(double *out, int iters, double a, double b)
{
    double c0 = threadIdx.x, c1 = c0 + 1, c2 = c0 + 2, c3 = c0 + 3, c4 = c0 + 4, c5 = c0 + 5, c6 = c0 + 6, c7 = c0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            c0 = fma(c0, a, b); c1 = fma(c1, a, b); c2 = fma(c2, a, b); c3 = fma(c3, a, b);
            c4 = fma(c4, a, b); c5 = fma(c5, a, b); c6 = fma(c6, a, b); c7 = fma(c7, a, b);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = c0 + c1 + c2 + c3 + c4 + c5 + c6 + c7;
}

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// mode 1: every warp issues DMMA; mode 2: even warps DMMA, odd warps DFMA
__global__ void __launch_bounds__(512) probe_dmma(double *out, int iters, double a, double b, int mode)
{
    const int warp = threadIdx.x >> 5;
    double c0 = threadIdx.x, c1 = c0 + 1, c2 = c0 + 2, c3 = c0 + 3, c4 = c0 + 4, c5 = c0 + 5, c6 = c0 + 6, c7 = c0 + 7;
    if (mode == 1 || (warp & 1) == 0) {
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                dmma884(c0, c1, a, b); dmma884(c2, c3, a, b); dmma884(c4, c5, a, b); dmma884(c6, c7, a, b);
            }
        }
    } else {
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                c0 = fma(c0, a, b); c1 = fma(c1, a, b); c2 = fma(c2, a, b); c3 = fma(c3, a, b);
                c4 = fma(c4, a, b); c5 = fma(c5, a, b); c6 = fma(c6, a, b); c7 = fma(c7, a, b);
            }
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = c0 + c1 + c2 + c3 + c4 + c5 + c6 + c7;
}

}  // namespace

extern "C" int elpa2_bt_probe_fp64(int kind, int iters, int reps, double *tflops)
{
    if (kind < 0 || kind > 2 || iters < 1 || reps < 1 || !tflops) return -1;
    int dev = 0, nsm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return (int)e;
    if ((e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return (int)e;
    const int threads = 512, blocks = nsm * 4;
    double *out = nullptr;
    if ((e = cudaMalloc(&out, sizeof(double) * threads * blocks)) != cudaSuccess) return (int)e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    auto launch = [&]() {
        if (kind == 0) probe_dfma<<<blocks, threads>>>(out, iters, 0.999999, 1e-9);
        else probe_dmma<<<blocks, threads>>>(out, iters, 0.5, 0.25, kind);
    };
    launch();   // warm-up
    cudaEventRecord(t0);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(t1);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(out);
    if (e != cudaSuccess) return (int)e;
    // flops per thread per iter: DFMA path 64 FMA = 128 flops; DMMA path 8 mma x 256 FMA / 32 lanes
    // = 64 FMA per lane = 128 flops: the same in every mode.
    const double flops = (double)reps * blocks * threads * (double)iters * 128.0;
    *tflops = flops / (ms * 1e-3) / 1e12;
    return 0;
}
