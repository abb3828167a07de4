// bench_probes.cu -- measurement aids of bench.py (`python bench.py --probes`), NOT part of libfew_b200 and not on the product
// path: small kernels that measure the facts of the B200 FP64 pipe the summation kernel is designed around (DESIGN.md
// section 5).  Built by __graft_entry__.build() / bench.py into bench_probes.so next to bench.py.
//
//   probe_dmma_mix(blocks, warps_dmma, iters, chain, mode, ms_out)
//     512-thread blocks = 16 warps = 4 per scheduler.  The warps 4 j .. 4 j + 3 with j < warps_dmma run batches of 16
//     DMMA.8x8x4 (mma.sync.m8n8k4.f64), 8 accumulators; between two batches each of them executes `chain` dependent DFMAs.
//     The other warps: mode 0 idle, mode 1 one dependent DFMA chain, mode 2 eight independent DFMA chains.
//     A DMMA holds the pipe 16 cycles, so warps_dmma warps per scheduler need 256 * warps_dmma cycles per iteration at best;
//     what the scalar instructions cost the DMMA stream is read off the iteration time.
#include <cuda_runtime.h>

namespace {

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(512, 1) probe_dmma_mix_kernel(int iters, int warps_dmma, int chain, int mode, double* sink)
{
    const int w = threadIdx.x >> 5;
    double r = 0.0;
    if ((w >> 2) < warps_dmma) {
        double c0[8], c1[8], a[4];
        const double b0 = 1e-3 * (threadIdx.x & 15), b1 = 2e-3 * ((threadIdx.x + 1) & 15);
#pragma unroll
        for (int g = 0; g < 8; ++g) c0[g] = c1[g] = 0.0;
#pragma unroll
        for (int g = 0; g < 4; ++g) a[g] = 1e-3 * (threadIdx.x + g);
        double x = 1.0 + 1e-9 * threadIdx.x;
        for (int it = 0; it < iters; ++it) {
            for (int q = 0; q < chain; ++q) x = fma(x, 1.0000001, 1e-9);     // dependent scalar FP64 between the batches
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                dmma(c0[g], c1[g], a[g], b0); dmma(c0[4 + g], c1[4 + g], a[g], b1);
                dmma(c0[g], c1[g], a[g], b1); dmma(c0[4 + g], c1[4 + g], a[g], b0);
            }
        }
#pragma unroll
        for (int g = 0; g < 8; ++g) r += c0[g] + c1[g];
        r += x;
    } else if (mode == 1) {
        double x = 1.0 + 1e-9 * threadIdx.x;
        for (int it = 0; it < iters * 8; ++it) x = fma(x, 1.0000001, 1e-9);
        r = x;
    } else if (mode == 2) {
        double x[8];
#pragma unroll
        for (int g = 0; g < 8; ++g) x[g] = 1.0 + 1e-9 * threadIdx.x + g;
        for (int it = 0; it < iters * 8; ++it) {
#pragma unroll
            for (int g = 0; g < 8; ++g) x[g] = fma(x[g], 1.0000001, 1e-9);
        }
#pragma unroll
        for (int g = 0; g < 8; ++g) r += x[g];
    }
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = r;
}

}  // namespace

extern "C" int probe_dmma_mix(int blocks, int warps_dmma, int iters, int chain, int mode, float* ms_out)
{
    if (blocks <= 0 || warps_dmma < 1 || warps_dmma > 4 || iters <= 0 || chain < 0 || !ms_out) return -1;
    double* sink = nullptr;
    if (cudaMalloc(&sink, (size_t)blocks * 512 * sizeof(double)) != cudaSuccess) return -2;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    probe_dmma_mix_kernel<<<blocks, 512>>>(iters / 10 + 1, warps_dmma, chain, mode, sink);
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    probe_dmma_mix_kernel<<<blocks, 512>>>(iters, warps_dmma, chain, mode, sink);
    cudaEventRecord(e1);
    const cudaError_t err = cudaDeviceSynchronize();
    cudaEventElapsedTime(ms_out, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    return err == cudaSuccess ? 0 : -3;
}
