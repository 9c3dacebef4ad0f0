// alu_probe.cu — micro-benchmark of the ALU pipe: the measured denominator of the "alu" roofline.
// NOT part of the product ABI: built into its own libsg_probe.so, loaded by bench.py only.
// ("verify SM count, pipe width and sustained clock with a dependent-free LOP3
// micro-benchmark; that measured number is the denominator").
//
// Every thread runs 8 independent LOP3 chains (no memory traffic); 2 x 1024 threads per SM keep the
// pipe saturated.  lane-ops/s = threads x 8 x iterations x launches / time.
#include <cuda_runtime.h>
#include <stdint.h>


namespace {

__global__ void __launch_bounds__(1024) k_probe_lop3(uint32_t *out, uint32_t a0, uint32_t b0, int iters)
{
    uint32_t x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = threadIdx.x * 0x9E3779B9u + k * 0x85EBCA6Bu + blockIdx.x;
    const uint32_t a = a0 ^ threadIdx.x, b = b0 + blockIdx.x;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[k]) : "r"(a), "r"(b));
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s ^= x[k];
    if (s == 0x12345678u) out[0] = s;      // never true in practice; keeps the chains alive
}

}  // namespace

// Measured peak of the ALU (INT/LOP3) pipe of the current device on `cuda_stream` (NULL = default
// stream); best of 5 launches of ~10 ms.  *lane_ops_per_s = 32-bit lane operations per second.
// Returns 0, or -1 bad argument, -2 allocation failure, -3 CUDA error.  Synchronous.
extern "C" int sgprobe_alu_peak(void *cuda_stream, double *lane_ops_per_s)
{
    if (!lane_ops_per_s) return -1;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    uint32_t *out = nullptr;
    if (cudaMalloc(&out, 256) != cudaSuccess) return -2;
    const int grid = 2 * sms, threads = 1024, iters = 4096, reps = 5;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    k_probe_lop3<<<grid, threads, 0, st>>>(out, 1u, 2u, 64);                 // warm-up
    double best = 0.0;
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0, st);
        k_probe_lop3<<<grid, threads, 0, st>>>(out, 1u, 2u, iters);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return -3; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double ops = (double)grid * threads * 64.0 * iters;
        if (ms > 0.f && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (cudaGetLastError() != cudaSuccess) return -3;
    *lane_ops_per_s = best;
    return 0;
}
