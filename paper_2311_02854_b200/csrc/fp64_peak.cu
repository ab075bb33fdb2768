// FP64 pipe micro-benchmarks: the roofline denominator of the sigma kernels.
// MEASURED_PEAKS.json carries HBM and BF16 numbers only, so bench.py measures the FP64 peak itself,
// in the same process and under the same clocks as the kernels it is compared with:
//   which = 0: independent DFMA chains (the CUDA-core FP64 path)
//   which = 1: independent DMMA.8x8x4 chains (mma.sync m8n8k4 f64, the FP64 tensor path of sm_100a)
#include "common.h"

namespace dmrg {
namespace {

constexpr int NACC = 8;

__global__ void __launch_bounds__(256) dfma_kernel(double* out, int iters, double a, double b) {
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; i++) acc[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NACC; i++) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; i++) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) dmma_kernel(double* out, int iters, double a, double b) {
    double c[NACC][2];
#pragma unroll
    for (int i = 0; i < NACC; i++) { c[i][0] = threadIdx.x * 1e-3 + i; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NACC; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; i++) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace
}  // namespace dmrg

extern "C" double dmrg_fp64_peak_tflops(int32_t which, double ms, void* cuda_stream) {
    using namespace dmrg;
    if (which != 0 && which != 1) { set_error("dmrg_fp64_peak_tflops: which must be 0 or 1"); return DMRG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        set_error("dmrg_fp64_peak_tflops: no CUDA device");
        return DMRG_ECUDA;
    }
    const int grid = prop.multiProcessorCount * 4, block = 256, iters = 20000;
    double* out = nullptr;
    if (cudaMalloc(&out, sizeof(double) * grid * block) != cudaSuccess) { set_error("dmrg_fp64_peak_tflops: cudaMalloc failed"); return DMRG_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const double flop_per_launch = (double)grid * block * iters * NACC * (which == 0 ? 2.0 : 2.0 * 8 * 8 * 4 / 32);
    auto run = [&]() {
        if (which == 0) dfma_kernel<<<grid, block, 0, st>>>(out, iters, 1.0000001, 1e-9);
        else dmma_kernel<<<grid, block, 0, st>>>(out, iters, 1.0000001, 1e-9);
    };
    run();   // warm-up
    cudaEventRecord(e0, st); run(); cudaEventRecord(e1, st);
    double result = DMRG_ECUDA;
    if (cudaEventSynchronize(e1) == cudaSuccess) {
        float one = 0.f;
        cudaEventElapsedTime(&one, e0, e1);
        const int reps = std::max(1, (int)(ms / std::max(one, 1e-3f)));
        cudaEventRecord(e0, st);
        for (int r = 0; r < reps; r++) run();
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) == cudaSuccess) {
            float tot = 0.f;
            cudaEventElapsedTime(&tot, e0, e1);
            result = flop_per_launch * reps / (tot * 1e-3) * 1e-12;
        }
    }
    if (result < 0) set_error("dmrg_fp64_peak_tflops: %s", cudaGetErrorString(cudaGetLastError()));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return result;
}
