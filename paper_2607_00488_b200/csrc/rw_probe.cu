// rw_probe.cu -- measurement helper of bench.py (include/rw_probe.h), built as librw_probe.so and not linked
// into librw.so: register-resident FP64 issue-rate probes that give the denominators of the FP64 roofline
// (DESIGN.md section 6).
//   kind 0: DFMA chains (16 independent accumulators per thread)
//   kind 1: DMMA m8n8k4 (8 independent accumulator tiles per warp)
#include <cuda_runtime.h>

#include "../../include/rw_probe.h"

namespace rw {

__global__ void __launch_bounds__(256) k_probe_dfma(double *out, int iters, double a, double b)
{
    double acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_probe_dmma(double *out, int iters, double a, double b)
{
    double c0[8], c1[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c0[i] = threadIdx.x * 1e-9 + i; c1[i] = i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c0[i]), "+d"(c1[i]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace rw

static int probe_grid()
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return 0;
    return sms * 2;
}

extern "C" size_t rw_probe_scratch_bytes(void) { return (size_t)probe_grid() * 256 * sizeof(double); }

extern "C" int rw_probe_fp64_peak(int32_t kind, int32_t iters, void *scratch_dev, size_t scratch_bytes, double *tflops,
                                  void *cuda_stream)
{
    const int grid = probe_grid();
    if (grid == 0) return -3;
    if (!tflops || !scratch_dev || iters <= 0 || (kind != 0 && kind != 1) ||
        scratch_bytes < (size_t)grid * 256 * sizeof(double))
        return -1;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    double *buf = (double *)scratch_dev;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -3;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, s);
        if (kind == 0) rw::k_probe_dfma<<<grid, 256, 0, s>>>(buf, iters, 1.0000001, 1e-9);
        else rw::k_probe_dmma<<<grid, 256, 0, s>>>(buf, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (cudaStreamSynchronize(s) != cudaSuccess || cudaGetLastError() != cudaSuccess) return -3;
    const double flop = (kind == 0) ? 2.0 * 16 * (double)iters * 256.0 * grid
                                    : 512.0 * 8 * (double)iters * 8.0 * grid;
    *tflops = flop / (best * 1e-3) / 1e12;
    return 0;
}
