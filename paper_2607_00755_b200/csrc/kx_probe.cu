// kx_probe.cu -- measurement aid: peak FP64 throughput of this GPU, the denominator of the roofline fraction that
// bench.py reports for the contraction kernel.  Register-resident dependent chains, no memory traffic:
//   kind 0: DFMA, 16 independent chains per thread;  kind 1: DMMA.8x8x4 (mma.sync.m8n8k4.f64), 8 chains per warp.
#include "kx_internal.cuh"

namespace {

__global__ void k_probe_dfma(double* out, int iters, double a, double b)
{
    double x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = threadIdx.x * 1e-9 + k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) x[k] = fma(x[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_probe_dmma(double* out, int iters, double a, double b)
{
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k][0] = threadIdx.x; c[k][1] = k; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" kx_status_t kx_probe_flops(int device, int32_t kind, double* tflops)
{
    if (!tflops || (kind != 0 && kind != 1)) return KX_ERR_INVALID_ARG;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return KX_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return KX_ERR_CUDA;
    const int grid = prop.multiProcessorCount * 2, threads = 256, iters = 20000;
    double* out = nullptr;
    cudaEvent_t e0, e1;
    kx_status_t rc = KX_OK;
    if (cudaMalloc(&out, (size_t)grid * threads * 8) != cudaSuccess) { cudaSetDevice(prev); return KX_ERR_ALLOC; }
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) k_probe_dfma<<<grid, threads>>>(out, iters, 1.0000001, 1e-9);
        else k_probe_dmma<<<grid, threads>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = KX_ERR_CUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    const double flop = kind == 0 ? 2.0 * 16 * iters * (double)grid * threads
                                  : 2.0 * 256 * 8 * iters * (double)grid * threads / 32;
    *tflops = flop / (best * 1e-3) * 1e-12;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    cudaSetDevice(prev);
    return rc;
}
