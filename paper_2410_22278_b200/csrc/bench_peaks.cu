// Measurement helpers for bench.py -- NOT part of the product ABI (include/pbc_jk.h) and not linked into libpbc_jk.so.
// Built as libpbc_jk_benchpeaks.so.  Each entry point runs a dependency-free instruction stream on every SM of the
// current device and returns the achieved rate: the roofline denominators of the real-space kernels (FP64 FMA pipe,
// FP32 FMA pipe for the mixed-precision quartets) and of the reciprocal-space GEMMs (FP64 tensor cores, DMMA).
#include <cuda_runtime.h>
#include <cstdint>

namespace {

__global__ void __launch_bounds__(256) fp64_fma_kernel(int iters, double *out)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double b = 1.0000001, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 1.2345) out[0] = s;
}

__global__ void __launch_bounds__(256) fp32_fma_kernel(int iters, double *out)
{
    float a0 = threadIdx.x * 1e-6f, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const float b = 1.00001f, c = 1e-6f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fmaf(a0, b, c); a1 = fmaf(a1, b, c); a2 = fmaf(a2, b, c); a3 = fmaf(a3, b, c);
            a4 = fmaf(a4, b, c); a5 = fmaf(a5, b, c); a6 = fmaf(a6, b, c); a7 = fmaf(a7, b, c);
        }
    }
    const float s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 1.2345f) out[0] = s;
}

// mma.sync.m8n8k4.f64: 8x8x4 = 256 FMA = 512 flop per warp instruction; 8 independent accumulator pairs per warp
__global__ void __launch_bounds__(256) fp64_dmma_kernel(int iters, double *out)
{
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k][0] = threadIdx.x * 1e-9 + k; c[k][1] = k; }
    const double a = 1.0000001, b = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[k][0]), "+d"(c[k][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    if (s == 1.2345) out[0] = s;
}

// even warps issue DMMA, odd warps DFMA: do the FP64 tensor instruction and the FP64 FMA have pipes of their own?
// (B200: no -- the two rates add up to the single-instruction peak)
__global__ void __launch_bounds__(256) fp64_mixed_pipe_kernel(int iters, double *out)
{
    double s = 0;
    if (((threadIdx.x >> 5) & 1) == 0) {
        double c[8][2];
#pragma unroll
        for (int k = 0; k < 8; ++k) { c[k][0] = threadIdx.x * 1e-9 + k; c[k][1] = k; }
        const double a = 1.0000001, b = 1e-9;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                             : "+d"(c[k][0]), "+d"(c[k][1])
                             : "d"(a), "d"(b));
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    } else {
        double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
        const double b = 1.0000001, c = 1e-9;
        for (int i = 0; i < iters; ++i) {                   // 8 DFMA per iteration against the other warps' 8 DMMA
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
        s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    }
    if (s == 1.2345) out[0] = s;
}

// The inner loop of dgemm_kernel without its global loads: one 256-thread CTA per SM, 64 x 32 warp tiles, per k-step 12
// 8-byte shared-memory loads and 32 DMMA, a barrier per 8 k-steps; the same tile strides (36 and 136 doubles).
__global__ void __launch_bounds__(256) fp64_dmma_loop_kernel(int iters, double *out)
{
    constexpr int SA = 36, SB = 136;
    extern __shared__ double As[];                          // [128][SA], then Bs [32][SB]
    double *Bs = As + 128 * SA;
    for (int i = threadIdx.x; i < 128 * SA; i += 256) As[i] = 1e-9 * i;
    for (int i = threadIdx.x; i < 32 * SB; i += 256) Bs[i] = 1e-9 * i;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, wm = w >> 2, wn = w & 3;
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const double *as = As + (wm * 64 + (lane >> 2)) * SA + (lane & 3);
    const double *bs = Bs + (lane & 3) * SB + wn * 32 + (lane >> 2);
    for (int it = 0; it < iters; ++it) {
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 32; kk += 4) {
            double a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = as[i * 8 * SA + kk];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = bs[kk * SB + j * 8];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                                 : "+d"(acc[i][j][0]), "+d"(acc[i][j][1])
                                 : "d"(a[i]), "d"(b[j]));
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 1.2345) out[0] = s;
}

template <class Kern>
double run(Kern kern, int iters, double flop_per_thread_iter, int blocks_per_sm = 8, int dyn_smem = 0)
{
    int dev = 0, nsm = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return -1.0; }
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    double *d = nullptr;
    if (cudaMalloc(&d, 8) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = nsm * blocks_per_sm;
    kern<<<blocks, 256, dyn_smem>>>(iters / 8 + 1, d);
    cudaEventRecord(e0);
    kern<<<blocks, 256, dyn_smem>>>(iters, d);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (cudaGetLastError() != cudaSuccess || ms <= 0) return -1.0;
    return flop_per_thread_iter * (double)iters * 256.0 * blocks / (ms * 1e-3) * 1e-12;
}

}  // namespace

extern "C" {
// each returns 0 and the achieved TFLOP/s, or -1 without a usable CUDA device
int bench_fp64_fma_peak(int32_t iters, double *tflops)
{
    const double v = run(fp64_fma_kernel, iters, 2.0 * 64.0);
    if (v < 0 || !tflops) return -1;
    *tflops = v;
    return 0;
}
int bench_fp32_fma_peak(int32_t iters, double *tflops)
{
    const double v = run(fp32_fma_kernel, iters, 2.0 * 64.0);
    if (v < 0 || !tflops) return -1;
    *tflops = v;
    return 0;
}
int bench_fp64_dmma_peak(int32_t iters, double *tflops)
{
    const double v = run(fp64_dmma_kernel, iters, 8.0 * 512.0 / 32.0);
    if (v < 0 || !tflops) return -1;
    *tflops = v;
    return 0;
}
// DMMA (even warps) and DFMA (odd warps) side by side: the SUM of the two rates
int bench_fp64_mixed_pipe_peak(int32_t iters, double *tflops)
{
    const double v = run(fp64_mixed_pipe_kernel, iters, 0.5 * (8.0 * 512.0 / 32.0 + 8.0 * 2.0));
    if (v < 0 || !tflops) return -1;
    *tflops = v;
    return 0;
}
// dgemm_kernel's inner loop (shared-memory fragment loads, DMMA, barrier) without the global loads
int bench_fp64_dmma_loop_peak(int32_t iters, double *tflops)
{
    const int smem = (128 * 36 + 32 * 136) * 8;
    if (cudaFuncSetAttribute(fp64_dmma_loop_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    const double v = run(fp64_dmma_loop_kernel, iters / 16 + 1, 8.0 * 32.0 * 512.0 / 32.0, 1, smem);
    if (v < 0 || !tflops) return -1;
    *tflops = v;
    return 0;
}
}
