// Roofline denominators measured on the box the bench runs on (bench.py calls these before its
// timed region): register-resident FP64 loops -- DMMA.8x8x4 (the FP64 tensor pipe the Gram kernel
// uses) and DFMA -- and a STREAM-style 128-bit copy.  MEASURED_PEAKS.json carries no FP64 figure,
// so the Gram's `roofline.peak` is this probe's DMMA number.
// Not part of librsdft's ABI; built as libpeakprobe.so.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

template <int ILP>
__global__ void dfma_loop(double *out, int iters, double a, double b)
{
    double acc[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) acc[i] = threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int NACC>
__global__ void dmma_loop(double *out, int iters, double a, double b)
{
    double c0[NACC], c1[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) { c0[i] = 0; c1[i] = 0; }
    const double fa = a + threadIdx.x * 1e-9, fb = b;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c0[i]), "+d"(c1[i]) : "d"(fa), "d"(fb));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void copy_loop(const double2 *__restrict__ in, double2 *__restrict__ out, size_t n)
{
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) out[i] = in[i];
}

}  // namespace

extern "C" {

// kind 0: DMMA.8x8x4, kind 1: DFMA.  Runs `reps` back-to-back launches (~2.6 ms each) and returns
// FLOP/s over the whole train (sustained figure when reps is large).  Returns 0 or a cudaError_t.
int peak_probe_fp64(int kind, int reps, double *tflops)
{
    int dev = 0, nsm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    double *out = nullptr;
    if ((e = cudaMalloc((void **)&out, (size_t)nsm * 2 * 512 * sizeof(double))) != cudaSuccess) return (int)e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = nsm * 2;
    double flops_per_launch;
    if (kind == 0) {
        dmma_loop<16><<<blocks, 256>>>(out, 100, 1.0, 1e-9);
        flops_per_launch = 2.0 * 256 * 16 * 5000.0 * 8 * blocks;
    } else {
        dfma_loop<8><<<blocks, 512>>>(out, 100, 1.0000001, 1e-9);
        flops_per_launch = 2.0 * 8 * 20000.0 * 512 * blocks;
    }
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    for (int r = 0; r < reps; ++r) {
        if (kind == 0) dmma_loop<16><<<blocks, 256>>>(out, 5000, 1.0, 1e-9);
        else dfma_loop<8><<<blocks, 512>>>(out, 20000, 1.0000001, 1e-9);
    }
    cudaEventRecord(e1);
    e = cudaDeviceSynchronize();
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    *tflops = flops_per_launch * reps / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return (int)e;
}

// 128-bit grid-stride copy over 2 x 2 GiB; GB/s counts read + write bytes; best of `reps`.
int peak_probe_copy(int reps, double *gbs)
{
    int dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const size_t n = (size_t)1 << 27;
    double2 *a = nullptr, *b = nullptr;
    cudaError_t e = cudaMalloc((void **)&a, n * 16);
    if (e == cudaSuccess) e = cudaMalloc((void **)&b, n * 16);
    if (e != cudaSuccess) { cudaFree(a); return (int)e; }
    cudaMemset(a, 0, n * 16);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0);
        copy_loop<<<nsm * 16, 512>>>(a, b, n);
        cudaEventRecord(e1);
        e = cudaDeviceSynchronize();
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double v = 2.0 * n * 16 / (ms * 1e-3) / 1e9;
        if (r > 0 && v > best) best = v;
    }
    *gbs = best;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(a);
    cudaFree(b);
    return (int)e;
}

}  // extern "C"
