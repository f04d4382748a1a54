// probe.cu -- libgcamb_probe.so (include/gcamb_probe.h): FP64 roofline denominators measured on the
// device by bench.py.  Not part of the method; shares nothing with libgcamb_los.so.
#include <cuda_runtime.h>
#include <stdint.h>

#include "gcamb_probe.h"

namespace {

__global__ void dfma_probe_kernel(long long iters, double *out)
{
    double a[8], m = 1.0 - 1e-9 * (threadIdx.x & 7), c = 1e-12;
#pragma unroll
    for (int q = 0; q < 8; ++q) a[q] = 1.0 + q;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) a[q] = fma(a[q], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += a[q];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void dmma_probe_kernel(long long iters, double *out)
{
    double d0[8], d1[8];
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (threadIdx.x & 7);
#pragma unroll
    for (int q = 0; q < 8; ++q) d0[q] = d1[q] = q;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(d0[q]), "+d"(d1[q]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += d0[q] + d1[q];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" int gcamb_probe_dfma(int32_t blocks, int32_t threads, int64_t iters, double *d_out, void *cuda_stream)
{
    if (blocks < 1 || threads < 1 || threads > 1024 || iters < 1 || !d_out) return (int)cudaErrorInvalidValue;
    dfma_probe_kernel<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>((long long)iters, d_out);
    return (int)cudaGetLastError();
}

extern "C" int gcamb_probe_dmma(int32_t blocks, int32_t threads, int64_t iters, double *d_out, void *cuda_stream)
{
    if (blocks < 1 || threads < 32 || threads > 1024 || threads % 32 || iters < 1 || !d_out) return (int)cudaErrorInvalidValue;
    dmma_probe_kernel<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>((long long)iters, d_out);
    return (int)cudaGetLastError();
}
