// rqr_probe.cu -- FP64 peak probes (rqr_probe.h).  Measurement only: built into librqr_probe.so, which bench.py and
// the sweep scripts load for the roofline denominator; not part of librqr.so.
#include <cuda_runtime.h>
#include <stdint.h>
#include "rqr_probe.h"

__global__ void __launch_bounds__(256)
k_probe_dfma(int iters, double* __restrict__ sink)
{
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * blockIdx.x;
    double acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = (double)k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = fma(acc[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += acc[k];
    sink[(size_t)blockIdx.x * 256 + threadIdx.x] = s;
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256)
k_probe_dmma(int iters, double* __restrict__ sink)
{
    double a = 1e-3 * (threadIdx.x & 31), b = 1e-3 * (blockIdx.x & 7);
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k][0] = k; c[k][1] = -k; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) dmma884(c[k][0], c[k][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    sink[(size_t)blockIdx.x * 256 + threadIdx.x] = s;
}

// Even warps run the DFMA chains, odd warps the DMMA chains: if the two instruction kinds had pipes of their own
// the sum would approach DFMA peak + DMMA peak; if they share one FP64 data path it stays at the single peak.
__global__ void __launch_bounds__(256)
k_probe_mix(int iters, double* __restrict__ sink)
{
    const bool tensor = (threadIdx.x >> 5) & 1;
    double a = 1e-3 * (threadIdx.x & 31), b = 1e-3 * (blockIdx.x & 7);
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k][0] = k; c[k][1] = -k; }
    if (tensor) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 8; ++k) dmma884(c[k][0], c[k][1], a, b);
        }
    } else {
        a += 1.0;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 8; ++k) c[k][0] = fma(c[k][0], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    sink[(size_t)blockIdx.x * 256 + threadIdx.x] = s;
}

extern "C" int rqr_probe_fp64(int kind, int iters, int blocks, double* d_sink, double* flops_out,
                              void* stream)
{
    if (kind != RQR_PROBE_DFMA && kind != RQR_PROBE_DMMA && kind != RQR_PROBE_MIX) return -1;
    if (iters < 1) return -2;
    if (blocks < 1) return -3;
    if (!d_sink) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    if (kind == RQR_PROBE_DFMA) {
        k_probe_dfma<<<blocks, 256, 0, st>>>(iters, d_sink);
        if (flops_out) *flops_out = (double)blocks * 256.0 * iters * 8.0 * 2.0;
    } else if (kind == RQR_PROBE_DMMA) {
        k_probe_dmma<<<blocks, 256, 0, st>>>(iters, d_sink);
        if (flops_out) *flops_out = (double)blocks * 8.0 /*warps*/ * iters * 8.0 * 512.0;
    } else {
        k_probe_mix<<<blocks, 256, 0, st>>>(iters, d_sink);
        if (flops_out) *flops_out = (double)blocks * 4.0 * iters * 8.0 * 512.0 + (double)blocks * 128.0 * iters * 8.0 * 2.0;
    }
    return cudaGetLastError() == cudaSuccess ? 0 : -1000;
}
