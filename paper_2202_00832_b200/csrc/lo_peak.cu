// lo_peak.cu -- in-run roofline denominators (lo_measure_peak): register-resident DMMA.8x8x4 and DFMA loops
// (FP64 tensor / FMA pipes) and an HBM stream copy.  BASELINE.json:north_star asks for the FP64 peak measured by
// an in-run microbenchmark; MEASURED_PEAKS.json has no FP64 entry.
#include <algorithm>

#include "lo_internal.h"

namespace lo {
namespace {

__global__ void __launch_bounds__(256) k_peak_dmma(double* out, int iters, double x) {
    double c[16][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = x * threadIdx.x, b = x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(256) k_peak_dfma(double* out, int iters, double m) {
    double acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = threadIdx.x * 1e-3 + i;
    const double a = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[i] = fma(acc[i], m, a);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i];
    if (s == 12345.678) out[0] = s;
}

__global__ void k_copy(const double4* __restrict__ src, double4* __restrict__ dst, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x, stride = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) dst[i] = src[i];
}

}  // namespace

lo_status measure_peak(int device, int kind, double* value) {
#define PK(call)                                                                                      \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess) { set_error(std::string(#call) + ": " + cudaGetErrorString(e_)); return LO_ECUDA; } \
    } while (0)
    PK(cudaSetDevice(device));
    cudaDeviceProp prop;
    PK(cudaGetDeviceProperties(&prop, device));
    cudaEvent_t e0, e1;
    PK(cudaEventCreate(&e0));
    PK(cudaEventCreate(&e1));
    double best = 0;
    if (kind == 0 || kind == 1) {
        double* d = nullptr;
        PK(cudaMalloc(&d, 8));
        const int grid = prop.multiProcessorCount * 4, thr = 256, iters = 40000;
        for (int rep = 0; rep < 4; ++rep) {
            PK(cudaEventRecord(e0));
            if (kind == 0) k_peak_dmma<<<grid, thr>>>(d, iters, 1e-9);
            else k_peak_dfma<<<grid, thr>>>(d, iters, 1.0000001);
            PK(cudaEventRecord(e1));
            PK(cudaEventSynchronize(e1));
            float ms = 0;
            PK(cudaEventElapsedTime(&ms, e0, e1));
            double fl = kind == 0 ? 2.0 * 256 * 16 * (double)iters * grid * (thr / 32) : 2.0 * 8 * (double)iters * grid * thr;
            if (rep > 0) best = std::max(best, fl / (ms * 1e-3) * 1e-12);
        }
        cudaFree(d);
    } else if (kind == 2) {
        const size_t bytes = (size_t)2 << 30;   // 2 GiB each way, far larger than the 126 MB L2
        double4 *a = nullptr, *b = nullptr;
        PK(cudaMalloc(&a, bytes));
        PK(cudaMalloc(&b, bytes));
        PK(cudaMemset(a, 1, bytes));
        for (int rep = 0; rep < 6; ++rep) {
            PK(cudaEventRecord(e0));
            k_copy<<<prop.multiProcessorCount * 16, 512>>>(a, b, bytes / 32);
            PK(cudaEventRecord(e1));
            PK(cudaEventSynchronize(e1));
            float ms = 0;
            PK(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0) best = std::max(best, 2.0 * bytes / (ms * 1e-3) * 1e-9);
        }
        cudaFree(a);
        cudaFree(b);
    } else if (kind == 3 || kind == 4) {
        // gated experiment, not a roofline denominator: INT8-sliced tile on tcgen05 (3: microseconds per tile, 4: error vs fp64)
        double us = 0, err = 0;
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
        lo_status st = measure_int8_slicing(device, &us, &err);
        if (st != LO_OK) return st;
        *value = kind == 3 ? us : err;
        return LO_OK;
    } else {
        set_error("lo_measure_peak: kind must be 0 (DMMA), 1 (DFMA), 2 (HBM copy), 3 / 4 (INT8-slicing probe: us per tile / error)");
        return LO_EINVAL;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *value = best;
    return LO_OK;
#undef PK
}

}  // namespace lo
