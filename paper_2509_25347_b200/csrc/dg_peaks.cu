// dg_peaks.cu — microbenchmark kernels behind dg_peak_kernel (include/dg.h): the roofline denominators that
// MEASURED_PEAKS.json does not hold (sustained fp64 FMA and fp64 tensor-core rates) and an fp64 copy.
// Not on the data path; bench.py times one launch of each with CUDA events.
#include <cstdint>

#include "../../include/dg.h"
#include "dg_internal.h"

namespace dg {
dg_status cuda_status(cudaError_t e);

namespace {

constexpr int kPeakThreads = 256;
constexpr int kChains = 8;

__global__ void __launch_bounds__(kPeakThreads) k_peak_dfma(int iters, double* sink) {
    double x[kChains];
    const double a = 0.999999 + 1e-9 * threadIdx.x, b = 1e-7;
#pragma unroll
    for (int k = 0; k < kChains; ++k) x[k] = 1.0 + k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int k = 0; k < kChains; ++k) x[k] = fma(x[k], a, b);
    }
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < kChains; ++k) acc += x[k];
    if (acc == 123.456) sink[0] = acc;  // never true; keeps the chains alive
}

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_dmma(int iters, double* sink) {
    double c[4][2];
    const double a = 1e-3 * (threadIdx.x & 31), b = 1e-3;
#pragma unroll
    for (int k = 0; k < 4; ++k) c[k][0] = c[k][1] = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int k = 0; k < 4; ++k) dmma884(c[k][0], c[k][1], a, b);
    }
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) acc += c[k][0] + c[k][1];
    if (acc == 123.456) sink[0] = acc;
}

// per iteration and warp: 4 DMMA (4 * 256 FMA) and 32 DFMA per lane (32 * 32 FMA): the same FMA count on each pipe
__global__ void __launch_bounds__(kPeakThreads) k_peak_mixed(int iters, double* sink) {
    double c[4][2], x[kChains];
    const double a = 1e-3 * (threadIdx.x & 31), b = 1e-3, fa = 0.999999, fb = 1e-7;
#pragma unroll
    for (int k = 0; k < 4; ++k) c[k][0] = c[k][1] = 0.0;
#pragma unroll
    for (int k = 0; k < kChains; ++k) x[k] = 1.0 + k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            dmma884(c[k][0], c[k][1], a, b);
#pragma unroll
            for (int j = 0; j < kChains; ++j) x[j] = fma(x[j], fa, fb);
        }
    }
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) acc += c[k][0] + c[k][1];
#pragma unroll
    for (int k = 0; k < kChains; ++k) acc += x[k];
    if (acc == 123.456) sink[0] = acc;
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_copy(const double2* __restrict__ src, double2* __restrict__ dst,
                                                            long long n2) {
    const long long stride = (long long)gridDim.x * kPeakThreads;
    for (long long i = (long long)blockIdx.x * kPeakThreads + threadIdx.x; i < n2; i += stride) dst[i] = src[i];
}

}  // namespace
}  // namespace dg

using namespace dg;

extern "C" dg_status dg_peak_kernel(int kind, int iters, double* scratch, long long scratch_bytes, double* work,
                                    void* stream) {
    if (scratch == nullptr || work == nullptr) return DG_ENULL;
    if (scratch_bytes < (1 << 20) || kind < 0 || kind > 3 || iters < 1) return DG_EINVAL;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_status(e);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int blocks = sms * 8;  // 2048 resident threads per SM
    const double threads = (double)blocks * kPeakThreads;
    switch (kind) {
        case 0:
            k_peak_dfma<<<blocks, kPeakThreads, 0, st>>>(iters, scratch);
            *work = threads * iters * 4.0 * kChains * 2.0;
            break;
        case 1:
            k_peak_dmma<<<blocks, kPeakThreads, 0, st>>>(iters, scratch);
            *work = (threads / 32.0) * iters * 8.0 * (2.0 * 8 * 8 * 4);
            break;
        case 2:
            k_peak_mixed<<<blocks, kPeakThreads, 0, st>>>(iters, scratch);
            *work = (threads / 32.0) * iters * 4.0 * (2.0 * 8 * 8 * 4) + threads * iters * 4.0 * kChains * 2.0;
            break;
        case 3: {
            const long long half = (scratch_bytes / 2) & ~255LL;
            const long long n2 = half / (long long)sizeof(double2);
            k_peak_copy<<<sms * 16, kPeakThreads, 0, st>>>(reinterpret_cast<const double2*>(scratch),
                                                          reinterpret_cast<double2*>((char*)scratch + half), n2);
            *work = 2.0 * (double)half;
            break;
        }
    }
    return cuda_status(cudaGetLastError());
}
