// Measured arithmetic ceilings of the device the library runs on, for the roofline of the kernels that are bound by
// instruction issue / the fp64 pipe rather than by HBM (the neighbor-matrix build: DESIGN.md section 6).  Not on the
// time-step path.  Register-resident loops timed with CUDA events on the caller's stream:
//   fp64: 8 independent DFMA chains per thread, 1024 resident threads per SM  -> TFLOP/s (2 flops per DFMA)
//   fp32: the same with FFMA
#include <algorithm>

#include "md_types.h"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_fma_peak(T *out, int iters, T a, T b)
{
    T x[8];
#pragma unroll
    for (int k = 0; k < 8; k++) x[k] = (T)(threadIdx.x + k) * (T)1e-9;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < 8; k++) x[k] = fma(x[k], a, b);
    }
    T s = 0;
#pragma unroll
    for (int k = 0; k < 8; k++) s += x[k];
    if (s == (T)123456.789) out[blockIdx.x] = s;        // never true: keeps the loop alive
}

template <typename T>
double measure(cudaStream_t st, int sms, T *scratch)
{
    const int blocks = sms * 8, iters = sizeof(T) == 8 ? 4096 : 16384;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 0.0;
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        cudaEventRecord(e0, st);
        k_fma_peak<T><<<blocks, 256, 0, st>>>(scratch, iters, (T)0.999999, (T)1e-7);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 8.0 * (double)iters * 256.0 * (double)blocks;
        if (rep > 0 && ms > 0.f) best = std::max(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best;
}

}  // namespace

// scratch: at least 8 * sms doubles of device memory.  Returns TFLOP/s (0 on failure).
double mdk_peak_fp64(cudaStream_t st, int sms, double *scratch) { return measure<double>(st, sms, scratch); }
double mdk_peak_fp32(cudaStream_t st, int sms, double *scratch) { return measure<float>(st, sms, (float *)scratch); }
