// peaks.cu -- measured fp64 peaks of the device the library runs on (
// DESIGN.md section 9): register-only kernels that keep the plain fp64 pipe busy, timed with CUDA
// events.  bench.py reports the transform kernels' flop rate against these numbers instead of
// the nominal 148 SM x 64 lanes x 2 x clock figure.
//   kind 0: DFMA only (2 flop per instruction)
//   kind 1: DADD and DMUL alternating (1 flop per instruction) -- the rate the butterflies'
//           add/sub-heavy parts can reach
#include <cmath>
#include "nsc_internal.h"

namespace nsc {

constexpr int PK_CHAINS = 8;      // independent dependency chains per thread
constexpr int PK_INNER = 64;      // unrolled instructions per chain per outer iteration

template <int KIND>
__global__ void __launch_bounds__(256) k_fp64_peak(double* sink, int outer, double a, double b) {
    double x[PK_CHAINS];
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) x[i] = 1.0 + 1e-9 * (double)(threadIdx.x + i);
    for (int o = 0; o < outer; ++o) {
#pragma unroll
        for (int k = 0; k < PK_INNER; ++k) {
#pragma unroll
            for (int i = 0; i < PK_CHAINS; ++i) {
                if (KIND == 0)
                    x[i] = fma(x[i], a, b);
                else if (k & 1)
                    x[i] = __dmul_rn(x[i], a);
                else
                    x[i] = __dadd_rn(x[i], b);
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) s += x[i];
    if (s == 123.456) sink[0] = s;      // never true: keeps the chains alive
}

}  // namespace nsc

using namespace nsc;

extern "C" int nsc_fp64_peak(int kind, int device, double* h_tflops) {
    if (!h_tflops || (kind != 0 && kind != 1)) return NSC_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return NSC_ECUDA;
    }
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return NSC_ECUDA;
    if (dev >= ndev) return NSC_EINVAL;
    DeviceGuard on_device(dev);                  // the caller's current device is put back on every return path
    if (!on_device.ok()) return NSC_ECUDA;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return NSC_ECUDA;
    double* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return NSC_ENOMEM;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        if (e0) cudaEventDestroy(e0);
        cudaFree(sink);
        return NSC_ECUDA;
    }
    const int grid = sms * 8, outer = 2048;     // 8 CTAs of 8 warps per SM: every scheduler has 16 warps to pick from
    const double a = 0.999999999, b = 1e-9;
    double best = 0.0;
    bool failed = false;
    for (int rep = 0; rep < 6 && !failed; ++rep) {   // first repetitions warm the clocks up; the best one counts
        failed = cudaEventRecord(e0) != cudaSuccess;
        if (kind == 0)
            k_fp64_peak<0><<<grid, 256>>>(sink, outer, a, b);
        else
            k_fp64_peak<1><<<grid, 256>>>(sink, outer, a, b);
        failed = failed || cudaGetLastError() != cudaSuccess || cudaEventRecord(e1) != cudaSuccess ||
                 cudaEventSynchronize(e1) != cudaSuccess;
        float ms = 0.f;
        if (failed || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) {
            failed = true;
            break;
        }
        if (!(ms > 0.f)) continue;                   // a timer reading of zero would report an infinite rate
        const double inst = (double)grid * 256.0 * outer * PK_INNER * PK_CHAINS;
        const double tf = inst * (kind == 0 ? 2.0 : 1.0) / ((double)ms * 1e-3) / 1e12;
        if (std::isfinite(tf) && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (failed || cudaGetLastError() != cudaSuccess || !(best > 0.0) || !std::isfinite(best)) return NSC_ECUDA;
    *h_tflops = best;
    return NSC_OK;
}
