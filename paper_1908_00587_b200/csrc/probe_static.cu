// probe_static.cu -- nsc_probe_static: the point probe of nsc_probe (Fig. 3b: a velocity
// component recorded at a fixed location) for callers that may not allocate device memory.
//
// Who that is.  A probe is usually read by something that watches a run rather than owns it: a monitoring
// hook called once per time step, or a host program that keeps the flow state in buffers of its own (torch
// tensors, another solver's arrays) and only wants the library's diagnostic.  Such a caller often cannot go
// through cudaMalloc:
//   - the device is full on purpose.  The N_r = 512 configuration takes 148 of the 180 GB, and host frameworks
//     reserve what is left for their own pools, so a late cudaMalloc fails or takes memory the run counted on;
//   - cudaMalloc and cudaFree stall the whole device while they run, which a once-per-step call placed
//     between the solver's kernels would turn into a stall of every step;
//   - the call sits in a region where the host program forbids runtime calls that allocate.
// nsc_probe needs a context (whose creation allocates the state, the work arrays and a small accumulator).
// This entry point needs neither: inputs and the output are the caller's, and the only other global memory the
// kernel touches -- one partial sum per thread block and the arrival counter of the blocks -- lives in the
// file-scope array g_probe_scratch below, which is part of the loaded library image on every device
// (NSC_PROBE_STATIC_SCRATCH_BYTES, 4.5 KB, held from the moment a GPU loads this module until the process exits).
//
// Two things follow from sharing one array between all calls.  It still holds whatever the previous call left
// there, so every call first clears the part that has to start at zero (the arrival counter) on the caller's
// stream.  And two calls that are in flight on one GPU at the same time -- different streams, or different
// host threads -- write the same partial sums and the same counter: they race, and both results are garbage.
// Calls on one stream, or ordered by events, are safe.
//
// Host code cannot use the name g_probe_scratch as a pointer: in host code that name denotes a host-side
// shadow object of the symbol, not memory on the GPU.  The device address is obtained once per device with
// cudaGetSymbolAddress (scratch_address below) and that pointer is what the kernel receives.
#include <cmath>
#include <mutex>
#include <string>
#include "nsc_internal.h"

namespace nsc {

constexpr int PS_THREADS = 256;
constexpr int PS_PER_THREAD = 4;                              // modes per thread
constexpr int PS_PER_BLOCK = PS_THREADS * PS_PER_THREAD;      // 1024 modes per block
constexpr int PS_MAX_M = 512, PS_MAX_K = 512;                 // the limits of nsc_create (nsc.h)
constexpr long long PS_MAX_MODES = (long long)(PS_MAX_M + 1) * (2 * PS_MAX_K + 1);              // 525 825
constexpr int PS_MAX_BLOCKS = (int)((PS_MAX_MODES + PS_PER_BLOCK - 1) / PS_PER_BLOCK);          // 514
constexpr int PS_HEADER = 32;                                 // doubles; word 0 of it is the arrival counter
constexpr int PS_SCRATCH_DOUBLES = PS_HEADER + 544;           // 576 doubles = 4608 bytes
static_assert(PS_MAX_BLOCKS <= PS_SCRATCH_DOUBLES - PS_HEADER, "scratch too small for the largest mode set");
static_assert(PS_SCRATCH_DOUBLES * sizeof(double) == NSC_PROBE_STATIC_SCRATCH_BYTES, "nsc.h states another size");

// [0, 32): header, the first 4 bytes are the arrival counter; [32, 32 + blocks): one partial sum per block.
static __device__ __align__(256) double g_probe_scratch[PS_SCRATCH_DOUBLES];

// Same sum as k_probe (linear.cu): Re sum_k f(0,k) e^{i kappa z} + 2 Re sum_{m>=1,k} f(m,k) e^{i (n theta + kappa z)}
// with n = m k_theta0, kappa = (kk - K_z) alpha, but summed in a fixed order: every block leaves its partial in
// scratch, the block that arrives last adds the partials in index order and writes the caller's output.
// `scratch` is the device address of g_probe_scratch.
__global__ void __launch_bounds__(PS_THREADS) k_probe_static(const cd* __restrict__ fj, int M1, int NK, int K_z,
                                                             double k_theta0, double alpha, double theta, double z,
                                                             double* scratch, double* __restrict__ out) {
    __shared__ double sh[PS_THREADS / 32];
    __shared__ bool last;
    const int n = M1 * NK;
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PS_PER_THREAD; ++i) {
        const int e = blockIdx.x * PS_PER_BLOCK + i * PS_THREADS + threadIdx.x;
        if (e < n) {
            const int m = e / NK, kk = e - m * NK;
            double sn, cs;
            sincos((double)m * k_theta0 * theta + (double)(kk - K_z) * alpha * z, &sn, &cs);
            const cd v = fj[e];
            const double re = v.x * cs - v.y * sn;
            s += (m == 0) ? re : 2.0 * re;
        }
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (l == 0) sh[w] = s;
    __syncthreads();
    unsigned int* arrived = reinterpret_cast<unsigned int*>(scratch);
    double* partial = scratch + PS_HEADER;
    if (threadIdx.x == 0) {
        double S = 0.0;
        for (int i = 0; i < PS_THREADS / 32; ++i) S += sh[i];
        partial[blockIdx.x] = S;
        __threadfence();                                      // the partial is visible before the arrival is counted
        last = atomicAdd(arrived, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();                                          // the other blocks' partials, not a stale cache line
    double t = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += PS_THREADS) t += __ldcg(partial + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    if (l == 0) sh[w] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double S = 0.0;
        for (int i = 0; i < PS_THREADS / 32; ++i) S += sh[i];
        *out = S;
    }
}

// Device address of g_probe_scratch on the current device, asked for once per device and kept.
constexpr int PS_MAX_DEVICES = 64;
static std::mutex g_ps_mutex;
static double* g_ps_addr[PS_MAX_DEVICES] = {};

static int scratch_address(double** addr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "nsc_probe_static: cudaGetDevice");
    if (dev < 0 || dev >= PS_MAX_DEVICES)
        return fail(nullptr, NSC_EINVAL, "nsc_probe_static: device ordinal " + std::to_string(dev) + " is beyond the " +
                                             std::to_string(PS_MAX_DEVICES) + " devices this entry point keeps track of");
    std::lock_guard<std::mutex> lock(g_ps_mutex);
    if (!g_ps_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_probe_scratch);        // of the copy on the device that is current now
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "nsc_probe_static: cudaGetSymbolAddress(g_probe_scratch)");
        if (!p) return fail(nullptr, NSC_ECUDA, "nsc_probe_static: cudaGetSymbolAddress returned a null address");
        g_ps_addr[dev] = static_cast<double*>(p);
    }
    *addr = g_ps_addr[dev];
    return NSC_OK;
}

}  // namespace nsc

using namespace nsc;

extern "C" int nsc_probe_static(const void* d_field, int N_r, int M_theta, int K_z, int k_theta0, double alpha, int j,
                                double theta, double z, double* d_value, void* cuda_stream) {
    // every argument check comes before the first CUDA call
    if (!d_field || !d_value) return fail(nullptr, NSC_EINVAL, "nsc_probe_static: d_field and d_value must not be NULL");
    if (M_theta < 1 || K_z < 1 || N_r < 1)
        return fail(nullptr, NSC_EINVAL, "nsc_probe_static: N_r, M_theta and K_z must be >= 1");
    if (M_theta > PS_MAX_M || K_z > PS_MAX_K)
        return fail(nullptr, NSC_EINVAL,
                    "nsc_probe_static: M_theta = " + std::to_string(M_theta) + ", K_z = " + std::to_string(K_z) +
                        " exceed the maximum M_theta <= 512, K_z <= 512 (525825 modes) that the fixed scratch array of " +
                        std::to_string(NSC_PROBE_STATIC_SCRATCH_BYTES) + " bytes is laid out for");
    if (j < 0 || j >= N_r) return fail(nullptr, NSC_EINVAL, "nsc_probe_static: radial node j outside 0 <= j < N_r");
    if (k_theta0 < 1 || !(alpha > 0.0) || !std::isfinite(alpha) || !std::isfinite(theta) || !std::isfinite(z))
        return fail(nullptr, NSC_EINVAL, "nsc_probe_static: k_theta0 >= 1, alpha > 0 and finite theta, z are required");

    double* scratch = nullptr;
    int rc = scratch_address(&scratch);
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int M1 = M_theta + 1, NK = 2 * K_z + 1;
    const int n = M1 * NK;
    const int blocks = (n + PS_PER_BLOCK - 1) / PS_PER_BLOCK;
    // the counter still holds the previous call's count (or that of a call that never finished): back to zero
    cudaError_t e = cudaMemsetAsync(scratch, 0, PS_HEADER * sizeof(double), stream);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "nsc_probe_static: cudaMemsetAsync(arrival counter)");
    const cd* fj = static_cast<const cd*>(d_field) + (size_t)j * (size_t)n;
    k_probe_static<<<blocks, PS_THREADS, 0, stream>>>(fj, M1, NK, K_z, (double)k_theta0, alpha, theta, z, scratch,
                                                        d_value);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "nsc_probe_static: kernel launch");
    return NSC_OK;
}
