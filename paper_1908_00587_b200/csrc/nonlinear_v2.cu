// nonlinear_v2.cu -- instantiation and launchers of the length-768 transform kernels
// (nonlinear_v2.cuh).  Persistent grids sized from the SM count (148 on a B200).
#include "nonlinear_v2.cuh"

namespace nsc {

static int sm_count() {
    static int n = 0;
    if (!n) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    }
    return n;
}

// the attribute is per device: set on every launch (a few microseconds) rather than cached per process
template <class Kern> static int set_smem(Kern k, size_t smem) {
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    return e == cudaSuccess ? 0 : (int)e;
}

int launch_dr(const DrArgs& a, int nf, cudaStream_t st) {
    dim3 grid((unsigned)((a.ncols + DR_TB - 1) / DR_TB), nf);
    k_dr<<<grid, DR_TB, 0, st>>>(a);
    return (int)cudaGetLastError();
}

int launch_zinv2(const Nl2Args& a, cudaStream_t st) {
    if (int e = set_smem(k_zinv2, Z2_SMEM_INV)) return e;
    int grid = 2 * sm_count();
    if (grid > a.nitems) grid = a.nitems;
    k_zinv2<<<grid, Z2_THREADS, Z2_SMEM_INV, st>>>(a);
    return (int)cudaGetLastError();
}

int launch_zfwd2(const Nl2Args& a, cudaStream_t st) {
    if (int e = set_smem(k_zfwd2, Z2_SMEM_FWD)) return e;
    int grid = 2 * sm_count();
    if (grid > a.nitems) grid = a.nitems;
    k_zfwd2<<<grid, Z2_THREADS, Z2_SMEM_FWD, st>>>(a);
    return (int)cudaGetLastError();
}

int launch_theta2(const Nl2Args& a, bool tmem, cudaStream_t st) {
    const int nlines = a.b.nj * a.b.Nz;
    if (tmem) {
        using C = T2Cfg<true>;
            if (int e = set_smem(k_theta2<true>, C::SMEM)) return e;
        int grid = sm_count();
        if (grid > (nlines + C::WARPS - 1) / C::WARPS) grid = (nlines + C::WARPS - 1) / C::WARPS;
        k_theta2<true><<<grid, C::WARPS * 32, C::SMEM, st>>>(a);
    } else {
        using C = T2Cfg<false>;
            if (int e = set_smem(k_theta2<false>, C::SMEM)) return e;
        int grid = sm_count();
        if (grid > (nlines + C::WARPS - 1) / C::WARPS) grid = (nlines + C::WARPS - 1) / C::WARPS;
        k_theta2<false><<<grid, C::WARPS * 32, C::SMEM, st>>>(a);
    }
    return (int)cudaGetLastError();
}

}  // namespace nsc
