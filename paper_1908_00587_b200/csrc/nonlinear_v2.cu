// nonlinear_v2.cu -- instantiation and launchers of the warp-transform kernels for the lengths 768 and 384
// (nonlinear_v2.cuh).  Persistent grids sized from the SM count (148 on a B200).
#include "nonlinear_v3.cuh"

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

int warp_na(int n, int modes) {
    if (n == 768 && modes <= 256) return 24;
    if (n == 384 && modes <= 128) return 12;
    if (n == 1536 && modes <= 512) return 48;
    return 0;
}

int warp_mtile(int na) { return na == 12 ? Z2Cfg<12>::MT : 4; }

static int launch_zinv3(const Nl2Args& a, cudaStream_t st) {
    if (int e = set_smem(k_zinv3, P3_SMEM_INV)) return e;
    int grid = sm_count();
    if (grid > a.nitems) grid = a.nitems;
    k_zinv3<<<grid, P3_THREADS, P3_SMEM_INV, st>>>(a);
    return (int)cudaGetLastError();
}

static int launch_zfwd3(const Nl2Args& a, cudaStream_t st) {
    if (int e = set_smem(k_zfwd3, P3_SMEM_FWD)) return e;
    int grid = sm_count();
    if (grid > a.nitems) grid = a.nitems;
    k_zfwd3<<<grid, P3_THREADS, P3_SMEM_FWD, st>>>(a);
    return (int)cudaGetLastError();
}

template <int NF, bool CFL> static int launch_theta3_c(const Nl2Args& a, cudaStream_t st) {
    const int nlines = a.b.nj * a.b.Nz;
    if (int e = set_smem(k_theta3<NF, CFL>, P3_SMEM_THETA)) return e;
    int grid = sm_count();
    if (grid > (nlines + P3_PAIRS - 1) / P3_PAIRS) grid = (nlines + P3_PAIRS - 1) / P3_PAIRS;
    k_theta3<NF, CFL><<<grid, P3_THREADS, P3_SMEM_THETA, st>>>(a);
    return (int)cudaGetLastError();
}
template <int NF> static int launch_theta3_t(const Nl2Args& a, cudaStream_t st) {
    return a.b.cfl ? launch_theta3_c<NF, true>(a, st) : launch_theta3_c<NF, false>(a, st);
}

template <int NA> static int launch_zinv2_t(const Nl2Args& a, cudaStream_t st) {
    using C = Z2Cfg<NA>;
    if (int e = set_smem(k_zinv2<NA>, C::SMEM_INV)) return e;
    int grid = 2 * sm_count();
    if (grid > a.nitems) grid = a.nitems;
    k_zinv2<NA><<<grid, Z2_THREADS, C::SMEM_INV, st>>>(a);
    return (int)cudaGetLastError();
}

template <int NA> static int launch_zfwd2_t(const Nl2Args& a, cudaStream_t st) {
    using C = Z2Cfg<NA>;
    if (int e = set_smem(k_zfwd2<NA>, C::SMEM_FWD)) return e;
    int grid = 2 * sm_count();
    if (grid > a.nitems) grid = a.nitems;
    k_zfwd2<NA><<<grid, Z2_THREADS, C::SMEM_FWD, st>>>(a);
    return (int)cudaGetLastError();
}

template <int NA, int NF, bool CFL> static int launch_theta2_c(const Nl2Args& a, cudaStream_t st) {
    using C = T2Cfg<NA>;
    const int nwarps = (a.b.nj * a.b.Nz + C::LPW - 1) / C::LPW;      // warps' worth of point-lines
    if (int e = set_smem(k_theta2<NA, NF, CFL>, C::SMEM)) return e;
    int grid = sm_count();
    if (grid > (nwarps + T2_WARPS - 1) / T2_WARPS) grid = (nwarps + T2_WARPS - 1) / T2_WARPS;
    k_theta2<NA, NF, CFL><<<grid, T2_WARPS * 32, C::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
template <int NA, int NF> static int launch_theta2_t(const Nl2Args& a, cudaStream_t st) {
    return a.b.cfl ? launch_theta2_c<NA, NF, true>(a, st) : launch_theta2_c<NA, NF, false>(a, st);
}

int launch_zinv2(int na, const Nl2Args& a, cudaStream_t st) {
    if (na == 48) return launch_zinv3(a, st);
    return na == 24 ? launch_zinv2_t<24>(a, st) : launch_zinv2_t<12>(a, st);
}

int launch_zfwd2(int na, const Nl2Args& a, cudaStream_t st) {
    if (na == 48) return launch_zfwd3(a, st);
    return na == 24 ? launch_zfwd2_t<24>(a, st) : launch_zfwd2_t<12>(a, st);
}

int launch_theta2(int na, const Nl2Args& a, cudaStream_t st) {
    if (na == 48) return a.b.nf == 3 ? launch_theta3_t<3>(a, st) : launch_theta3_t<4>(a, st);
    if (na == 24) return a.b.nf == 3 ? launch_theta2_t<24, 3>(a, st) : launch_theta2_t<24, 4>(a, st);
    return a.b.nf == 3 ? launch_theta2_t<12, 3>(a, st) : launch_theta2_t<12, 4>(a, st);
}

}  // namespace nsc
