// nonlinear_inst.cu -- instantiates the transform kernels for ONE line length, selected with
// -DNSC_FFT_N=<12|24|48|96|192>; the build compiles this file once per length
// (in parallel) and nonlinear.cu dispatches on the run-time lengths N_theta, N_z.
#include "nonlinear_kernels.cuh"

#ifndef NSC_FFT_N
#error "compile with -DNSC_FFT_N=<length>"
#endif

namespace nsc {

#define NSC_CAT2(a, b) a##b
#define NSC_CAT(a, b) NSC_CAT2(a, b)
constexpr int LEN = NSC_FFT_N;

// raises the dynamic shared-memory limit of kernel k (a per-device attribute: set on every launch)
template <int ID, class Kern> static int prep(Kern k, size_t smem) {
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    return e == cudaSuccess ? 0 : (int)e;
}

int NSC_CAT(launch_zinv_, NSC_FFT_N)(const NlArgs& a, cudaStream_t st) {
    using C = ZCfg<LEN>;
    if (int e = prep<0>(k_zinv<LEN>, C::SMEM)) return e;
    const int nlines = a.nj * a.M1;
    dim3 grid((nlines + C::LPC - 1) / C::LPC, a.nf);
    k_zinv<LEN><<<grid, C::THREADS, C::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}

int NSC_CAT(launch_zfwd_, NSC_FFT_N)(const NlArgs& a, cudaStream_t st) {
    using C = ZCfg<LEN>;
    if (int e = prep<1>(k_zfwd<LEN>, C::SMEM)) return e;
    const int nlines = a.nj * a.M1;
    dim3 grid((nlines + C::LPC - 1) / C::LPC, a.nf);
    k_zfwd<LEN><<<grid, C::THREADS, C::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}

int NSC_CAT(launch_theta_, NSC_FFT_N)(const NlArgs& a, cudaStream_t st) {
    using C = TCfg<LEN>;
    const int nlines = a.nj * a.Nz;
    dim3 grid((nlines + C::LPC - 1) / C::LPC);
    if (a.nf == 3) {
        if (int e = prep<2>(k_theta<LEN, 3>, C::SMEM)) return e;
        k_theta<LEN, 3><<<grid, C::THREADS, C::SMEM, st>>>(a);
    } else {
        if (int e = prep<3>(k_theta<LEN, 4>, C::SMEM)) return e;
        k_theta<LEN, 4><<<grid, C::THREADS, C::SMEM, st>>>(a);
    }
    return (int)cudaGetLastError();
}

}  // namespace nsc
