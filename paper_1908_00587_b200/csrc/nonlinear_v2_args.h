// nonlinear_v2_args.h -- argument blocks and host-side launchers of the warp-transform kernels for the line
// lengths 768 and 384 (nonlinear_v2.cuh), shared by the driver (nonlinear.cu) and the kernels' translation unit.
#pragma once
#include "nonlinear_kernels.cuh"

namespace nsc {

struct DrArgs {
    const cd* f[MAXF];
    cd* out[MAXF];
    const double* D1;
    int N_r;
    size_t plane;          // stride between radial levels (complex elements)
    size_t ncols;          // columns of one field per level (<= plane)
};

struct Nl2Args {
    NlArgs b;              // the generic argument block (fields, work arrays, sizes)
    const cd* dr[MAXF];    // radial derivatives of the input fields, spectral layout
    const cd* tw_z;        // [24][33] twiddle matrix of fft_warp.cuh for the z length (plan.cu)
    const cd* tw_t;        // ... for the theta length
    const cd* tw_cz;       // [768] exp(-2 pi i k / 1536): combine twiddles of the warp-pair transform (length 1536), z
    const cd* tw_ct;       // ... theta
    double alpha;          // axial base wavenumber
    double ktheta0;        // azimuthal base wavenumber
    int nitems;            // work items of the launch
};

// host-side launchers (nonlinear_v2.cu)
int launch_dr(const DrArgs& a, int nf, cudaStream_t st);
// na = 24 (length 768), 12 (length 384) or 48 (length 1536 = 2 x 768 on warp pairs, nonlinear_v3.cuh);
// warp_na(n, modes): the na of length n if the warp kernels serve it, else 0
int warp_na(int n, int modes);
int warp_mtile(int na);    // m-lines per work item of the z kernels
int launch_zinv2(int na, const Nl2Args& a, cudaStream_t st);
int launch_zfwd2(int na, const Nl2Args& a, cudaStream_t st);
int launch_theta2(int na, const Nl2Args& a, cudaStream_t st);

}  // namespace nsc
