// nonlinear_v2_args.h -- argument blocks and host-side launchers of the length-768 transform
// kernels (nonlinear_v2.cuh), shared by the driver (nonlinear.cu) and the kernels' translation unit.
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
    const cd* tw768;       // [24][33] twiddle matrix of fft768.cuh
    double alpha;          // axial base wavenumber
    double ktheta0;        // azimuthal base wavenumber
    int nitems;            // work items of the launch
};

// host-side launchers (nonlinear_v2.cu)
int launch_dr(const DrArgs& a, int nf, cudaStream_t st);
int launch_zinv2(const Nl2Args& a, cudaStream_t st);
int launch_zfwd2(const Nl2Args& a, cudaStream_t st);
int launch_theta2(const Nl2Args& a, bool tmem, cudaStream_t st);

}  // namespace nsc
