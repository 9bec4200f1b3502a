// regrid.cu -- restart on another resolution ("At every restart, the spatial
// resolution can be changed using an automated interpolation and mode padding functionality"; reading R18):
// the state of one context is carried onto the radial grid and the mode set of another.
//   radial   degree-8 Lagrange interpolation on the nine source nodes around the source node nearest to the target
//            node (window start clamp(c - 4, 0, N_src - 9), the placement rule of the finite-difference stencils, R3);
//            weights from Fornberg's recursion in extended precision (order-0 row)
//   modes    coefficients of modes the source does not hold are zero (padding), modes the target does not hold are
//            dropped (truncation)
#include <cmath>
#include <vector>
#include "nsc_internal.h"

namespace nsc {

typedef long double ld;

// order-0 weights of the interpolant through x[0..n-1] at z (Fornberg 1988, derivative order 0 only)
static void interp_weights(ld z, const ld* x, int n, ld* w) {
    ld c1 = 1, c4 = x[0] - z;
    for (int i = 0; i < n; ++i) w[i] = 0;
    w[0] = 1;
    for (int i = 1; i < n; ++i) {
        ld c2 = 1, c5 = c4;
        c4 = x[i] - z;
        for (int j = 0; j < i; ++j) {
            const ld c3 = x[i] - x[j];
            c2 *= c3;
            if (j == i - 1) w[i] = -c1 * c5 * w[i - 1] / c2;
            w[j] = c4 * w[j] / c3;
        }
        c1 = c2;
    }
}

struct RegridArgs {
    const cd* src[5];
    cd* dst[5];
    const double* w;      // [N_dst][9]
    const int* s0;        // [N_dst] first source node of the window
    int nfld;
    int N_dst, M1d, NKd, Kd;
    int M1s, NKs, Ks;
};

// one thread per target coefficient (j, m, kk) and field
__global__ void __launch_bounds__(256) k_regrid(RegridArgs a) {
    const size_t plane_d = (size_t)a.M1d * a.NKd, plane_s = (size_t)a.M1s * a.NKs;
    const size_t total = (size_t)a.N_dst * plane_d;
    const int f = blockIdx.y;
    const cd* src = f == 0 ? a.src[0] : f == 1 ? a.src[1] : f == 2 ? a.src[2] : f == 3 ? a.src[3] : a.src[4];
    cd* dst = f == 0 ? a.dst[0] : f == 1 ? a.dst[1] : f == 2 ? a.dst[2] : f == 3 ? a.dst[3] : a.dst[4];
    if (!dst) return;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(i / plane_d);
        const int e = (int)(i % plane_d);
        const int m = e / a.NKd, k = e % a.NKd - a.Kd;
        cd v = mk(0.0, 0.0);
        if (src && m < a.M1s && k >= -a.Ks && k <= a.Ks) {
            const cd* col = src + (size_t)a.s0[j] * plane_s + (size_t)m * a.NKs + (size_t)(k + a.Ks);
            const double* w = a.w + j * NPT;
#pragma unroll
            for (int l = 0; l < NPT; ++l) {
                const cd s = col[(size_t)l * plane_s];
                v.x = fma(w[l], s.x, v.x);
                v.y = fma(w[l], s.y, v.y);
            }
        }
        dst[i] = v;
    }
}

}  // namespace nsc

using namespace nsc;

extern "C" int nsc_regrid(nsc_ctx* d, nsc_ctx* s) {
    if (!d || !s) return NSC_EINVAL;
    if (d == s) return fail(d, NSC_EINVAL, "nsc_regrid: source and target must be two contexts (the kernel reads the source rows while it writes the target)");
    if (d->dev != s->dev)
        return fail(d, NSC_EINVAL, "nsc_regrid: the two contexts live on different devices (" + std::to_string(s->dev) + " and " +
                                       std::to_string(d->dev) + ")");
    if (!s->have_state) return fail(d, NSC_ESTATE, "nsc_regrid: the source context has no state");
    if (d->p.eta != s->p.eta || d->p.alpha != s->p.alpha || d->p.k_theta0 != s->p.k_theta0)
        return fail(d, NSC_EINVAL, "nsc_regrid: eta, alpha and k_theta0 of the two contexts must agree (same domain, same wavenumbers)");
    if (d->heated && !s->heated) return fail(d, NSC_EINVAL, "nsc_regrid: the target has a temperature field, the source has none");
    // interpolation table of the target nodes on the source grid
    const int Nd = d->N_r, Ns = s->N_r;
    std::vector<ld> xs(Ns);
    for (int j = 0; j < Ns; ++j) xs[j] = (ld)s->r[j];
    std::vector<double> w((size_t)Nd * NPT);
    std::vector<int> s0(Nd);
    for (int j = 0; j < Nd; ++j) {
        const double r = d->r[j];
        int c = 0;                                         // nearest source node (the lower one on a tie)
        for (int i = 1; i < Ns; ++i)
            if (fabs(s->r[i] - r) < fabs(s->r[c] - r)) c = i;
        int st = c - NPT / 2;
        if (st < 0) st = 0;
        if (st > Ns - NPT) st = Ns - NPT;
        s0[j] = st;
        ld wl[NPT];
        interp_weights((ld)r, &xs[st], NPT, wl);
        for (int l = 0; l < NPT; ++l) w[(size_t)j * NPT + l] = (double)wl[l];
    }
    double* d_w = nullptr;
    int* d_s0 = nullptr;
    DeviceGuard on_device(d->dev);                         // the tables and the launch belong to the contexts' device
    if (!on_device.ok()) return fail(d, NSC_ECUDA, "nsc_regrid: cannot make the contexts' device current");
    NSC_CUDA(d, cudaStreamSynchronize(s->stream));         // the source state is complete
    NSC_CUDA(d, cudaMalloc(&d_w, sizeof(double) * w.size()));
    cudaError_t e = cudaMalloc(&d_s0, sizeof(int) * s0.size());
    if (e != cudaSuccess) {
        cudaFree(d_w);
        return cuda_fail(d, e, "cudaMalloc(regrid table)");
    }
    cudaMemcpyAsync(d_w, w.data(), sizeof(double) * w.size(), cudaMemcpyHostToDevice, d->stream);
    cudaMemcpyAsync(d_s0, s0.data(), sizeof(int) * s0.size(), cudaMemcpyHostToDevice, d->stream);
    RegridArgs a{};
    for (int f = 0; f < 5; ++f) {
        a.src[f] = s->state[f];
        a.dst[f] = d->state[f];                            // null for T without temperature
    }
    a.w = d_w;
    a.s0 = d_s0;
    a.N_dst = Nd;
    a.M1d = d->M1;
    a.NKd = d->NK;
    a.Kd = d->K;
    a.M1s = s->M1;
    a.NKs = s->NK;
    a.Ks = s->K;
    prof_begin(d, NSC_K_DR);
    k_regrid<<<dim3(148 * 4, 5), 256, 0, d->stream>>>(a);
    prof_end(d);
    e = cudaGetLastError();
    cudaError_t e2 = cudaStreamSynchronize(d->stream);     // the tables are freed below
    cudaFree(d_w);
    cudaFree(d_s0);
    if (e != cudaSuccess) return cuda_fail(d, e, "k_regrid launch");
    if (e2 != cudaSuccess) return cuda_fail(d, e2, "k_regrid");
    int rc = launch_radial_derivative(d, d->state[4], d->DP);      // D1 p of the new state (linear stage)
    if (rc) return rc;
    d->have_state = true;
    return NSC_OK;
}
