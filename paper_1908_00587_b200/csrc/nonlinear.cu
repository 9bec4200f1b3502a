// nonlinear.cu -- host driver of the nonlinear term N(u, T) (DESIGN.md steps N1-N6;
// BASELINE.json north_star (a)): per radial chunk  k_zinv -> k_theta -> k_zfwd.
#include "nonlinear_v2_args.h"

namespace nsc {

typedef int (*launch_fn)(const NlArgs&, cudaStream_t);
struct LenEntry {
    int n;
    launch_fn zinv, zfwd, theta;
};
#define NSC_LEN(N) {N, launch_zinv_##N, launch_zfwd_##N, launch_theta_##N}
// generic three-pass kernels (nonlinear_kernels.cuh): the short lengths; 384, 768 and 1536 run the warp-transform
// kernels of nonlinear_v2.cuh / nonlinear_v3.cuh
static const LenEntry kLens[] = {NSC_LEN(12), NSC_LEN(24), NSC_LEN(48), NSC_LEN(96), NSC_LEN(192)};
#undef NSC_LEN

static const LenEntry* find_len(int n) {
    for (const LenEntry& e : kLens)
        if (e.n == n) return &e;
    return nullptr;
}

bool fft_length_supported(int n) { return find_len(n) != nullptr || warp_na(n, 1) != 0; }

int launch_radial_derivative(nsc_ctx* c, const cd* f, cd* out) {
    DrArgs d{};
    d.f[0] = f;
    d.out[0] = out;
    d.D1 = c->t.D1;
    d.N_r = c->N_r;
    d.plane = (size_t)c->M1 * c->NK;
    d.ncols = d.plane;
    prof_begin(c, NSC_K_DR);
    if (int e = launch_dr(d, 1, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_dr launch");
    prof_end(c);
    return NSC_OK;
}

int launch_nonlinear(nsc_ctx* c, cd* const* f, cd* const* out) {
    const LenEntry* lz = find_len(c->Nz);
    const LenEntry* lt = find_len(c->Nt);
    if ((!lz && !c->z_na) || (!lt && !c->t_na)) return fail(c, NSC_EINVAL, "unsupported physical grid size");
    NlArgs a{};
    for (int i = 0; i < c->nf; ++i) {
        a.f[i] = f[i];
        a.out[i] = out[i];
    }
    a.zbuf = c->zbuf;
    a.tbuf = c->tbuf;
    a.D1 = c->t.D1;
    a.s0 = c->t.s0;
    a.rinv = c->t.rinv;
    a.nm = c->t.nm;
    a.kap = c->t.kap;
    a.N_r = c->N_r;
    a.M1 = c->M1;
    a.NK = c->NK;
    a.K = c->K;
    a.M = c->M;
    a.MP = c->MP;
    a.JC = c->JC;
    a.Nz = c->Nz;
    a.nf = c->nf;
    a.scale = 1.0 / ((double)c->Nt * (double)c->Nz);
    a.buoy = c->heated ? c->p.Ra / c->p.Pr : 0.0;
    a.cfl = c->want_cfl ? c->cfl_max : nullptr;
    Nl2Args a2{};
    a2.tw_z = c->t.tw_wz;
    a2.tw_t = c->t.tw_wt;
    a2.tw_cz = c->t.tw_c1536;
    a2.tw_ct = c->t.tw_c1536;
    a2.alpha = c->p.alpha;
    a2.ktheta0 = (double)c->p.k_theta0;
    // N1, radial derivative.  One radial chunk (JC = N_r): D1 is applied to the z-transformed fields inside the
    // work array after k_zinv (two transforms per line instead of three; D1 commutes with the z transform).
    // Several chunks: D1 f of every spectral field once per evaluation, transformed as a third line.
    const bool dr_after_z = c->z_na && c->JC == c->N_r;
    if (c->z_na && !dr_after_z) {
        DrArgs d{};
        for (int i = 0; i < c->nf; ++i) {
            d.f[i] = f[i];
            d.out[i] = c->DR[i];
            a2.dr[i] = c->DR[i];
        }
        d.D1 = c->t.D1;
        d.N_r = c->N_r;
        d.plane = (size_t)c->M1 * c->NK;
        d.ncols = d.plane;
        prof_begin(c, NSC_K_DR);
        if (int e = launch_dr(d, c->nf, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_dr launch");
        prof_end(c);
    }
    const size_t rowZ = (size_t)3 * c->nf * c->Nz * c->MP;      // one radial level of zbuf
    for (int j0 = c->wj0; j0 < c->wj1; j0 += c->JC) {
        a.j0 = j0;
        a.nj = (c->wj1 - j0 < c->JC) ? c->wj1 - j0 : c->JC;
        a.zbuf = c->zbuf;
        if (dr_after_z) {
            // the work array holds every level at its own row; D1 at level j reads the z-transformed fields at the
            // nine rows s0(j) .. s0(j) + 8 with s0(j) = clamp(j - 4, 0, N_r - 9): four levels beyond the window on
            // either side, and all nine rows next to a wall even when the window is shorter than five levels
            const int smax = c->N_r - NPT, jl = j0 + a.nj - 1;
            const int h0 = j0 - NPT / 2 < 0 ? 0 : (j0 - NPT / 2 > smax ? smax : j0 - NPT / 2);
            const int h1 = (jl - NPT / 2 < 0 ? 0 : (jl - NPT / 2 > smax ? smax : jl - NPT / 2)) + NPT;
            a.j0 = h0;
            a.nj = h1 - h0;
            a.zbuf = c->zbuf + (size_t)h0 * rowZ;
        }
        a.tw = c->t.tw_z;
        prof_begin(c, NSC_K_ZINV);
        if (c->z_na) {
            a2.b = a;
            a2.nitems = c->nf * a.nj * (c->MP / warp_mtile(c->z_na));
            if (int e = launch_zinv2(c->z_na, a2, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_zinv2 launch");
        } else if (int e = lz->zinv(a, c->stream)) {
            return cuda_fail(c, (cudaError_t)e, "k_zinv launch");
        }
        prof_end(c);
        if (dr_after_z) {
            a.j0 = j0;
            a.nj = (c->wj1 - j0 < c->JC) ? c->wj1 - j0 : c->JC;
            a.zbuf = c->zbuf + (size_t)j0 * rowZ;
        }
        if (dr_after_z) {
            DrArgs d{};
            const size_t qstride = (size_t)c->Nz * c->MP;
            for (int i = 0; i < c->nf; ++i) {
                d.f[i] = c->zbuf + (size_t)(3 * i) * qstride;
                d.out[i] = c->zbuf + (size_t)(3 * i + 2) * qstride;
            }
            d.D1 = c->t.D1;
            d.N_r = c->N_r;
            d.plane = (size_t)3 * c->nf * qstride;
            d.ncols = qstride;
            prof_begin(c, NSC_K_DR);
            if (int e = launch_dr(d, c->nf, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_dr launch");
            prof_end(c);
        }
        a.tw = c->t.tw_t;
        prof_begin(c, NSC_K_THETA);
        if (c->t_na) {
            a2.b = a;
            a2.nitems = a.nj * a.Nz;
            if (int e = launch_theta2(c->t_na, a2, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_theta2 launch");
        } else if (int e = lt->theta(a, c->stream)) {
            return cuda_fail(c, (cudaError_t)e, "k_theta launch");
        }
        prof_end(c);
        a.tw = c->t.tw_z;
        prof_begin(c, NSC_K_ZFWD);
        if (c->z_na) {
            a2.b = a;
            a2.nitems = c->nf * a.nj * (c->MP / warp_mtile(c->z_na));
            if (int e = launch_zfwd2(c->z_na, a2, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_zfwd2 launch");
        } else if (int e = lz->zfwd(a, c->stream)) {
            return cuda_fail(c, (cudaError_t)e, "k_zfwd launch");
        }
        prof_end(c);
    }
    return NSC_OK;
}

}  // namespace nsc
