// nonlinear.cu -- host driver of the nonlinear term N(u, T) (DESIGN.md steps N1-N6;
// BASELINE.json north_star (a)): per radial chunk  k_zinv -> k_theta -> k_zfwd.
#include "nonlinear_kernels.cuh"

namespace nsc {

typedef int (*launch_fn)(const NlArgs&, cudaStream_t);
struct LenEntry {
    int n;
    launch_fn zinv, zfwd, theta;
};
#define NSC_LEN(N) {N, launch_zinv_##N, launch_zfwd_##N, launch_theta_##N}
static const LenEntry kLens[] = {NSC_LEN(12), NSC_LEN(24), NSC_LEN(48), NSC_LEN(96),
                                 NSC_LEN(192), NSC_LEN(384), NSC_LEN(768), NSC_LEN(1536)};
#undef NSC_LEN

static const LenEntry* find_len(int n) {
    for (const LenEntry& e : kLens)
        if (e.n == n) return &e;
    return nullptr;
}

bool fft_length_supported(int n) { return find_len(n) != nullptr; }

int launch_nonlinear(nsc_ctx* c, cd* const* f, cd* const* out) {
    const LenEntry* lz = find_len(c->Nz);
    const LenEntry* lt = find_len(c->Nt);
    if (!lz || !lt) return fail(c, NSC_EINVAL, "unsupported physical grid size");
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
    for (int j0 = 0; j0 < c->N_r; j0 += c->JC) {
        a.j0 = j0;
        a.nj = (c->N_r - j0 < c->JC) ? c->N_r - j0 : c->JC;
        a.tw = c->t.tw_z;
        prof_begin(c, NSC_K_ZINV);
        if (int e = lz->zinv(a, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_zinv launch");
        prof_end(c);
        a.tw = c->t.tw_t;
        prof_begin(c, NSC_K_THETA);
        if (int e = lt->theta(a, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_theta launch");
        prof_end(c);
        a.tw = c->t.tw_z;
        prof_begin(c, NSC_K_ZFWD);
        if (int e = lz->zfwd(a, c->stream)) return cuda_fail(c, (cudaError_t)e, "k_zfwd launch");
        prof_end(c);
    }
    return NSC_OK;
}

}  // namespace nsc
