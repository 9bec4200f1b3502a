// plan.cu -- host-side plan of a context: radial grid, finite-difference weight tables,
// operator band tables, band envelopes, wavenumbers and twiddle tables, all evaluated in
// extended precision (x86 long double) and rounded once, then uploaded.
//
// PAPER.md:42  "High-order finite differences (FD) are used in r ... The user can select the
//               distribution of radial grid points at runtime and the stencil-length of the FD
//               scheme is specified at compile time with a default of nine points."
// Readings R1-R4 of DESIGN.md fix the rest (gap = 1, grid families, shifted wall stencils).
// The weights come from Fornberg's recursion (Math. Comp. 51, 1988), a different route from
// the oracle's closed-form Lagrange derivatives.
#include <cmath>
#include <cstring>
#include "nsc_internal.h"
#include "fft_warp.cuh"

namespace nsc {

typedef long double ld;

static ld pi_ld() { return 4 * atanl((ld)1); }

// Weights c[i][k] of the k-th derivative (k = 0..2) at z on nodes x[0..n-1] (Fornberg 1988).
static void fornberg(ld z, const ld* x, int n, ld c[][3]) {
    for (int i = 0; i < n; ++i) c[i][0] = c[i][1] = c[i][2] = 0;
    ld c1 = 1, c4 = x[0] - z;
    c[0][0] = 1;
    for (int i = 1; i < n; ++i) {
        int mn = i < 2 ? i : 2;
        ld c2 = 1, c5 = c4;
        c4 = x[i] - z;
        for (int j = 0; j < i; ++j) {
            ld c3 = x[i] - x[j];
            c2 *= c3;
            if (j == i - 1) {
                for (int k = mn; k >= 1; --k) c[i][k] = c1 * (k * c[i - 1][k - 1] - c5 * c[i - 1][k]) / c2;
                c[i][0] = -c1 * c5 * c[i - 1][0] / c2;
            }
            for (int k = mn; k >= 1; --k) c[j][k] = (c4 * c[j][k] - k * c[j][k - 1]) / c3;
            c[j][0] = c4 * c[j][0] / c3;
        }
        c1 = c2;
    }
}

template <class T> static int upload(nsc_ctx* c, T** dst, const std::vector<T>& src) {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, src.size() * sizeof(T));
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMalloc(table)");
    c->allocs.push_back(p);
    c->dev_bytes += (long long)(src.size() * sizeof(T));
    e = cudaMemcpy(p, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemcpy(table)");
    *dst = (T*)p;
    return NSC_OK;
}

static int finish_shape(nsc_ctx* c, BandShape& s, int wmax) {
    const int N = c->N_r;
    for (int j = 1; j < N; ++j)
        if (s.h_hi[j] < s.h_hi[j - 1]) s.h_hi[j] = s.h_hi[j - 1];
    for (int j = N - 2; j >= 0; --j)
        if (s.h_lo[j] > s.h_lo[j + 1]) s.h_lo[j] = s.h_lo[j + 1];
    s.h_offL.assign(N, 0);
    s.h_offU.assign(N, 0);
    size_t oL = 0, oU = 0;
    for (int j = 0; j < N; ++j) {
        int nl = j - s.h_lo[j], nu = s.h_hi[j] - j;
        if (nl < 0 || nu < 0 || nl > wmax || nu > wmax) return fail(c, NSC_EINVAL, "band envelope exceeds the solver window");
        s.h_offL[j] = (int)oL;
        s.h_offU[j] = (int)oU;
        oL += nl;
        oU += nu + 1;
    }
    s.nL = oL;
    s.nU = oU;
    int rc;
    if ((rc = upload(c, &s.lo, s.h_lo))) return rc;
    if ((rc = upload(c, &s.hi, s.h_hi))) return rc;
    if ((rc = upload(c, &s.offL, s.h_offL))) return rc;
    if ((rc = upload(c, &s.offU, s.h_offU))) return rc;
    return NSC_OK;
}

int build_plan(nsc_ctx* c) {
    const int N = c->N_r;
    const nsc_params& p = c->p;
    // ---- O1 radial grid (R1: gap 1, r_i = eta / (1 - eta); R2: families)
    std::vector<ld> r(N);
    ld eta = (ld)p.eta, r_i = eta / (1 - eta);
    for (int j = 0; j < N; ++j) {
        if (p.radial_grid == 0)
            r[j] = r_i + (ld)j / (N - 1);
        else
            r[j] = r_i + (1 - cosl(pi_ld() * j / (N - 1))) / 2;
    }
    c->r.resize(N);
    for (int j = 0; j < N; ++j) c->r[j] = (double)r[j];

    // ---- O2 nine-point weights on the shifted window s0[j] = clamp(j - 4, 0, N - 9) (R3)
    std::vector<int> s0(N);
    std::vector<ld> D1(N * NPT), D2(N * NPT), L0(N * NPT);
    for (int j = 0; j < N; ++j) {
        int s = j - NPT / 2;
        if (s < 0) s = 0;
        if (s > N - NPT) s = N - NPT;
        s0[j] = s;
        ld w[NPT][3];
        fornberg(r[j], &r[s], NPT, w);
        for (int l = 0; l < NPT; ++l) {
            D1[j * NPT + l] = w[l][1];
            D2[j * NPT + l] = w[l][2];
            L0[j * NPT + l] = w[l][2] + w[l][1] / r[j];
        }
    }
    // ---- Q = (D1 + diag(1/r)) G~,  G~ = D1 with the two wall rows zeroed (R9)
    std::vector<int> q0(N);
    std::vector<ld> Q(N * QW, (ld)0);
    std::vector<int> qw(N);
    for (int j = 0; j < N; ++j) {
        int cmin = N, cmax = -1;
        for (int l = s0[j]; l < s0[j] + NPT; ++l) {
            if (l == 0 || l == N - 1) continue;
            if (s0[l] < cmin) cmin = s0[l];
            if (s0[l] + NPT - 1 > cmax) cmax = s0[l] + NPT - 1;
        }
        if (cmax - cmin + 1 > QW) return fail(c, NSC_EINVAL, "Poisson row wider than 17");
        q0[j] = cmin;
        qw[j] = cmax - cmin + 1;
        for (int l = s0[j]; l < s0[j] + NPT; ++l) {
            if (l == 0 || l == N - 1) continue;
            ld a = D1[j * NPT + (l - s0[j])] + (l == j ? 1 / r[j] : (ld)0);
            for (int q = 0; q < NPT; ++q) Q[j * QW + (s0[l] + q - cmin)] += a * D1[l * NPT + q];
        }
    }
    auto to_double = [](const std::vector<ld>& v) {
        std::vector<double> d(v.size());
        for (size_t i = 0; i < v.size(); ++i) d[i] = (double)v[i];
        return d;
    };
    std::vector<double> rinv(N);
    for (int j = 0; j < N; ++j) rinv[j] = (double)(1 / r[j]);
    std::vector<double> nm(c->M1), kap(c->NK);
    for (int m = 0; m < c->M1; ++m) nm[m] = (double)m * p.k_theta0;
    for (int k = -c->K; k <= c->K; ++k) kap[k + c->K] = (double)k * p.alpha;
    auto twiddles = [](int n) {
        std::vector<cd> t(n);
        for (int i = 0; i < n; ++i) {
            ld a = 2 * pi_ld() * i / n;
            t[i] = mk((double)cosl(a), (double)(-sinl(a)));
        }
        return t;
    };
    int rc;
    if ((rc = upload(c, &c->t.D1, to_double(D1)))) return rc;
    if ((rc = upload(c, &c->t.L0, to_double(L0)))) return rc;
    if ((rc = upload(c, &c->t.s0, s0))) return rc;
    if ((rc = upload(c, &c->t.Q, to_double(Q)))) return rc;
    if ((rc = upload(c, &c->t.q0, q0))) return rc;
    if ((rc = upload(c, &c->t.rinv, rinv))) return rc;
    if ((rc = upload(c, &c->t.nm, nm))) return rc;
    if ((rc = upload(c, &c->t.kap, kap))) return rc;
    if ((rc = upload(c, &c->t.tw_t, twiddles(c->Nt)))) return rc;
    if ((rc = upload(c, &c->t.tw_z, twiddles(c->Nz)))) return rc;
    // twiddle matrices of the warp transforms (fft_warp.cuh): tw[t][n2] = exp(-2 pi i (t % NA) n2 / N), row stride 33
    auto warp_table = [&](int n, cd** dst) -> int {
        if (n == fw::NPAIR) n /= 2;                      // a warp pair runs two transforms of length 768
        const int na = n / fw::NB;
        std::vector<cd> t(fw::XBUF, mk(0.0, 0.0));
        for (int r = 0; r < fw::NV; ++r)
            for (int n2 = 0; n2 < fw::NB; ++n2) {
                ld a = 2 * pi_ld() * (ld)((r % na) * n2) / n;
                t[r * fw::XS + n2] = mk((double)cosl(a), (double)(-sinl(a)));
            }
        return upload(c, dst, t);
    };
    if (c->z_na && (rc = warp_table(c->Nz, &c->t.tw_wz))) return rc;
    if (c->t_na && (rc = warp_table(c->Nt, &c->t.tw_wt))) return rc;
    if (c->z_na == 48 || c->t_na == 48) {
        std::vector<cd> t(fw::NPAIR / 2);
        for (int k = 0; k < fw::NPAIR / 2; ++k) {
            ld a = 2 * pi_ld() * (ld)k / fw::NPAIR;
            t[k] = mk((double)cosl(a), (double)(-sinl(a)));
        }
        if ((rc = upload(c, &c->t.tw_c1536, t))) return rc;
    }

    // ---- band envelopes.  Helmholtz: identity rows at the walls (Dirichlet), stencil rows inside.
    c->shH.h_lo.resize(N);
    c->shH.h_hi.resize(N);
    c->shP.h_lo.resize(N);
    c->shP.h_hi.resize(N);
    for (int j = 0; j < N; ++j) {
        bool wall = (j == 0 || j == N - 1);
        c->shH.h_lo[j] = wall ? j : s0[j];
        c->shH.h_hi[j] = wall ? j : s0[j] + NPT - 1;
        // Poisson: Neumann rows D1[wall] at the walls, Q rows inside
        c->shP.h_lo[j] = wall ? s0[j] : q0[j];
        c->shP.h_hi[j] = wall ? s0[j] + NPT - 1 : q0[j] + qw[j] - 1;
    }
    if ((rc = finish_shape(c, c->shH, 8))) return rc;
    if ((rc = finish_shape(c, c->shP, 12))) return rc;
    return NSC_OK;
}

}  // namespace nsc
