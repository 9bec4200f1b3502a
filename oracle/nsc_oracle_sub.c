/* nsc_oracle_sub.c -- plain C restatement of the oracle's implicit sub-step O6 (steps L1-L5 of
 * SURVEY.md 8(a); "predictor-corrector ... implicit", "linear terms ...
 * independently per Fourier mode"), for the 20-step parity runs at the large configurations.
 *
 * TEST INFRASTRUCTURE ONLY, part of oracle/: nothing in the product path may link or load it, and it
 * shares no code, table or constant with the CUDA path (its tables are handed in by
 * oracle/nsc_oracle.py, which builds them in long double from closed-form Lagrange derivatives).
 * It is the third solver backend of the oracle (solve="c"), pinned to the dense LAPACK backend and
 * to the numpy banded backend in tests/test_oracle_banded.py.
 *
 * One Fourier mode at a time, in the order of DESIGN.md section 2 (O6):
 *   L1  rhs_+- = u_+- + dt[(1-c) L_+- u_+- + E_+- - (D1 p -+ (n/r) p)],  rhs_z, rhs_T likewise
 *   L2  (I - c dt L) x = rhs, identity rows carrying the wall values (Dirichlet)
 *   L3  ur' = (x_+ + x_-)/2, ut' = (x_+ - x_-)/(2i), g = D1 ur' + ur' / r + (i n/r) ut' + i kappa uz'
 *   L4  P phi = g, P = Q - diag(n^2/r^2 + kappa^2), wall rows D1 phi = 0; mode (0,0) not projected (O8)
 *   L5  u = u' - (G~ phi, (i n/r) phi, i kappa phi), p += phi/dt, u_r(0,0) := 0
 * Linear systems: Gaussian elimination without pivoting inside the band (BASELINE.json north_star:
 * "dense or banded Gaussian elimination").  OpenMP over the modes only.
 */
#include <complex.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

enum { NPT = 9, HKL = 8, HKU = 8, PKL = 12, PKU = 12 };

/* a[j][d] = A[j][j - kl + d], d = 0 .. kl + ku; b overwritten by the solution */
static void band_solve(int N, int kl, int ku, double* a, cplx* b) {
    const int W = kl + ku + 1;
    for (int j = 0; j < N - 1; ++j) {
        const double piv = a[j * W + kl];
        const int imax = j + kl < N - 1 ? j + kl : N - 1;
        for (int i = j + 1; i <= imax; ++i) {
            const int o = kl - (i - j);
            const double v = a[i * W + o];
            if (v == 0.0) continue;
            const double l = v / piv;
            for (int d = 0; d <= ku; ++d) a[i * W + o + d] -= l * a[j * W + kl + d];
            b[i] -= l * b[j];
        }
    }
    for (int j = N - 1; j >= 0; --j) {
        cplx acc = b[j];
        const int dmax = ku < N - 1 - j ? ku : N - 1 - j;
        for (int d = 1; d <= dmax; ++d) acc -= a[j * W + kl + d] * b[j + d];
        b[j] = acc / a[j * W + kl];
    }
}

/* out[j] = sum_l rows[j][l] f[s0[j] + l] */
static void rows9(int N, const double* rows, const int* s0, const cplx* f, cplx* out) {
    for (int j = 0; j < N; ++j) {
        cplx acc = 0.0;
        for (int l = 0; l < NPT; ++l) acc += rows[j * NPT + l] * f[s0[j] + l];
        out[j] = acc;
    }
}

/* (I - coef (L0 - diag(q))) x = rhs with identity rows at the walls; rhs overwritten by x */
static void helmholtz(int N, const double* L0rows, const int* s0, const double* q, double coef, double* band, cplx* rhs) {
    const int W = HKL + HKU + 1;
    memset(band, 0, sizeof(double) * (size_t)N * W);
    for (int j = 1; j < N - 1; ++j) {
        for (int l = 0; l < NPT; ++l) band[j * W + (s0[j] + l - j + HKL)] = -coef * L0rows[j * NPT + l];
        band[j * W + HKL] += 1.0 + coef * q[j];
    }
    band[HKL] = 1.0;
    band[(N - 1) * W + HKL] = 1.0;
    band_solve(N, HKL, HKU, band, rhs);
}

int orc_substep(int N_r, int M1, int NK, int K, int nf, const double* r, const double* n, const double* kappa,
                const double* D1rows, const double* L0rows, const int* s0,
                const double* Pband, /* [N_r][25]: Q with the wall rows replaced by D1's, kl = ku = 12 */
                const cplx* ur, const cplx* ut, const cplx* uz, const cplx* T, const cplx* pr, const cplx* Er,
                const cplx* Et, const cplx* Ez, const cplx* ET, double dt, double c, double Pr, double Re_i,
                double Re_o, const int* IM, const int* IK, int nB, cplx* o_ur, cplx* o_ut, cplx* o_uz, cplx* o_T,
                cplx* o_p) {
    const int N = N_r;
    const size_t plane = (size_t)M1 * NK;
    const int heated = nf == 4;
    int failed = 0;
#pragma omp parallel
    {
        const int WP = PKL + PKU + 1, WH = HKL + HKU + 1;
        cplx* w = (cplx*)malloc(sizeof(cplx) * (size_t)N * 16);
        double* band = (double*)malloc(sizeof(double) * (size_t)N * (WP > WH ? WP : WH));
        double* q = (double*)malloc(sizeof(double) * (size_t)N);
        if (!w || !band || !q) {
#pragma omp atomic write
            failed = 1;
        } else {
            cplx *cur = w, *cut = w + N, *cuz = w + 2 * N, *cT = w + 3 * N, *cp = w + 4 * N, *up = w + 5 * N,
                 *um = w + 6 * N, *dp = w + 7 * N, *lap = w + 8 * N, *rp = w + 9 * N, *rm = w + 10 * N,
                 *rz = w + 11 * N, *rT = w + 12 * N, *g = w + 13 * N, *tmp = w + 14 * N, *uts = w + 15 * N;
#pragma omp for schedule(dynamic, 8)
            for (int b = 0; b < nB; ++b) {
                const int m = IM[b], kk = IK[b];
                const double nn = n[m], kap = kappa[kk];
                const int m00 = (m == 0 && kk == K);
                const size_t e = (size_t)m * NK + kk;
                for (int j = 0; j < N; ++j) {
                    const size_t o = (size_t)j * plane + e;
                    cur[j] = ur[o];
                    cut[j] = ut[o];
                    cuz[j] = uz[o];
                    cp[j] = pr[o];
                    if (heated) cT[j] = T[o];
                    up[j] = cur[j] + I * cut[j];
                    um[j] = cur[j] - I * cut[j];
                }
                /* L1 */
                rows9(N, D1rows, s0, cp, dp);
                rows9(N, L0rows, s0, up, lap);
                for (int j = 0; j < N; ++j) {
                    const size_t o = (size_t)j * plane + e;
                    const double qq = (nn + 1.0) * (nn + 1.0) / (r[j] * r[j]) + kap * kap;
                    rp[j] = up[j] + dt * ((1.0 - c) * (lap[j] - qq * up[j]) + (Er[o] + I * Et[o]) - (dp[j] - nn / r[j] * cp[j]));
                }
                rows9(N, L0rows, s0, um, lap);
                for (int j = 0; j < N; ++j) {
                    const size_t o = (size_t)j * plane + e;
                    const double qq = (nn - 1.0) * (nn - 1.0) / (r[j] * r[j]) + kap * kap;
                    rm[j] = um[j] + dt * ((1.0 - c) * (lap[j] - qq * um[j]) + (Er[o] - I * Et[o]) - (dp[j] + nn / r[j] * cp[j]));
                }
                rows9(N, L0rows, s0, cuz, lap);
                for (int j = 0; j < N; ++j) {
                    const size_t o = (size_t)j * plane + e;
                    const double qq = nn * nn / (r[j] * r[j]) + kap * kap;
                    rz[j] = cuz[j] + dt * ((1.0 - c) * (lap[j] - qq * cuz[j]) + Ez[o] - I * kap * cp[j]);
                }
                if (heated) {
                    rows9(N, L0rows, s0, cT, lap);
                    for (int j = 0; j < N; ++j) {
                        const size_t o = (size_t)j * plane + e;
                        const double qq = nn * nn / (r[j] * r[j]) + kap * kap;
                        rT[j] = cT[j] + dt * ((1.0 - c) / Pr * (lap[j] - qq * cT[j]) + ET[o]);
                    }
                }
                /* Dirichlet data (R1) */
                rp[0] = rp[N - 1] = rm[0] = rm[N - 1] = rz[0] = rz[N - 1] = 0.0;
                if (heated) rT[0] = rT[N - 1] = 0.0;
                if (m00) {
                    rp[0] = I * Re_i;
                    rp[N - 1] = I * Re_o;
                    rm[0] = -I * Re_i;
                    rm[N - 1] = -I * Re_o;
                    if (heated) {
                        rT[0] = 0.5;
                        rT[N - 1] = -0.5;
                    }
                }
                /* L2 */
                for (int j = 0; j < N; ++j) q[j] = (nn + 1.0) * (nn + 1.0) / (r[j] * r[j]) + kap * kap;
                helmholtz(N, L0rows, s0, q, c * dt, band, rp);
                for (int j = 0; j < N; ++j) q[j] = (nn - 1.0) * (nn - 1.0) / (r[j] * r[j]) + kap * kap;
                helmholtz(N, L0rows, s0, q, c * dt, band, rm);
                for (int j = 0; j < N; ++j) q[j] = nn * nn / (r[j] * r[j]) + kap * kap;
                helmholtz(N, L0rows, s0, q, c * dt, band, rz);
                if (heated) helmholtz(N, L0rows, s0, q, c * dt / Pr, band, rT);
                /* L3: rp <- ur', uts <- ut' */
                for (int j = 0; j < N; ++j) {
                    const cplx a = rp[j], bq = rm[j];
                    rp[j] = (a + bq) / 2.0;
                    uts[j] = (a - bq) / (2.0 * I);
                }
                rows9(N, D1rows, s0, rp, tmp);
                for (int j = 0; j < N; ++j) g[j] = tmp[j] + rp[j] / r[j] + I * nn / r[j] * uts[j] + I * kap * rz[j];
                g[0] = g[N - 1] = 0.0;
                /* L4 */
                if (m00) {
                    for (int j = 0; j < N; ++j) g[j] = 0.0;
                } else {
                    memcpy(band, Pband, sizeof(double) * (size_t)N * WP);
                    for (int j = 1; j < N - 1; ++j) band[j * WP + PKL] -= q[j];
                    band_solve(N, PKL, PKU, band, g);
                }
                /* L5 (g holds phi) */
                rows9(N, D1rows, s0, g, tmp);
                tmp[0] = tmp[N - 1] = 0.0;
                for (int j = 0; j < N; ++j) {
                    const size_t o = (size_t)j * nB + b;
                    o_ur[o] = m00 ? 0.0 : rp[j] - tmp[j];
                    o_ut[o] = uts[j] - I * nn / r[j] * g[j];
                    o_uz[o] = rz[j] - I * kap * g[j];
                    if (heated) o_T[o] = rT[j];
                    o_p[o] = cp[j] + g[j] / dt;
                }
            }
        }
        free(w);
        free(band);
        free(q);
    }
    return failed ? -1 : 0;
}
