// linear.cu -- the implicit sub-step (DESIGN.md steps L1-L5; BASELINE.json north_star (b)):
//   L1 right-hand sides, L2 banded Helmholtz solves for u_+- = u_r +- i u_theta, u_z, T,
//   L3 recombination + divergence, L4 pressure-Poisson solve, L5 correction and update.
// PAPER.md:46 (predictor-corrector, implicit linear terms), PAPER.md:64 ("linear terms ...
// independently per Fourier mode").
//
// Per-mode matrices differ from mode to mode only on the diagonal:
//   Helmholtz  A = I - coef (L0 - diag((n + shift)^2 / r^2 + kappa^2)),  identity rows at the walls
//   Poisson    P = Q - diag(n^2 / r^2 + kappa^2),  Neumann rows D1[wall] at the walls (R9)
// and are the same for +k and -k.  They are LU-factored without pivoting inside their row envelope
// (no fill-in outside it) once per dt (Helmholtz) / once per context (Poisson), pair-major
// ("pair" = (m, |k|)).  The sub-step is four marching sweeps over the radial index, one thread per
// (mode, field), every row's operands prefetched into shared memory by a cp.async row pipeline:
//   k_rhs_fwd (up) -> k_bwd_div (down) -> k_poisson_fwd (up) -> k_poisson_bwd_correct (down).
#include <cstdint>
#include "nsc_internal.h"

namespace nsc {

// ------------------------------------------------------------------------------------------
// factorisation (set-up; generic, one thread per pair, row scratch in local memory)
struct FacArgs {
    const double* band;   // [N_r][BW] operator rows (L0 or Q)
    const int* bcol0;     // [N_r] first column of the stored row
    const double* D1;     // wall rows of the Poisson matrix
    const int* s0;
    const double* rinv;
    const double* nm;
    const double* kap;
    const int *lo, *hi, *offL, *offU;
    double* L;
    double* U;
    int N_r, K, P, bw;
    int kind;             // 0 Helmholtz, 1 Poisson
    double coef, shift;
};

constexpr int ROWMAX = 32;

__global__ void k_factor(FacArgs a) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.P) return;
    const int m = p / (a.K + 1), ka = p % (a.K + 1);
    const double n = a.nm[m] + a.shift;
    const double kap = a.kap[a.K + ka];
    const size_t P = a.P;
    const bool singular = (a.kind == 1 && m == 0 && ka == 0);   // O8: mode (0,0) is not projected
    double w[ROWMAX];
    for (int j = 0; j < a.N_r; ++j) {
        const int lo = a.lo[j], hi = a.hi[j];
        const int width = hi - lo + 1;
        for (int i = 0; i < width; ++i) w[i] = 0.0;
        const bool wall = (j == 0 || j == a.N_r - 1);
        const double ri = a.rinv[j];
        const double q = n * n * ri * ri + kap * kap;
        if (a.kind == 0) {
            if (wall) {
                w[j - lo] = 1.0;
            } else {
                const int c0 = a.bcol0[j];
                for (int l = 0; l < a.bw; ++l) w[c0 + l - lo] = -a.coef * a.band[j * a.bw + l];
                w[j - lo] += 1.0 + a.coef * q;
            }
        } else {
            if (wall) {
                const int c0 = a.s0[j];
                for (int l = 0; l < NPT; ++l) w[c0 + l - lo] = a.D1[j * NPT + l];
            } else {
                const int c0 = a.bcol0[j];
                for (int l = 0; l < a.bw; ++l) {
                    const int col = c0 + l;
                    if (col <= hi) w[col - lo] = a.band[j * a.bw + l];
                }
                w[j - lo] -= q;
            }
        }
        // eliminate columns lo..j-1 with the already factored rows
        for (int cidx = lo; cidx < j; ++cidx) {
            const size_t ou = (size_t)a.offU[cidx];
            const double l = w[cidx - lo] * a.U[ou * P + p];          // times 1/pivot of row cidx
            a.L[((size_t)a.offL[j] + (cidx - lo)) * P + p] = singular ? 0.0 : l;
            const int nu = a.hi[cidx] - cidx;
            for (int i = 1; i <= nu; ++i) w[cidx + i - lo] -= l * a.U[(ou + i) * P + p];
        }
        const size_t ou = (size_t)a.offU[j];
        a.U[ou * P + p] = singular ? 0.0 : 1.0 / w[j - lo];
        for (int i = 1; i <= hi - j; ++i) a.U[(ou + i) * P + p] = singular ? 0.0 : w[j + i - lo];
    }
}

// ------------------------------------------------------------------------------------------
// Fused sweeps.  One thread serves one (mode, field): field 0 u_+, 1 u_-, 2 u_z, 3 T;
// the factors of the pair (m, |k|) are read by both of its modes (the second read hits L2).
//
// With A = I - c dt nu L and gamma = (1 - c) / c the right-hand side of step L1 is
//     u + dt (1 - c) nu L u + dt R  =  u / c - gamma A u + dt R        (R = E - pressure-gradient term),
// so   x = A^-1 (u / c + dt R) - gamma u   at interior rows: no radial stencil acts on u.  D1 p is kept
// as an array of its own (DP), updated by k_poisson_bwd_correct with D1 phi / dt (D1 is linear).  Wall rows of A are identity rows: b_wall = BC + gamma u_wall.
//
//   k_rhs_fwd  (marching up)   : b from u, E, p, D1 p, forward
//                                substitution with the stored L factors, y -> W[field]
//   k_bwd_div  (marching down) : back substitution, - gamma u, recombination of u_+- into
//                                (u_r*, u_theta*), divergence g (L2, L3) -- see below
struct FusedArgs {
    const cd* u[MAXF];
    const cd* p;
    const cd* DP;          // D1 p (interior rows)
    const cd* E0[MAXF];
    const cd* E1[MAXF];    // may be null
    cd* W[MAXF];
    cd* G;
    const double* L[MAXF];
    const double* U[MAXF];
    const int *lo, *hi, *offL, *offU;
    const double *D1, *rinv, *nm, *kap;
    const int* s0;
    int N_r, M1, NK, K, P, nf;
    int offL4, offU4;      // offL[4], offU[4]: the interior rows 4 .. N_r - 5 have regular offsets
    int e_begin, e_end;    // slice of modes [e_begin, e_end) this launch serves
    double dt, c, w0, w1, Re_i, Re_o;
};

constexpr int FW = 8;       // forward / backward substitution window (rows), Helmholtz envelope <= 7
constexpr int FWI = 4;      // interior lower / upper width

__device__ __forceinline__ cd ldcs(const cd* p) {
    const double2 v = __ldcs(reinterpret_cast<const double2*>(p));
    return mk(v.x, v.y);
}

// ---- row pipeline: every row's operands arrive in shared memory by cp.async, PIPE - 1 rows ahead of
// the row being eliminated, so that the marching threads never wait on HBM with a single row in flight
constexpr int PBK = 32;          // modes per block
// shared-memory row slots of the four sweeps (rows in flight = slots - 1); measured: more resident blocks beat deeper pipelines
constexpr int PIPE_F = 3, PIPE_B = 3, PIPE_PF = 3, PIPE_PB = 2;
__device__ __forceinline__ void cpa16(void* s, const void* g) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(s)), "l"(g) : "memory");
}
__device__ __forceinline__ void cpa8(void* s, const void* g) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(s)), "l"(g) : "memory");
}
__device__ __forceinline__ void cpa_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPEND> __device__ __forceinline__ void cpa_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(NPEND) : "memory");
}

// The substitution windows are rings indexed by (row & (ring - 1)) held in registers; the row loops are
// unrolled by the ring length so that every ring index is a compile-time constant (no register moves).
template <int R> struct RowTag { static constexpr int value = R; };
#define NSC_ROWS8(F, j0)                                                                             \
    F(RowTag<0>{}, (j0) + 0); F(RowTag<1>{}, (j0) + 1); F(RowTag<2>{}, (j0) + 2); F(RowTag<3>{}, (j0) + 3); \
    F(RowTag<4>{}, (j0) + 4); F(RowTag<5>{}, (j0) + 5); F(RowTag<6>{}, (j0) + 6); F(RowTag<7>{}, (j0) + 7)
#define NSC_ROWS16(F, j0) \
    NSC_ROWS8(F, j0);     \
    F(RowTag<8>{}, (j0) + 8); F(RowTag<9>{}, (j0) + 9); F(RowTag<10>{}, (j0) + 10); F(RowTag<11>{}, (j0) + 11); \
    F(RowTag<12>{}, (j0) + 12); F(RowTag<13>{}, (j0) + 13); F(RowTag<14>{}, (j0) + 14); F(RowTag<15>{}, (j0) + 15)
#define NSC_ROWS16_DOWN(F, j0) \
    F(RowTag<15>{}, (j0) + 15); F(RowTag<14>{}, (j0) + 14); F(RowTag<13>{}, (j0) + 13); F(RowTag<12>{}, (j0) + 12); \
    F(RowTag<11>{}, (j0) + 11); F(RowTag<10>{}, (j0) + 10); F(RowTag<9>{}, (j0) + 9); F(RowTag<8>{}, (j0) + 8); \
    NSC_ROWS8_DOWN(F, j0)
#define NSC_ROWS8_DOWN(F, j0)                                                                        \
    F(RowTag<7>{}, (j0) + 7); F(RowTag<6>{}, (j0) + 6); F(RowTag<5>{}, (j0) + 5); F(RowTag<4>{}, (j0) + 4); \
    F(RowTag<3>{}, (j0) + 3); F(RowTag<2>{}, (j0) + 2); F(RowTag<1>{}, (j0) + 1); F(RowTag<0>{}, (j0) + 0)

// k_rhs_fwd: block = (PBK modes) x (NF fields).  Slot arrays: u[NF], p, DP, E0[NF], E1[NF] (if present).
template <int NF> struct FwdSlot {
    cd fld[3 * NF + 2][PBK];
    double L[NF][FWI][PBK];
};

template <int NF>
__global__ void __launch_bounds__(PBK * NF, 1) k_rhs_fwd(FusedArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FwdSlot<NF>* slots = reinterpret_cast<FwdSlot<NF>*>(smem_raw);
    const int tx = threadIdx.x, fld = threadIdx.y;
    const int plane_i = a.M1 * a.NK;
    const int e0 = a.e_begin + blockIdx.x * PBK + tx;
    const bool valid = e0 < a.e_end;
    const int e = valid ? e0 : a.e_end - 1;
    const int m = e / a.NK, kk = e % a.NK;
    const int ka = kk >= a.K ? kk - a.K : a.K - kk;
    const size_t P = a.P;
    const size_t plane = (size_t)plane_i;
    const int N = a.N_r;
    const double n = a.nm[m], kap = a.kap[kk];
    const double ic = 1.0 / a.c, gam = (1.0 - a.c) / a.c, dt = a.dt;
    const bool m00 = (m == 0 && ka == 0);
    const bool two = a.E1[0] != nullptr;
    const int narr = two ? 3 * NF + 2 : 2 * NF + 2;
    const double* Lf = (fld == 0 ? a.L[0] : fld == 1 ? a.L[1] : fld == 2 ? a.L[2] : a.L[3]) + (size_t)m * (a.K + 1) + ka;
    cd* Wf = fld == 0 ? a.W[0] : fld == 1 ? a.W[1] : fld == 2 ? a.W[2] : a.W[3];
    const int ja = FWI, jb = N - FWI;                    // interior rows [ja, jb): nl = 4, offL regular
    // array q of the slot: 0..NF-1 u, NF p, NF+1 DP, NF+2.. E0, 2NF+2.. E1
    auto src_of = [&](int q) -> const cd* {
        if (q < NF) return q == 0 ? a.u[0] : q == 1 ? a.u[1] : q == 2 ? a.u[2] : a.u[3];
        if (q == NF) return a.p;
        if (q == NF + 1) return a.DP;
        q -= NF + 2;
        if (q < NF) return q == 0 ? a.E0[0] : q == 1 ? a.E0[1] : q == 2 ? a.E0[2] : a.E0[3];
        q -= NF;
        return q == 0 ? a.E1[0] : q == 1 ? a.E1[1] : q == 2 ? a.E1[2] : a.E1[3];
    };
    // this thread requests arrays fld, fld + NF, ... of every row: source pointers resolved once
    constexpr int NQ = (3 * NF + 2 + NF - 1) / NF;
    const cd* gp[NQ];
#pragma unroll
    for (int k = 0; k < NQ; ++k) gp[k] = (fld + k * NF < narr) ? src_of(fld + k * NF) + e : nullptr;
    auto issue = [&](int j) {
        if (j < N) {
            FwdSlot<NF>& s = slots[j % PIPE_F];
            const size_t o = (size_t)j * plane;
#pragma unroll
            for (int k = 0; k < NQ; ++k)
                if (gp[k]) cpa16(&s.fld[fld + k * NF][tx], gp[k] + o);
            if (j >= ja && j < jb) {
                const double* Lr = Lf + (size_t)(a.offL4 + FWI * (j - ja)) * P;
#pragma unroll
                for (int i = 0; i < FWI; ++i) cpa8(&s.L[fld][i][tx], Lr + (size_t)i * P);
            }
        }
        cpa_commit();
    };
    cd w[FW];                                           // ring: y_j lives in w[j & 7]
#pragma unroll
    for (int i = 0; i < FW; ++i) w[i] = mk(0.0, 0.0);
#pragma unroll
    for (int d = 0; d < PIPE_F - 1; ++d) issue(d);
    auto row = [&](auto tag, int j) {
        constexpr int R = decltype(tag)::value;
        if (j >= N) return;
        cpa_wait<PIPE_F - 2>();
        __syncthreads();
        issue(j + PIPE_F - 1);
        const FwdSlot<NF>& s = slots[j % PIPE_F];
        const bool wall = (j == 0 || j == N - 1);
        cd b;
        if (fld < 2) {
            const double sg = fld == 0 ? 1.0 : -1.0;
            const cd ur = s.fld[0][tx], ut = s.fld[1][tx];
            const cd u = mk(ur.x - sg * ut.y, ur.y + sg * ut.x);         // u_r + sg i u_theta
            if (wall) {
                const double v = m00 ? sg * (j == 0 ? a.Re_i : a.Re_o) : 0.0;
                b = mk(gam * u.x, v + gam * u.y);
            } else {
                cd Er = a.w0 * s.fld[NF + 2][tx], Et = a.w0 * s.fld[NF + 3][tx];
                if (two) {
                    Er = Er + a.w1 * s.fld[2 * NF + 2][tx];
                    Et = Et + a.w1 * s.fld[2 * NF + 3][tx];
                }
                const cd Dp = s.fld[NF + 1][tx], pr = s.fld[NF][tx];
                const double nr = sg * n * a.rinv[j];
                // R = (E_r + sg i E_theta) - (D1 p - sg (n / r) p)
                const cd R = mk(Er.x - sg * Et.y - Dp.x + nr * pr.x, Er.y + sg * Et.x - Dp.y + nr * pr.y);
                b = mk(fma(dt, R.x, ic * u.x), fma(dt, R.y, ic * u.y));
            }
        } else {
            const cd u = s.fld[fld][tx];
            if (wall) {
                const double v = (fld == 3 && m00) ? (j == 0 ? 0.5 : -0.5) : 0.0;
                b = mk(v + gam * u.x, gam * u.y);
            } else {
                cd E = a.w0 * s.fld[NF + 2 + fld][tx];
                if (two) E = E + a.w1 * s.fld[2 * NF + 2 + fld][tx];
                if (fld == 2) {                         // - i kappa p
                    const cd pr = s.fld[NF][tx];
                    E = mk(E.x + kap * pr.y, E.y - kap * pr.x);
                }
                b = mk(fma(dt, E.x, ic * u.x), fma(dt, E.y, ic * u.y));
            }
        }
        // forward substitution: y_j = b_j - sum_{d=1..nl} L[j][nl - d] y_{j-d}
        if (j >= ja && j < jb) {
#pragma unroll
            for (int d = FWI; d >= 1; --d) {
                const double l = s.L[fld][FWI - d][tx];
                b.x = fma(-l, w[(R - d) & 7].x, b.x);
                b.y = fma(-l, w[(R - d) & 7].y, b.y);
            }
        } else {
            const int nl = j - a.lo[j];
            const double* Lr = Lf + (size_t)a.offL[j] * P;
#pragma unroll
            for (int d = FW - 1; d >= 1; --d) {
                if (d <= nl) {
                    const double l = Lr[(size_t)(nl - d) * P];
                    b.x = fma(-l, w[(R - d) & 7].x, b.x);
                    b.y = fma(-l, w[(R - d) & 7].y, b.y);
                }
            }
        }
        w[R] = b;
        if (valid) Wf[(size_t)j * plane + e] = b;
    };
    for (int j0 = 0; j0 < N; j0 += 8) {
        NSC_ROWS8(row, j0);
    }
    cpa_wait<0>();
}

// k_bwd_div: block = (PBK modes) x (NF field roles + 1 divergence role), marching down.  Field role f
// back-substitutes its system, subtracts gamma u_f and hands x_f(j) to the divergence role through
// a double-buffered shared-memory slot (one barrier per row, the divergence role runs one row behind); the divergence role forms
// u_r* = (x_+ + x_-)/2, u_theta* = (x_+ - x_-)/(2i), stores them and emits
// g = D1 u_r* + u_r*/r + (i n / r) u_theta* + i kappa u_z* four rows behind the march, from a ring of the
// last rows of u_r* in shared memory (g = 0 in the wall rows).  Slot arrays: y[NF] (in W), u[NF], U rows.
template <int NF> struct BwdSlot {
    cd fld[2 * NF][PBK];
    double U[NF][FWI + 1][PBK];
};

template <int NF>
__global__ void __launch_bounds__(PBK * (NF + 1), NF == 3 ? 5 : 3) k_bwd_div(FusedArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    BwdSlot<NF>* slots = reinterpret_cast<BwdSlot<NF>*>(smem_raw);
    __shared__ cd exch[2][3][PBK];
    __shared__ cd ring_ur[16][PBK];                     // u_r* of the last rows (column tx is private to the
    __shared__ cd ring_g[FW][PBK];                      // divergence-role thread tx), stencil-free part of g
    const int tx = threadIdx.x, role = threadIdx.y;
    const int plane_i = a.M1 * a.NK;
    const int e0 = a.e_begin + blockIdx.x * PBK + tx;
    const bool valid = e0 < a.e_end;
    const int e = valid ? e0 : a.e_end - 1;
    const int m = e / a.NK, kk = e % a.NK;
    const int ka = kk >= a.K ? kk - a.K : a.K - kk;
    const size_t P = a.P;
    const size_t plane = (size_t)plane_i;
    const int N = a.N_r;
    const double n = a.nm[m], kap = a.kap[kk];
    const double gam = (1.0 - a.c) / a.c;
    const bool is_field = role < NF;
    const int f = is_field ? role : 0;
    const double* Uf = (f == 0 ? a.U[0] : f == 1 ? a.U[1] : f == 2 ? a.U[2] : a.U[3]) + (size_t)m * (a.K + 1) + ka;
    cd* Wf = f == 0 ? a.W[0] : f == 1 ? a.W[1] : f == 2 ? a.W[2] : a.W[3];
    const double sg = f == 0 ? 1.0 : -1.0;
    const int ja = FWI, jb = N - FWI;                    // interior rows [ja, jb): nu = 4, offU regular
    auto src_of = [&](int q) -> const cd* {
        if (q < NF) return q == 0 ? a.W[0] : q == 1 ? a.W[1] : q == 2 ? a.W[2] : a.W[3];
        q -= NF;
        return q == 0 ? a.u[0] : q == 1 ? a.u[1] : q == 2 ? a.u[2] : a.u[3];
    };
    // this thread requests arrays role, role + NF + 1 of every row: source pointers resolved once
    constexpr int NQ = (2 * NF + NF) / (NF + 1);
    const cd* gp[NQ];
#pragma unroll
    for (int k = 0; k < NQ; ++k) gp[k] = (role + k * (NF + 1) < 2 * NF) ? src_of(role + k * (NF + 1)) + e : nullptr;
    // row j travels in slot (N - 1 - j) % PIPE_B
    auto issue = [&](int j) {
        if (j >= 0) {
            BwdSlot<NF>& s = slots[(N - 1 - j) % PIPE_B];
            const size_t o = (size_t)j * plane;
#pragma unroll
            for (int k = 0; k < NQ; ++k)
                if (gp[k]) cpa16(&s.fld[role + k * (NF + 1)][tx], gp[k] + o);
            if (is_field && j >= ja && j < jb) {
                const double* Ur = Uf + (size_t)(a.offU4 + (FWI + 1) * (j - ja)) * P;
#pragma unroll
                for (int i = 0; i <= FWI; ++i) cpa8(&s.U[f][i][tx], Ur + (size_t)i * P);
            }
        }
        cpa_commit();
    };
    cd w[FW];                                           // back-substitution ring: x_j lives in w[j & 7]
#pragma unroll
    for (int i = 0; i < FW; ++i) w[i] = mk(0.0, 0.0);
    // divergence role, row j (its x_+, x_-, x_z were left in exch[j & 1] one iteration earlier)
    auto div_row = [&](int j) {
        const size_t o = (size_t)j * plane + e;
        const cd xa = exch[j & 1][0][tx], xb = exch[j & 1][1][tx], xz = exch[j & 1][2][tx];
        const cd ur = 0.5 * (xa + xb);
        const cd ut = 0.5 * mul_mi(xa - xb);
        if (valid) {
            a.W[0][o] = ur;
            a.W[1][o] = ut;
        }
        const double ri = a.rinv[j], nr = n * ri;
        ring_ur[j & 15][tx] = ur;
        // u_r*/r + (i n / r) u_theta* + i kappa u_z*
        ring_g[j & (FW - 1)][tx] = mk(ri * ur.x - nr * ut.y - kap * xz.y, ri * ur.y + nr * ut.x + kap * xz.x);
        if (valid) {
            if (j == N - 1 || j == 0) a.G[o] = mk(0.0, 0.0);
            if (j <= N - NPT) {
                // rows whose stencil is the window j .. j + 8
                const int c_lo = (j == 0) ? 1 : j + NPT / 2;
                const int c_hi = (j == N - NPT) ? N - 2 : j + NPT / 2;
                for (int jc = c_lo; jc <= c_hi; ++jc) {
                    const double* d = a.D1 + jc * NPT;
                    cd g = ring_g[jc & (FW - 1)][tx];
#pragma unroll
                    for (int l = 0; l < NPT; ++l) {
                        const double wt = __ldg(d + l);
                        const cd v = ring_ur[(j + l) & 15][tx];
                        g.x = fma(wt, v.x, g.x);
                        g.y = fma(wt, v.y, g.y);
                    }
                    a.G[(size_t)jc * plane + e] = g;
                }
            }
        }
    };
#pragma unroll
    for (int d = 0; d < PIPE_B - 1; ++d) issue(N - 1 - d);
    auto row = [&](auto tag, int j) {
        constexpr int R = decltype(tag)::value;
        if (j >= N) return;
        cpa_wait<PIPE_B - 2>();
        __syncthreads();                                 // row j has arrived; exch[(j + 1) & 1] is complete
        issue(j - (PIPE_B - 1));
        const BwdSlot<NF>& s = slots[(N - 1 - j) % PIPE_B];
        const size_t o = (size_t)j * plane + e;
        if (is_field) {
            cd y = s.fld[f][tx];
            // x_j = (y_j - sum_{d=1..nu} U[j][d] x_{j+d}) / pivot;  x_j lives in w[j & 7]
            if (j >= ja && j < jb) {
#pragma unroll
                for (int d = FWI; d >= 1; --d) {
                    const double u = s.U[f][d][tx];
                    y.x = fma(-u, w[(R + d) & 7].x, y.x);
                    y.y = fma(-u, w[(R + d) & 7].y, y.y);
                }
                y = s.U[f][0][tx] * y;
            } else {
                const int nu = a.hi[j] - j;
                const double* Ur = Uf + (size_t)a.offU[j] * P;
#pragma unroll
                for (int d = FW - 1; d >= 1; --d) {
                    if (d <= nu) {
                        const double u = Ur[(size_t)d * P];
                        y.x = fma(-u, w[(R + d) & 7].x, y.x);
                        y.y = fma(-u, w[(R + d) & 7].y, y.y);
                    }
                }
                y = Ur[0] * y;
            }
            w[R] = y;
            cd u;                                        // u_f of the state the sub-step starts from
            if (f < 2) {
                const cd ur = s.fld[NF][tx], ut = s.fld[NF + 1][tx];
                u = mk(ur.x - sg * ut.y, ur.y + sg * ut.x);
            } else {
                u = s.fld[NF + f][tx];
            }
            const cd x = mk(fma(-gam, u.x, y.x), fma(-gam, u.y, y.y));
            if (f < 3) exch[j & 1][f][tx] = x;
            if (f >= 2 && valid) Wf[o] = x;
        }
        if (!is_field && j < N - 1) div_row(j + 1);      // one row behind the field roles
    };
    for (int j0 = (N - 1) & ~7; j0 >= 0; j0 -= 8) {
        NSC_ROWS8_DOWN(row, j0);
    }
    __syncthreads();
    if (!is_field) div_row(0);
    cpa_wait<0>();
}

// ------------------------------------------------------------------------------------------
// Pressure stage of the fused path (L4, L5), one thread per mode, same row pipeline:
//   k_poisson_fwd (marching up)  : forward substitution of P phi = g with the stored L factors, in place in G
//   k_poisson_bwd_correct (down) : back substitution, phi kept in a shared-memory ring (never stored);
//                                  four rows behind the march  u = u* - (G~ phi, (i n / r) phi, i kappa phi),
//                                  p += phi / dt, D1 p += D1 phi / dt, u_r(0,0) := 0 (O8)
struct PoisArgs {
    cd* G;
    const double* L;
    const double* U;
    const int *lo, *hi, *offL, *offU;
    int jaL, jbL, offLa;   // rows [jaL, jbL): nl = PWI, offL[j] = offLa + PWI (j - jaL)
    int jaU, jbU, offUa;   // rows [jaU, jbU): nu = PWI, offU[j] = offUa + (PWI + 1)(j - jaU)
    const cd* W[MAXF];     // u_r*, u_theta*, u_z*, T
    cd* dst[MAXF];
    const cd* p;
    cd* p_dst;             // may be null: pressure discarded
    cd* DP_dst;            // D1 p of the new pressure (with p_dst)
    const cd* DP;
    const double *D1, *rinv, *nm, *kap;
    const int* s0;
    int N_r, M1, NK, K, P, nf;
    int copyT;             // dst[3] != W[3]
    int e_begin, e_end;    // slice of modes [e_begin, e_end) this launch serves
    double dt;
};

constexpr int PBP = 128;    // modes per block, forward sweep
constexpr int PBB = 64;     // modes per block, backward sweep + correction
constexpr int PW = 16;      // substitution ring (Poisson envelope <= 12)
constexpr int PWI = 8;      // interior lower / upper width

struct PFwdSlot {
    cd g[PBP];
    double L[PWI][PBP];
};

__global__ void __launch_bounds__(PBP) k_poisson_fwd(PoisArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PFwdSlot* slots = reinterpret_cast<PFwdSlot*>(smem_raw);
    const int tx = threadIdx.x;
    const int plane_i = a.M1 * a.NK;
    const int e0 = a.e_begin + blockIdx.x * PBP + tx;
    const bool valid = e0 < a.e_end;
    const int e = valid ? e0 : a.e_end - 1;
    const int m = e / a.NK, kk = e % a.NK;
    const int ka = kk >= a.K ? kk - a.K : a.K - kk;
    const size_t P = a.P;
    const size_t plane = (size_t)plane_i;
    const int N = a.N_r;
    const double* Lf = a.L + (size_t)m * (a.K + 1) + ka;
    auto issue = [&](int j) {
        if (j < N) {
            PFwdSlot& s = slots[j % PIPE_PF];
            cpa16(&s.g[tx], a.G + (size_t)j * plane + e);
            if (j >= a.jaL && j < a.jbL) {
                const double* Lr = Lf + (size_t)(a.offLa + PWI * (j - a.jaL)) * P;
#pragma unroll
                for (int i = 0; i < PWI; ++i) cpa8(&s.L[i][tx], Lr + (size_t)i * P);
            }
        }
        cpa_commit();
    };
    cd w[PW];                                           // ring: y_j lives in w[j & 15]
#pragma unroll
    for (int i = 0; i < PW; ++i) w[i] = mk(0.0, 0.0);
#pragma unroll
    for (int d = 0; d < PIPE_PF - 1; ++d) issue(d);
    auto row = [&](auto tag, int j) {
        constexpr int R = decltype(tag)::value;
        if (j >= N) return;
        cpa_wait<PIPE_PF - 2>();
        __syncthreads();
        issue(j + PIPE_PF - 1);
        const PFwdSlot& s = slots[j % PIPE_PF];
        cd b = s.g[tx];
        // y_j = b_j - sum_{d=1..nl} L[j][nl - d] y_{j-d}
        if (j >= a.jaL && j < a.jbL) {
#pragma unroll
            for (int d = PWI; d >= 1; --d) {
                const double l = s.L[PWI - d][tx];
                b.x = fma(-l, w[(R - d) & 15].x, b.x);
                b.y = fma(-l, w[(R - d) & 15].y, b.y);
            }
        } else {
            const int nl = j - a.lo[j];
            const double* Lr = Lf + (size_t)a.offL[j] * P;
#pragma unroll
            for (int d = 12; d >= 1; --d) {
                if (d <= nl) {
                    const double l = Lr[(size_t)(nl - d) * P];
                    b.x = fma(-l, w[(R - d) & 15].x, b.x);
                    b.y = fma(-l, w[(R - d) & 15].y, b.y);
                }
            }
        }
        w[R] = b;
        if (valid) a.G[(size_t)j * plane + e] = b;
    };
    for (int j0 = 0; j0 < N; j0 += 16) {
        NSC_ROWS16(row, j0);
    }
    cpa_wait<0>();
}

// slot of row j: y[j], U rows of j, and the correction operands of row j + 4 (u*, T, p, D1 p)
struct PBwdSlot {
    cd y[PBB];
    double U[PWI + 1][PBB];
    cd op[MAXF + 2][PBB];
};

__global__ void __launch_bounds__(PBB) k_poisson_bwd_correct(PoisArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PBwdSlot* slots = reinterpret_cast<PBwdSlot*>(smem_raw);
    const int tx = threadIdx.x;
    const int plane_i = a.M1 * a.NK;
    const int e0 = a.e_begin + blockIdx.x * PBB + tx;
    const bool valid = e0 < a.e_end;
    const int e = valid ? e0 : a.e_end - 1;
    const int m = e / a.NK, kk = e % a.NK;
    const int ka = kk >= a.K ? kk - a.K : a.K - kk;
    const size_t P = a.P;
    const size_t plane = (size_t)plane_i;
    const int N = a.N_r;
    const double n = a.nm[m], kap = a.kap[kk];
    const bool m00 = (m == 0 && ka == 0);
    const double idt = 1.0 / a.dt;
    const double* Uf = a.U + (size_t)m * (a.K + 1) + ka;
    const bool have_p = a.p_dst != nullptr;
    const bool heated = a.nf == 4;
    // rows whose correction operands ride in the pipeline: jc = j + 4 for j in [0, N - 9]
    auto issue = [&](int j) {
        if (j >= 0) {
            PBwdSlot& s = slots[(N - 1 - j) % PIPE_PB];
            cpa16(&s.y[tx], a.G + (size_t)j * plane + e);
            if (j >= a.jaU && j < a.jbU) {
                const double* Ur = Uf + (size_t)(a.offUa + (PWI + 1) * (j - a.jaU)) * P;
#pragma unroll
                for (int i = 0; i <= PWI; ++i) cpa8(&s.U[i][tx], Ur + (size_t)i * P);
            }
            if (j <= N - NPT) {
                const size_t oc = (size_t)(j + NPT / 2) * plane + e;
                cpa16(&s.op[0][tx], a.W[0] + oc);
                cpa16(&s.op[1][tx], a.W[1] + oc);
                cpa16(&s.op[2][tx], a.W[2] + oc);
                if (a.copyT) cpa16(&s.op[3][tx], a.W[3] + oc);
                if (have_p) {
                    cpa16(&s.op[MAXF][tx], a.p + oc);
                    cpa16(&s.op[MAXF + 1][tx], a.DP + oc);
                }
            }
        }
        cpa_commit();
    };
    cd w[12];                                           // w[d] = phi_{j+d}, d = 0 .. 11 (shifted every row)
#pragma unroll
    for (int i = 0; i < 12; ++i) w[i] = mk(0.0, 0.0);
#pragma unroll
    for (int d = 0; d < PIPE_PB - 1; ++d) issue(N - 1 - d);
    for (int j = N - 1; j >= 0; --j) {
        cpa_wait<PIPE_PB - 2>();
        __syncthreads();
        issue(j - (PIPE_PB - 1));
        const PBwdSlot& s = slots[(N - 1 - j) % PIPE_PB];
        cd y = s.y[tx];
        // phi_j = (y_j - sum_{d=1..nu} U[j][d] phi_{j+d}) / pivot;  here w[d-1] = phi_{j+d}
        if (j >= a.jaU && j < a.jbU) {
#pragma unroll
            for (int d = PWI; d >= 1; --d) {
                const double u = s.U[d][tx];
                y.x = fma(-u, w[d - 1].x, y.x);
                y.y = fma(-u, w[d - 1].y, y.y);
            }
            y = s.U[0][tx] * y;
        } else {
            const int nu = a.hi[j] - j;
            const double* Ur = Uf + (size_t)a.offU[j] * P;
#pragma unroll
            for (int d = 12; d >= 1; --d) {
                if (d <= nu) {
                    const double u = Ur[(size_t)d * P];
                    y.x = fma(-u, w[d - 1].x, y.x);
                    y.y = fma(-u, w[d - 1].y, y.y);
                }
            }
            y = Ur[0] * y;
        }
#pragma unroll
        for (int q = 11; q > 0; --q) w[q] = w[q - 1];
        w[0] = y;
        // L5 at the rows jc whose stencil rows j .. j + 8 = w[0 .. 8] are now complete (wall rows: no stencil);
        // the regular row jc = j + 4 has its operands in the slot, rows next to the walls read them from HBM
        int c_hi = -1, c_lo = 0;
        if (j == N - 1) {
            c_hi = c_lo = N - 1;
        } else if (j <= N - NPT) {
            c_hi = (j == N - NPT) ? N - 2 : j + NPT / 2;
            c_lo = (j == 0) ? 0 : j + NPT / 2;
        }
        for (int jc = c_hi; jc >= c_lo; --jc) {
            const size_t oc = (size_t)jc * plane + e;
            const bool piped = (jc == j + NPT / 2) && (j <= N - NPT);
            const cd z = mk(0.0, 0.0);
            const cd ur = piped ? s.op[0][tx] : a.W[0][oc];
            const cd ut = piped ? s.op[1][tx] : a.W[1][oc];
            const cd uz = piped ? s.op[2][tx] : a.W[2][oc];
            const cd T = a.copyT ? (piped ? s.op[3][tx] : a.W[3][oc]) : z;
            const cd pr = have_p ? (piped ? s.op[MAXF][tx] : a.p[oc]) : z;
            const cd dp = have_p ? (piped ? s.op[MAXF + 1][tx] : a.DP[oc]) : z;
            cd phi = w[NPT / 2];
            if (!piped) {                                // phi_jc = w[jc - j], picked by an exact 0/1 blend (keeps w in registers)
                phi = mk(0.0, 0.0);
#pragma unroll
                for (int d = 0; d < NPT; ++d) {
                    const double sel = (d == jc - j) ? 1.0 : 0.0;
                    phi.x = fma(sel, w[d].x, phi.x);
                    phi.y = fma(sel, w[d].y, phi.y);
                }
            }
            cd gphi = mk(0.0, 0.0);
            if (jc != 0 && jc != N - 1) {
                const double* dd = a.D1 + jc * NPT;
#pragma unroll
                for (int l = 0; l < NPT; ++l) {
                    const double wt = __ldg(dd + l);
                    gphi.x = fma(wt, w[l].x, gphi.x);
                    gphi.y = fma(wt, w[l].y, gphi.y);
                }
            }
            if (valid) {
                const double nr = n * a.rinv[jc];
                cd o0 = ur - gphi;
                if (m00) o0 = mk(0.0, 0.0);
                a.dst[0][oc] = o0;
                a.dst[1][oc] = mk(ut.x + nr * phi.y, ut.y - nr * phi.x);          // - (i n / r) phi
                a.dst[2][oc] = mk(uz.x + kap * phi.y, uz.y - kap * phi.x);        // - i kappa phi
                if (a.copyT) a.dst[3][oc] = T;
                if (have_p) {
                    a.p_dst[oc] = mk(fma(idt, phi.x, pr.x), fma(idt, phi.y, pr.y));
                    a.DP_dst[oc] = mk(fma(idt, gphi.x, dp.x), fma(idt, gphi.y, dp.y));
                }
            }
        }
    }
    cpa_wait<0>();
    (void)heated;
}

// ------------------------------------------------------------------------------------------
static int alloc_factors(nsc_ctx* c, BandFactors& f, const BandShape& s) {
    if (f.L) return NSC_OK;
    f.nL = s.nL;
    f.nU = s.nU;
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, sizeof(double) * (s.nL ? s.nL : 1) * c->P);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMalloc(L factors)");
    c->allocs.push_back(p);
    f.L = (double*)p;
    e = cudaMalloc(&p, sizeof(double) * s.nU * c->P);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMalloc(U factors)");
    c->allocs.push_back(p);
    f.U = (double*)p;
    c->dev_bytes += (long long)(sizeof(double) * (s.nL + s.nU) * c->P);
    return NSC_OK;
}

static int run_factor(nsc_ctx* c, BandFactors& f, const BandShape& s, int kind, double coef, double shift) {
    int rc = alloc_factors(c, f, s);
    if (rc) return rc;
    FacArgs a{};
    a.band = kind == 0 ? c->t.L0 : c->t.Q;
    a.bcol0 = kind == 0 ? c->t.s0 : c->t.q0;
    a.bw = kind == 0 ? NPT : QW;
    a.D1 = c->t.D1;
    a.s0 = c->t.s0;
    a.rinv = c->t.rinv;
    a.nm = c->t.nm;
    a.kap = c->t.kap;
    a.lo = s.lo;
    a.hi = s.hi;
    a.offL = s.offL;
    a.offU = s.offU;
    a.L = f.L;
    a.U = f.U;
    a.N_r = c->N_r;
    a.K = c->K;
    a.P = c->P;
    a.kind = kind;
    a.coef = coef;
    a.shift = shift;
    prof_begin(c, NSC_K_FACTOR);
    k_factor<<<(c->P + 63) / 64, 64, 0, c->stream>>>(a);
    prof_end(c);
    NSC_CUDA(c, cudaGetLastError());
    return NSC_OK;
}

int ensure_factors(nsc_ctx* c, double dt) {
    int rc;
    if (!c->facP_ready) {
        if ((rc = run_factor(c, c->facP, c->shP, 1, 0.0, 0.0))) return rc;
        c->facP_ready = true;
    }
    if (c->fac_dt != dt) {
        const double coef = c->p.c * dt;
        if ((rc = run_factor(c, c->facH[0], c->shH, 0, coef, +1.0))) return rc;
        if ((rc = run_factor(c, c->facH[1], c->shH, 0, coef, -1.0))) return rc;
        if ((rc = run_factor(c, c->facH[2], c->shH, 0, coef, 0.0))) return rc;
        if (c->heated) {
            if (c->p.Pr == 1.0) {
                c->facT_shared = true;
            } else {
                c->facT_shared = false;
                if ((rc = run_factor(c, c->facH[3], c->shH, 0, coef / c->p.Pr, 0.0))) return rc;
            }
        }
        c->fac_dt = dt;
    }
    return NSC_OK;
}

// ------------------------------------------------------------------------------------------
// convergence norm of the iterated corrector (R16): acc[0] += sum |b - a|^2, acc[1] += sum |b|^2
__global__ void __launch_bounds__(256) k_diff_norm(const cd* a, const cd* b, size_t n, double* acc) {
    double d = 0.0, s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const cd x = a[i], y = b[i];
        const double dx = y.x - x.x, dy = y.y - x.y;
        d = fma(dx, dx, fma(dy, dy, d));
        s = fma(y.x, y.x, fma(y.y, y.y, s));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        d += __shfl_down_sync(0xffffffffu, d, o);
        s += __shfl_down_sync(0xffffffffu, s, o);
    }
    __shared__ double sd[8], ss[8];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) {
        sd[w] = d;
        ss[w] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double D = 0.0, S = 0.0;
        for (int i = 0; i < 8; ++i) {
            D += sd[i];
            S += ss[i];
        }
        atomicAdd(acc, D);
        atomicAdd(acc + 1, S);
    }
}

int launch_diff_norm(nsc_ctx* c, cd* const* a, cd* const* b, double* d_acc) {
    NSC_CUDA(c, cudaMemsetAsync(d_acc, 0, 2 * sizeof(double), c->stream));
    for (int i = 0; i < c->nf; ++i) {
        prof_begin(c, NSC_K_RECOMBINE);
        k_diff_norm<<<148 * 8, 256, 0, c->stream>>>(a[i], b[i], c->F, d_acc);
        prof_end(c);
        NSC_CUDA(c, cudaGetLastError());
    }
    return NSC_OK;
}

// ------------------------------------------------------------------------------------------
// NEXT-3 diagnostics.  k_nusselt: out[0..1] heat, out[2..3] torque Nusselt numbers at the
// inner / outer wall from the mean mode (0,0): Nu = d_r T r ln(eta);  Nu_w = r^3 d_r(u_theta / r) / (-2 B).
__global__ void k_nusselt(const cd* ut, const cd* T, const double* D1, const int* s0, const double* rinv, int N_r,
                          size_t plane, size_t col00, double ln_eta, double B, double* out) {
    const int t = threadIdx.x;
    if (t >= 4) return;
    const int j = (t & 1) ? N_r - 1 : 0;
    const cd* f = (t < 2) ? T : ut;
    double v = nan("");
    if (f) {
        double d = 0.0;
        for (int l = 0; l < NPT; ++l) d = fma(D1[j * NPT + l], f[(size_t)(s0[j] + l) * plane + col00].x, d);
        const double ri = rinv[j], r = 1.0 / ri;
        if (t < 2) {
            v = d * r * ln_eta;
        } else if (B != 0.0) {
            const double dw = d * ri - f[(size_t)j * plane + col00].x * ri * ri;
            v = r * r * r * dw / (-2.0 * B);
        }
    }
    out[t] = v;
}

// k_probe: acc += Re sum_k f(0,k) e^{i kappa z} + 2 Re sum_{m>=1,k} f(m,k) e^{i(n theta + kappa z)} at one radial node
__global__ void __launch_bounds__(256) k_probe(const cd* fj, const double* nm, const double* kap, int M1, int NK,
                                               double theta, double z, double* acc) {
    double s = 0.0;
    const int n = M1 * NK;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const int m = e / NK, kk = e % NK;
        double sn, cs;
        sincos(nm[m] * theta + kap[kk] * z, &sn, &cs);
        const cd v = fj[e];
        const double re = v.x * cs - v.y * sn;
        s += (m == 0) ? re : 2.0 * re;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    __shared__ double sh[8];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double S = 0.0;
        for (int i = 0; i < 8; ++i) S += sh[i];
        atomicAdd(acc, S);
    }
}

int launch_nusselt(nsc_ctx* c, double* d_out) {
    const double eta = c->p.eta;
    const double B = eta * (c->p.Re_i - eta * c->p.Re_o) / ((1.0 - eta) * (1.0 - eta * eta));
    prof_begin(c, NSC_K_DIV);
    k_nusselt<<<1, 32, 0, c->stream>>>(c->state[1], c->heated ? c->state[3] : nullptr, c->t.D1, c->t.s0, c->t.rinv,
                                        c->N_r, (size_t)c->M1 * c->NK, (size_t)c->K, log(eta), B, d_out);
    prof_end(c);
    NSC_CUDA(c, cudaGetLastError());
    return NSC_OK;
}

int launch_probe(nsc_ctx* c, const cd* field, int j, double theta, double z, double* d_acc) {
    NSC_CUDA(c, cudaMemsetAsync(d_acc, 0, sizeof(double), c->stream));
    const int n = c->M1 * c->NK;
    int blocks = (n + 255) / 256;
    if (blocks > 592) blocks = 592;
    prof_begin(c, NSC_K_DIV);
    k_probe<<<blocks, 256, 0, c->stream>>>(field + (size_t)j * n, c->t.nm, c->t.kap, c->M1, c->NK, theta, z, d_acc);
    prof_end(c);
    NSC_CUDA(c, cudaGetLastError());
    return NSC_OK;
}

// longest run [ja, jb) of rows whose lower (upper) width equals `width`; off = offL[ja] (offU[ja])
static void interior_run(const BandShape& s, bool lower, int width, int& ja, int& jb, int& off) {
    const int N = (int)s.h_lo.size();
    int best_a = 0, best_b = 0, cur = -1;
    for (int j = 0; j <= N; ++j) {
        const bool in = j < N && (lower ? j - s.h_lo[j] : s.h_hi[j] - j) == width;
        if (in && cur < 0) cur = j;
        if (!in && cur >= 0) {
            if (j - cur > best_b - best_a) {
                best_a = cur;
                best_b = j;
            }
            cur = -1;
        }
    }
    ja = best_a;
    jb = best_b;
    off = (best_b > best_a) ? (lower ? s.h_offL[best_a] : s.h_offU[best_a]) : 0;
}

int launch_substep(nsc_ctx* c, cd* const* E0, double w0, cd* const* E1, double w1, double dt, cd* const* dst,
                   cd* p_dst, cd* DP_dst) {
    int rc = ensure_factors(c, dt);
    if (rc) return rc;
    const int plane = c->M1 * c->NK;
    {
        FusedArgs fa{};
        for (int i = 0; i < c->nf; ++i) {
            fa.u[i] = c->state[i];
            fa.E0[i] = E0[i];
            fa.E1[i] = E1 ? E1[i] : nullptr;
            fa.W[i] = c->W[i];
            const BandFactors& bf = (i == 3 && c->facT_shared) ? c->facH[2] : c->facH[i];
            fa.L[i] = bf.L;
            fa.U[i] = bf.U;
        }
        fa.p = c->state[4];
        fa.G = c->G;
        fa.lo = c->shH.lo;
        fa.hi = c->shH.hi;
        fa.offL = c->shH.offL;
        fa.offU = c->shH.offU;
        fa.D1 = c->t.D1;
        fa.rinv = c->t.rinv;
        fa.nm = c->t.nm;
        fa.kap = c->t.kap;
        fa.s0 = c->t.s0;
        fa.N_r = c->N_r;
        fa.M1 = c->M1;
        fa.NK = c->NK;
        fa.K = c->K;
        fa.P = c->P;
        fa.nf = c->nf;
        fa.dt = dt;
        fa.c = c->p.c;
        fa.w0 = w0;
        fa.w1 = w1;
        fa.Re_i = c->p.Re_i;
        fa.Re_o = c->p.Re_o;
        fa.DP = c->DP;
        fa.offL4 = c->shH.h_offL[FWI];
        fa.offU4 = c->shH.h_offU[FWI];
        {   // per device, so set on every launch (a few microseconds)
            cudaFuncSetAttribute(k_rhs_fwd<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(PIPE_F * sizeof(FwdSlot<3>)));
            cudaFuncSetAttribute(k_rhs_fwd<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(PIPE_F * sizeof(FwdSlot<4>)));
            cudaFuncSetAttribute(k_bwd_div<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(PIPE_B * sizeof(BwdSlot<3>)));
            cudaFuncSetAttribute(k_bwd_div<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(PIPE_B * sizeof(BwdSlot<4>)));
        }
        PoisArgs pa{};
        pa.G = c->G;
        pa.L = c->facP.L;
        pa.U = c->facP.U;
        pa.lo = c->shP.lo;
        pa.hi = c->shP.hi;
        pa.offL = c->shP.offL;
        pa.offU = c->shP.offU;
        interior_run(c->shP, true, PWI, pa.jaL, pa.jbL, pa.offLa);
        interior_run(c->shP, false, PWI, pa.jaU, pa.jbU, pa.offUa);
        for (int i = 0; i < c->nf; ++i) {
            pa.W[i] = c->W[i];
            pa.dst[i] = dst[i];
        }
        pa.p = c->state[4];
        pa.p_dst = p_dst;
        pa.DP = c->DP;
        pa.DP_dst = DP_dst ? DP_dst : c->DP;
        pa.D1 = c->t.D1;
        pa.rinv = c->t.rinv;
        pa.nm = c->t.nm;
        pa.kap = c->t.kap;
        pa.s0 = c->t.s0;
        pa.N_r = c->N_r;
        pa.M1 = c->M1;
        pa.NK = c->NK;
        pa.K = c->K;
        pa.P = c->P;
        pa.nf = c->nf;
        pa.copyT = (c->nf == 4 && dst[3] != c->W[3]) ? 1 : 0;
        pa.dt = dt;
        {
            cudaFuncSetAttribute(k_poisson_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(PIPE_PF * sizeof(PFwdSlot)));
            cudaFuncSetAttribute(k_poisson_bwd_correct, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(PIPE_PB * sizeof(PBwdSlot)));
        }
        // The four sweeps of a block of modes depend only on each other, so the mode range is cut into slices
        // whose kernel chains run on separate streams: while one slice's sweep drains (a march has no work
        // left for the SMs its finished columns occupied), the next sweep of the other slice fills the machine.
        // With per-kernel profiling on, one slice on the caller's stream (the event brackets need one stream).
        const int nsl = (c->profiling || !c->slice_stream[0]) ? 1 : c->n_slices;
        // the window of modes (default: all); not w0 / w1: those are this function's weights of E0 and E1
        const int we_lo = (int)c->we0, we_hi = (int)c->we1;
        const int per = ((we_hi - we_lo + nsl - 1) / nsl + 127) / 128 * 128;   // multiple of every block width
        if (nsl > 1) {
            NSC_CUDA(c, cudaEventRecord(c->slice_ev[0], c->stream));
        }
        for (int sl = 0; sl < nsl; ++sl) {
            const int eb = we_lo + sl * per, ee = (eb + per < we_hi) ? eb + per : we_hi;
            if (eb >= ee) continue;
            cudaStream_t st = (nsl > 1) ? c->slice_stream[sl] : c->stream;
            if (nsl > 1) NSC_CUDA(c, cudaStreamWaitEvent(st, c->slice_ev[0], 0));
            fa.e_begin = pa.e_begin = eb;
            fa.e_end = pa.e_end = ee;
            const int ne = ee - eb;
            const int nb = (ne + PBK - 1) / PBK;
            prof_begin(c, NSC_K_RHS);
            if (c->nf == 3)
                k_rhs_fwd<3><<<nb, dim3(PBK, 3), PIPE_F * sizeof(FwdSlot<3>), st>>>(fa);
            else
                k_rhs_fwd<4><<<nb, dim3(PBK, 4), PIPE_F * sizeof(FwdSlot<4>), st>>>(fa);
            prof_end(c);
            NSC_CUDA(c, cudaGetLastError());
            prof_begin(c, NSC_K_HELMHOLTZ);
            if (c->nf == 3)
                k_bwd_div<3><<<nb, dim3(PBK, 4), PIPE_B * sizeof(BwdSlot<3>), st>>>(fa);
            else
                k_bwd_div<4><<<nb, dim3(PBK, 5), PIPE_B * sizeof(BwdSlot<4>), st>>>(fa);
            prof_end(c);
            NSC_CUDA(c, cudaGetLastError());
            prof_begin(c, NSC_K_POISSON);
            k_poisson_fwd<<<(ne + PBP - 1) / PBP, PBP, PIPE_PF * sizeof(PFwdSlot), st>>>(pa);
            prof_end(c);
            NSC_CUDA(c, cudaGetLastError());
            prof_begin(c, NSC_K_CORRECT);
            k_poisson_bwd_correct<<<(ne + PBB - 1) / PBB, PBB, PIPE_PB * sizeof(PBwdSlot), st>>>(pa);
            prof_end(c);
            NSC_CUDA(c, cudaGetLastError());
            if (nsl > 1) {
                NSC_CUDA(c, cudaEventRecord(c->slice_ev[1 + sl], st));
                NSC_CUDA(c, cudaStreamWaitEvent(c->stream, c->slice_ev[1 + sl], 0));
            }
        }
    }
    return NSC_OK;
}

}  // namespace nsc
