// nonlinear_kernels.cuh -- the three transform kernels of the pseudospectral nonlinear term
// (DESIGN.md steps N1-N6; BASELINE.json north_star (a)):
//
//   k_zinv   N1 (d/dz = i kappa, d/dr = 9-point stencil, both applied to the spectral lines)
//            + N2 zero-padded inverse z-FFT.  One line = one (j, m) pair of one field; output
//            [q][jl][z][m] with m fastest, so that k_theta streams along m.
//   k_theta  N1 (d/dtheta = i n) + N3 inverse theta-FFT (Hermitian lines, two real lines packed
//            in one complex transform) + N4 products + N5 forward theta-FFT and truncation.
//            One line = one (j, z) point-line; the physical-space fields live only in
//            registers and shared memory.
//   k_zfwd   N6 forward z-FFT, truncation to |k| <= K, scaling 1/(N_theta N_z), buoyancy.
//
// Layout of the half-transformed work arrays: complex128 [j_local][q][N_z][MP] (the lines of one radial level are neighbours), MP = M+1 rounded up
// to a multiple of 8, radial index local to the chunk.
#pragma once
#include "nsc_internal.h"

namespace nsc {

struct NlArgs {
    const cd* f[MAXF];     // spectral input fields [N_r][M1][NK]
    cd* out[MAXF];         // spectral outputs N_r, N_theta, N_z, N_T
    cd* zbuf;              // [JC][3 nf][Nz][MP]: q = 3 f + {0: f, 1: dz f, 2: dr f}
    cd* tbuf;              // [JC][nf][Nz][MP]
    const double* D1;
    const int* s0;
    const double* rinv;
    const double* nm;
    const double* kap;
    const cd* tw;          // twiddles of the transform length of the kernel
    int N_r, M1, NK, K, M, MP, JC, Nz, j0, nj, nf;
    double scale, buoy;
    unsigned long long* cfl;   // [N_r][3] running maxima of |u_r|, |u_theta|, |u_z| per radial level, as the ordered
                           // bit patterns of non-negative doubles (theta kernels, atomicMax); null: not wanted
};

// largest of v >= 0 over the TPL threads of a line (a whole warp if TPL >= 32), merged into *dst by atomicMax
template <int TPL> __device__ __forceinline__ void line_atomic_max(unsigned long long* dst, double v, int tau) {
    unsigned long long b = (unsigned long long)__double_as_longlong(v);
#pragma unroll
    for (int o = (TPL < 32 ? TPL : 32) / 2; o > 0; o >>= 1) {
        const unsigned long long c = __shfl_xor_sync(0xffffffffu, b, o);
        b = c > b ? c : b;
    }
    if ((TPL >= 32 ? (int)(threadIdx.x & 31) : tau) == 0) atomicMax(dst, b);
}

// ------------------------------------------------------------------------------------------
template <int NZ> struct ZCfg {
    static constexpr int TPL = Plan<NZ>::TPL;
    static constexpr int LPC = TPL >= 64 ? 2 : (TPL == 32 ? 4 : 128 / TPL);
    static constexpr int THREADS = LPC * TPL;
    static constexpr size_t SMEM = sizeof(cd) * (NZ + (size_t)LPC * Geo<NZ>::PADDED);
};

// axial mode of padded-line index i, or NOK if the bin is zero padding
__device__ __forceinline__ bool z_bin_to_k(int i, int NZ, int K, int& kk) {
    if (i <= K) {
        kk = i + K;
        return true;
    }
    if (i >= NZ - K) {
        kk = i - NZ + K;
        return true;
    }
    return false;
}

template <int NZ>
__global__ void __launch_bounds__(ZCfg<NZ>::THREADS) k_zinv(NlArgs a) {
    using G = Geo<NZ>;
    constexpr int TPL = G::TPL, E = G::E, LPC = ZCfg<NZ>::LPC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    cd* buf = tw + NZ + (threadIdx.x / TPL) * G::PADDED;
    for (int i = threadIdx.x; i < NZ; i += blockDim.x) tw[i] = a.tw[i];
    __syncthreads();
    const int tau = threadIdx.x % TPL;
    const int nlines = a.nj * a.M1;
    int line = blockIdx.x * LPC + threadIdx.x / TPL;
    const bool valid = line < nlines;
    if (!valid) line = nlines - 1;
    const int jl = line / a.M1, m = line % a.M1, j = a.j0 + jl;
    const int fi = blockIdx.y;
    const size_t plane = (size_t)a.M1 * a.NK;
    const cd* src = a.f[fi] + (size_t)j * plane + (size_t)m * a.NK;
    const size_t zstride = a.MP;
    cd x[E];
    // ---- q = 0: f itself
#pragma unroll
    for (int e = 0; e < E; ++e) {
        int kk;
        x[e] = z_bin_to_k(G::idx(e, tau), NZ, a.K, kk) ? src[kk] : mk(0.0, 0.0);
    }
    fft_line<NZ, +1>(x, buf, tw, tau);
    {
        cd* dst = a.zbuf + ((size_t)jl * 3 * a.nf + (3 * fi + 0)) * NZ * zstride + m;
        if (valid)
#pragma unroll
            for (int e = 0; e < E; ++e) dst[(size_t)G::idx(e, tau) * zstride] = x[e];
    }
    // ---- q = 1: d/dz -> i kappa f
#pragma unroll
    for (int e = 0; e < E; ++e) {
        int kk;
        if (z_bin_to_k(G::idx(e, tau), NZ, a.K, kk))
            x[e] = a.kap[kk] * mul_i(src[kk]);
        else
            x[e] = mk(0.0, 0.0);
    }
    fft_line<NZ, +1>(x, buf, tw, tau);
    {
        cd* dst = a.zbuf + ((size_t)jl * 3 * a.nf + (3 * fi + 1)) * NZ * zstride + m;
        if (valid)
#pragma unroll
            for (int e = 0; e < E; ++e) dst[(size_t)G::idx(e, tau) * zstride] = x[e];
    }
    // ---- q = 2: d/dr -> sum_l D1[j][l] f[s0[j] + l]
    {
        const int s = a.s0[j];
        double w[NPT];
#pragma unroll
        for (int l = 0; l < NPT; ++l) w[l] = a.D1[j * NPT + l];
        const cd* base = a.f[fi] + (size_t)s * plane + (size_t)m * a.NK;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            int kk;
            cd acc = mk(0.0, 0.0);
            if (z_bin_to_k(G::idx(e, tau), NZ, a.K, kk)) {
#pragma unroll
                for (int l = 0; l < NPT; ++l) {
                    cd v = base[(size_t)l * plane + kk];
                    acc.x = fma(w[l], v.x, acc.x);
                    acc.y = fma(w[l], v.y, acc.y);
                }
            }
            x[e] = acc;
        }
    }
    fft_line<NZ, +1>(x, buf, tw, tau);
    {
        cd* dst = a.zbuf + ((size_t)jl * 3 * a.nf + (3 * fi + 2)) * NZ * zstride + m;
        if (valid)
#pragma unroll
            for (int e = 0; e < E; ++e) dst[(size_t)G::idx(e, tau) * zstride] = x[e];
    }
}

template <int NZ>
__global__ void __launch_bounds__(ZCfg<NZ>::THREADS) k_zfwd(NlArgs a) {
    using G = Geo<NZ>;
    constexpr int TPL = G::TPL, E = G::E, LPC = ZCfg<NZ>::LPC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    cd* buf = tw + NZ + (threadIdx.x / TPL) * G::PADDED;
    for (int i = threadIdx.x; i < NZ; i += blockDim.x) tw[i] = a.tw[i];
    __syncthreads();
    const int tau = threadIdx.x % TPL;
    const int nlines = a.nj * a.M1;
    int line = blockIdx.x * LPC + threadIdx.x / TPL;
    const bool valid = line < nlines;
    if (!valid) line = nlines - 1;
    const int jl = line / a.M1, m = line % a.M1, j = a.j0 + jl;
    const int fi = blockIdx.y;
    const size_t zstride = a.MP;
    const cd* src = a.tbuf + ((size_t)jl * a.nf + fi) * NZ * zstride + m;
    cd x[E];
#pragma unroll
    for (int e = 0; e < E; ++e) x[e] = src[(size_t)G::idx(e, tau) * zstride];
    fft_line<NZ, -1>(x, buf, tw, tau);
    const size_t off = ((size_t)j * a.M1 + m) * a.NK;
    cd* dst = a.out[fi] + off;
    const bool add_buoy = (fi == 2) && (a.buoy != 0.0);
    const cd* Th = add_buoy ? a.f[3] + off : nullptr;
    if (valid)
#pragma unroll
        for (int e = 0; e < E; ++e) {
            int kk;
            if (z_bin_to_k(G::idx(e, tau), NZ, a.K, kk)) {
                cd v = a.scale * x[e];
                if (add_buoy) {
                    cd t = Th[kk];
                    v.x = fma(a.buoy, t.x, v.x);
                    v.y = fma(a.buoy, t.y, v.y);
                }
                dst[kk] = v;
            }
        }
}

// ------------------------------------------------------------------------------------------
template <int NT> struct TCfg {
    static constexpr int TPL = Plan<NT>::TPL;
    static constexpr int LPC = TPL >= 64 ? 3 : (TPL == 32 ? 6 : 128 / TPL);
    static constexpr int THREADS = LPC * TPL;
    // per line: one padded complex work line + three real physical-space lines (U_r, U_theta, U_z)
    static constexpr size_t LINE_BYTES = sizeof(cd) * Geo<NT>::PADDED + sizeof(double) * 3 * NT;
    static constexpr size_t SMEM = sizeof(cd) * NT + (size_t)LPC * LINE_BYTES;
};

// Registers <- Z[i] = G_X(m) + i G_Y(m) with G(m) = mult * line[m] (m >= 0), G(-m) = conj(G(m)),
// G(0) real (the m = 0 line contributes its real part, R6); mult = 1 or i n_m (d/dtheta).
template <int NT>
__device__ __forceinline__ void load_pair(cd* x, const cd* X, bool dX, const cd* Y, bool dY, const double* nm,
                                          int M, int tau) {
    using G = Geo<NT>;
#pragma unroll
    for (int e = 0; e < G::E; ++e) {
        const int i = G::idx(e, tau);
        int m;
        bool neg;
        if (i <= M) {
            m = i;
            neg = false;
        } else if (i >= NT - M) {
            m = NT - i;
            neg = true;
        } else {
            x[e] = mk(0.0, 0.0);
            continue;
        }
        const double n = nm[m];
        cd gx = X[m];
        if (dX) gx = n * mul_i(gx);
        cd gy = mk(0.0, 0.0);
        if (Y) {
            gy = Y[m];
            if (dY) gy = n * mul_i(gy);
        }
        if (m == 0) {
            gx.y = 0.0;
            gy.y = 0.0;
        }
        if (neg) {
            gx.y = -gx.y;
            gy.y = -gy.y;
        }
        x[e] = mk(gx.x - gy.y, gx.y + gy.x);
    }
}

// Forward transform of the packed pair (a + i b), split into the two Hermitian half-lines and
// truncated to m <= M:  A[m] = (Z[m] + conj Z[N-m]) / 2,  B[m] = (Z[m] - conj Z[N-m]) / (2 i).
template <int NT>
__device__ __forceinline__ void forward_pair(cd* x, cd* buf, const cd* tw, int tau, cd* outA, cd* outB, int M,
                                             bool valid) {
    using G = Geo<NT>;
    fft_line<NT, -1>(x, buf, tw, tau);
#pragma unroll
    for (int e = 0; e < G::E; ++e) buf[pad_idx(G::idx(e, tau))] = x[e];
    line_sync<G::TPL>();
    if (valid)
        for (int m = tau; m <= M; m += G::TPL) {
            cd zp = buf[pad_idx(m)];
            cd zm = conj(buf[pad_idx(m == 0 ? 0 : NT - m)]);
            outA[m] = 0.5 * (zp + zm);
            if (outB) outB[m] = 0.5 * mul_mi(zp - zm);
        }
    line_sync<G::TPL>();
}

template <int NT, int NF>
__global__ void __launch_bounds__(TCfg<NT>::THREADS) k_theta(NlArgs a) {
    using G = Geo<NT>;
    constexpr int TPL = G::TPL, E = G::E, LPC = TCfg<NT>::LPC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    unsigned char* lbase = smem_raw + sizeof(cd) * NT + (size_t)(threadIdx.x / TPL) * TCfg<NT>::LINE_BYTES;
    cd* buf = reinterpret_cast<cd*>(lbase);
    double* Ub = reinterpret_cast<double*>(lbase + sizeof(cd) * G::PADDED);   // [3][E][TPL], thread-private slots
    for (int i = threadIdx.x; i < NT; i += blockDim.x) tw[i] = a.tw[i];
    __syncthreads();
    const int tau = threadIdx.x % TPL;
    const int nlines = a.nj * a.Nz;
    int line = blockIdx.x * LPC + threadIdx.x / TPL;
    const bool valid = line < nlines;
    if (!valid) line = nlines - 1;
    const int jl = line / a.Nz, z = line % a.Nz;
    const double ri = a.rinv[a.j0 + jl];
    const size_t qstride = (size_t)a.Nz * a.MP;
    const size_t loff = ((size_t)jl * 3 * a.nf * a.Nz + z) * a.MP;       // line (j, z) of q = 0 in zbuf
    const size_t loff_t = ((size_t)jl * a.nf * a.Nz + z) * a.MP;          // ... in tbuf
    const int M = a.M;
    // A_f = plain, B_f = d/dz, C_f = d/dr half-transformed lines of field f at this (j, z)
#define LINE_A(f) (a.zbuf + (size_t)(3 * (f) + 0) * qstride + loff)
#define LINE_B(f) (a.zbuf + (size_t)(3 * (f) + 1) * qstride + loff)
#define LINE_C(f) (a.zbuf + (size_t)(3 * (f) + 2) * qstride + loff)
#define LINE_O(f) (a.tbuf + (size_t)(f) * qstride + loff_t)
#define UB(c, e) Ub[((c) * E + (e)) * TPL + tau]
    cd x[E];
    double acc0[E], acc1[E];
    // P0: (u_r, u_theta)
    load_pair<NT>(x, LINE_A(0), false, LINE_A(1), false, a.nm, M, tau);
    fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        UB(0, e) = x[e].x;
        UB(1, e) = x[e].y;
    }
    if (a.cfl) {                                           // per-level maxima for the CFL rate (step-size control)
        double m0 = 0.0, m1 = 0.0;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            m0 = fmax(m0, fabs(x[e].x));
            m1 = fmax(m1, fabs(x[e].y));
        }
        line_atomic_max<TPL>(a.cfl + 3 * (a.j0 + jl), m0, tau);
        line_atomic_max<TPL>(a.cfl + 3 * (a.j0 + jl) + 1, m1, tau);
    }
    // P1: (u_z, d_r u_r)
    load_pair<NT>(x, LINE_A(2), false, LINE_C(0), false, a.nm, M, tau);
    fft_line<NT, +1>(x, buf, tw, tau);
    if (a.cfl) {
        double m2 = 0.0;
#pragma unroll
        for (int e = 0; e < E; ++e) m2 = fmax(m2, fabs(x[e].x));
        line_atomic_max<TPL>(a.cfl + 3 * (a.j0 + jl) + 2, m2, tau);
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        UB(2, e) = x[e].x;
        acc0[e] = UB(0, e) * x[e].y;
    }
    // P2: (d_theta u_r, d_z u_r);  N_r = -(u.grad u_r - u_theta^2 / r)
    load_pair<NT>(x, LINE_A(0), true, LINE_B(0), false, a.nm, M, tau);
    fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double utr = UB(1, e) * ri;
        double s = fma(utr, x[e].x, acc0[e]);
        s = fma(UB(2, e), x[e].y, s);
        s = fma(-utr, UB(1, e), s);
        acc0[e] = -s;
    }
    // P3: (d_r u_theta, d_theta u_theta)
    load_pair<NT>(x, LINE_C(1), false, LINE_A(1), true, a.nm, M, tau);
    fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double utr = UB(1, e) * ri;
        acc1[e] = fma(utr, x[e].y, UB(0, e) * x[e].x);
    }
    // P4: (d_z u_theta, d_r u_z);  N_theta = -(u.grad u_theta + u_r u_theta / r)
    double acc2[E];
    load_pair<NT>(x, LINE_B(1), false, LINE_C(2), false, a.nm, M, tau);
    fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double utr = UB(1, e) * ri;
        double s = fma(UB(2, e), x[e].x, acc1[e]);
        s = fma(UB(0, e), utr, s);
        acc1[e] = -s;
        acc2[e] = UB(0, e) * x[e].y;
    }
    // forward (N_r, N_theta)
#pragma unroll
    for (int e = 0; e < E; ++e) x[e] = mk(acc0[e], acc1[e]);
    forward_pair<NT>(x, buf, tw, tau, LINE_O(0), LINE_O(1), M, valid);
    // P5: (d_theta u_z, d_z u_z);  N_z = -(u.grad u_z)   (buoyancy is added in k_zfwd)
    load_pair<NT>(x, LINE_A(2), true, LINE_B(2), false, a.nm, M, tau);
    fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double utr = UB(1, e) * ri;
        double s = fma(utr, x[e].x, acc2[e]);
        s = fma(UB(2, e), x[e].y, s);
        acc2[e] = -s;
    }
    if (NF == 3) {
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = mk(acc2[e], 0.0);
        forward_pair<NT>(x, buf, tw, tau, LINE_O(2), nullptr, M, valid);
    } else {
        // P6: (d_r T, d_theta T);  P7: (d_z T, -);  N_T = -(u.grad T)
        load_pair<NT>(x, LINE_C(3), false, LINE_A(3), true, a.nm, M, tau);
        fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double utr = UB(1, e) * ri;
            acc0[e] = fma(utr, x[e].y, UB(0, e) * x[e].x);
        }
        load_pair<NT>(x, LINE_B(3), false, nullptr, false, a.nm, M, tau);
        fft_line<NT, +1>(x, buf, tw, tau);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            double s = fma(UB(2, e), x[e].x, acc0[e]);
            x[e] = mk(acc2[e], -s);
        }
        forward_pair<NT>(x, buf, tw, tau, LINE_O(2), LINE_O(3), M, valid);
    }
#undef LINE_A
#undef LINE_B
#undef LINE_C
#undef LINE_O
#undef UB
}

// ------------------------------------------------------------------------------------------
// per-length launchers (one translation unit per length, see nonlinear_inst.cu)
template <int N> int launch_zinv_n(const NlArgs& a, cudaStream_t st);
template <int N> int launch_zfwd_n(const NlArgs& a, cudaStream_t st);
template <int N> int launch_theta_n(const NlArgs& a, cudaStream_t st);

#define NSC_DECLARE_LEN(N)                                         \
    int launch_zinv_##N(const NlArgs& a, cudaStream_t st);         \
    int launch_zfwd_##N(const NlArgs& a, cudaStream_t st);         \
    int launch_theta_##N(const NlArgs& a, cudaStream_t st);
NSC_DECLARE_LEN(12)
NSC_DECLARE_LEN(24)
NSC_DECLARE_LEN(48)
NSC_DECLARE_LEN(96)
NSC_DECLARE_LEN(192)
#undef NSC_DECLARE_LEN

}  // namespace nsc
