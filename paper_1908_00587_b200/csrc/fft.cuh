// fft.cuh -- register/shared-memory fp64 FFT building blocks for lengths N = 3 * 2^p.
//
// Used by the transform kernels of the nonlinear term (K-zinv, K-theta,
// K-zfwd; BASELINE.json north_star (a): "batched inverse real 2-D FFTs ... forward FFTs").
//
// A line of length N is transformed by TPL = N / E cooperating threads (E = 24 complex values
// held in registers per thread; E = 12 for N = 12).  A transform is one or three Stockham
// passes with radices (R1, R2, R3), R1 == R3, chosen so that every pass uses exactly E values
// per thread.  Between passes the values are exchanged through a padded shared-memory line.
// The first pass reads its operands and the last pass leaves its results in the SAME register
// layout:   x[u*R1 + t]  <->  line index  tau + u*TPL + t*(N/R1),   u < E/R1, t < R1
// which lets the callers fuse loads, point-wise products and stores around the transforms
// without extra shared-memory round trips.
//
// DIR = -1: X[k] = sum_n x[n] exp(-2 pi i n k / N);  DIR = +1: the conjugate kernel (unnormalised).
// Everything here is __host__ __device__ so the index arithmetic can be exercised on the CPU.
#pragma once

#ifdef __CUDACC__
#define NSC_HD __host__ __device__ __forceinline__
#else
#define NSC_HD inline
#endif

namespace nsc {

struct alignas(16) cd {
    double x, y;
};

NSC_HD cd mk(double a, double b) { cd r; r.x = a; r.y = b; return r; }
NSC_HD cd operator+(cd a, cd b) { return mk(a.x + b.x, a.y + b.y); }
NSC_HD cd operator-(cd a, cd b) { return mk(a.x - b.x, a.y - b.y); }
NSC_HD cd operator*(cd a, cd b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
NSC_HD cd operator*(double s, cd a) { return mk(s * a.x, s * a.y); }
NSC_HD cd conj(cd a) { return mk(a.x, -a.y); }
NSC_HD cd mul_i(cd a) { return mk(-a.y, a.x); }     // i * a
NSC_HD cd mul_mi(cd a) { return mk(a.y, -a.x); }    // -i * a
template <int DIR> NSC_HD cd mul_di(cd a) { return DIR > 0 ? mul_i(a) : mul_mi(a); }  // (DIR i) * a

// ---------------------------------------------------------------- small DFTs in registers
template <int DIR> NSC_HD void dft2(cd& a, cd& b) {
    cd t = a - b;
    a = a + b;
    b = t;
}

template <int DIR> NSC_HD void dft3(cd& a, cd& b, cd& c) {
    const double s3 = 0.86602540378443864676372317075294;   // sin(2 pi / 3)
    cd t1 = b + c;
    cd t2 = mk(a.x - 0.5 * t1.x, a.y - 0.5 * t1.y);
    cd t3 = mul_di<DIR>(s3 * (b - c));
    a = a + t1;
    b = t2 + t3;
    c = t2 - t3;
}

template <int DIR> NSC_HD void dft4(cd& a, cd& b, cd& c, cd& d) {
    cd s0 = a + c, d0 = a - c, s1 = b + d, d1 = mul_di<DIR>(b - d);
    a = s0 + s1;
    c = s0 - s1;
    b = d0 + d1;
    d = d0 - d1;
}

template <int DIR> NSC_HD void dft8(cd* x) {
    const double h = 0.70710678118654752440084436210485;    // 1 / sqrt(2)
    dft4<DIR>(x[0], x[2], x[4], x[6]);                      // even samples -> E0..E3 in x[0,2,4,6]
    dft4<DIR>(x[1], x[3], x[5], x[7]);                      // odd samples  -> O0..O3 in x[1,3,5,7]
    cd o1 = x[3], o2 = x[5], o3 = x[7];
    // W8^1 = (1 + DIR i)/sqrt2,  W8^2 = DIR i,  W8^3 = (-1 + DIR i)/sqrt2
    o1 = h * (o1 + mul_di<DIR>(o1));
    o2 = mul_di<DIR>(o2);
    o3 = h * (mul_di<DIR>(o3) - o3);
    cd e0 = x[0], e1 = x[2], e2 = x[4], e3 = x[6], o0 = x[1];
    x[0] = e0 + o0;
    x[4] = e0 - o0;
    x[1] = e1 + o1;
    x[5] = e1 - o1;
    x[2] = e2 + o2;
    x[6] = e2 - o2;
    x[3] = e3 + o3;
    x[7] = e3 - o3;
}

#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int inv_mod(int a, int m) {
    for (int i = 1; i < m; ++i)
        if ((a * i) % m == 1) return i;
    return 1;
}

template <int R, int DIR> struct Dft;
template <int DIR> struct Dft<2, DIR> { static NSC_HD void run(cd* x) { dft2<DIR>(x[0], x[1]); } };
template <int DIR> struct Dft<3, DIR> { static NSC_HD void run(cd* x) { dft3<DIR>(x[0], x[1], x[2]); } };
template <int DIR> struct Dft<4, DIR> { static NSC_HD void run(cd* x) { dft4<DIR>(x[0], x[1], x[2], x[3]); } };
template <int DIR> struct Dft<8, DIR> { static NSC_HD void run(cd* x) { dft8<DIR>(x); } };

// R = 3 * N2, gcd(3, N2) = 1: Good-Thomas prime-factor mapping (no twiddles between the factors):
//   n = (N2 n1 + 3 n2) mod R,  k = (N2 a k1 + 3 b k2) mod R,  a = N2^-1 mod 3,  b = 3^-1 mod N2.
template <int N2, int DIR> struct DftPfa3 {
    static constexpr int R = 3 * N2;
    static NSC_HD void run(cd* x) {
        cd t[N2][3];
#pragma unroll
        for (int n2 = 0; n2 < N2; ++n2)
#pragma unroll
            for (int n1 = 0; n1 < 3; ++n1) t[n2][n1] = x[(N2 * n1 + 3 * n2) % R];
#pragma unroll
        for (int n2 = 0; n2 < N2; ++n2) dft3<DIR>(t[n2][0], t[n2][1], t[n2][2]);
        constexpr int a = inv_mod(N2 % 3, 3), b = inv_mod(3 % N2, N2);
#pragma unroll
        for (int k1 = 0; k1 < 3; ++k1) {
            cd c[N2];
#pragma unroll
            for (int n2 = 0; n2 < N2; ++n2) c[n2] = t[n2][k1];
            Dft<N2, DIR>::run(c);
#pragma unroll
            for (int k2 = 0; k2 < N2; ++k2) x[(N2 * a * k1 + 3 * b * k2) % R] = c[k2];
        }
    }
};
template <int DIR> struct Dft<6, DIR> { static NSC_HD void run(cd* x) { DftPfa3<2, DIR>::run(x); } };
template <int DIR> struct Dft<12, DIR> { static NSC_HD void run(cd* x) { DftPfa3<4, DIR>::run(x); } };
template <int DIR> struct Dft<24, DIR> { static NSC_HD void run(cd* x) { DftPfa3<8, DIR>::run(x); } };

// ---------------------------------------------------------------- plans
template <int N> struct Plan;
template <> struct Plan<12>   { static constexpr int TPL = 1,  NP = 1, R1 = 12, R2 = 1,  R3 = 12; };
template <> struct Plan<24>   { static constexpr int TPL = 1,  NP = 1, R1 = 24, R2 = 1,  R3 = 24; };
template <> struct Plan<48>   { static constexpr int TPL = 2,  NP = 3, R1 = 4,  R2 = 3,  R3 = 4; };
template <> struct Plan<96>   { static constexpr int TPL = 4,  NP = 3, R1 = 4,  R2 = 6,  R3 = 4; };
template <> struct Plan<192>  { static constexpr int TPL = 8,  NP = 3, R1 = 8,  R2 = 3,  R3 = 8; };
template <> struct Plan<384>  { static constexpr int TPL = 16, NP = 3, R1 = 8,  R2 = 6,  R3 = 8; };
template <> struct Plan<768>  { static constexpr int TPL = 32, NP = 3, R1 = 8,  R2 = 12, R3 = 8; };
template <> struct Plan<1536> { static constexpr int TPL = 64, NP = 3, R1 = 8,  R2 = 24, R3 = 8; };

template <int N> struct Geo {
    using P = Plan<N>;
    static constexpr int TPL = P::TPL;
    static constexpr int E = N / TPL;                  // complex values per thread
    static constexpr int R1 = P::R1;
    static constexpr int BPT1 = E / R1;                // first/last-pass butterflies per thread
    static constexpr int PADDED = N + (N >> 3);        // shared-memory line length (elements)
    // line index of register slot e = u*R1 + t of thread tau (first-pass input == last-pass output)
    static NSC_HD int idx(int e, int tau) { return tau + (e / R1) * TPL + (e % R1) * (N / R1); }
};

NSC_HD int pad_idx(int i) { return i + (i >> 3); }

// ---------------------------------------------------------------- one Stockham pass, in pieces
template <int N, int R, int TPL> NSC_HD void pass_load(cd* x, const cd* buf, int tau) {
    constexpr int BPT = N / R / TPL;
#pragma unroll
    for (int u = 0; u < BPT; ++u)
#pragma unroll
        for (int t = 0; t < R; ++t) x[u * R + t] = buf[pad_idx(tau + u * TPL + t * (N / R))];
}

// tw[i] = exp(-2 pi i * i / N), i < N
template <int N, int R, int NS, int TPL, int DIR> NSC_HD void pass_compute(cd* x, const cd* tw, int tau) {
    constexpr int BPT = N / R / TPL;
#pragma unroll
    for (int u = 0; u < BPT; ++u) {
        if (NS > 1) {
            const int k = (tau + u * TPL) % NS;
#pragma unroll
            for (int t = 1; t < R; ++t) {
                cd w = tw[k * t * (N / (NS * R))];
                if (DIR > 0) w = conj(w);
                x[u * R + t] = x[u * R + t] * w;
            }
        }
        Dft<R, DIR>::run(x + u * R);
    }
}

template <int N, int R, int NS, int TPL> NSC_HD void pass_store(const cd* x, cd* buf, int tau) {
    constexpr int BPT = N / R / TPL;
#pragma unroll
    for (int u = 0; u < BPT; ++u) {
        const int b = tau + u * TPL;
        const int k = b % NS;
        const int base = (b - k) * R + k;
#pragma unroll
        for (int t = 0; t < R; ++t) buf[pad_idx(base + t * NS)] = x[u * R + t];
    }
}

// The four phases of a three-pass transform; the caller separates them by a barrier over the
// TPL threads of the line (phase A may only start once every thread has finished reading the
// line buffer in the previous phase D / epilogue).
template <int N, int DIR> NSC_HD void fft_phase_a(cd* x, cd* buf, const cd* tw, int tau) {
    using P = Plan<N>;
    pass_compute<N, P::R1, 1, P::TPL, DIR>(x, tw, tau);
    pass_store<N, P::R1, 1, P::TPL>(x, buf, tau);
}
template <int N, int DIR> NSC_HD void fft_phase_b(cd* x, const cd* buf, int tau) {
    using P = Plan<N>;
    pass_load<N, P::R2, P::TPL>(x, buf, tau);
}
template <int N, int DIR> NSC_HD void fft_phase_c(cd* x, cd* buf, const cd* tw, int tau) {
    using P = Plan<N>;
    pass_compute<N, P::R2, P::R1, P::TPL, DIR>(x, tw, tau);
    pass_store<N, P::R2, P::R1, P::TPL>(x, buf, tau);
}
template <int N, int DIR> NSC_HD void fft_phase_d(cd* x, const cd* buf, const cd* tw, int tau) {
    using P = Plan<N>;
    pass_load<N, P::R3, P::TPL>(x, buf, tau);
    pass_compute<N, P::R3, P::R1 * P::R2, P::TPL, DIR>(x, tw, tau);
}

#ifdef __CUDACC__
// Barrier over the threads that share one line buffer.
template <int TPL> __device__ __forceinline__ void line_sync() {
    if (TPL <= 32)
        __syncwarp();
    else
        __syncthreads();
}

// Full transform of one line: x (first-pass layout) -> x (same layout), through buf.
template <int N, int DIR> __device__ __forceinline__ void fft_line(cd* x, cd* buf, const cd* tw, int tau) {
    using P = Plan<N>;
    if constexpr (P::NP == 1) {
        Dft<P::R1, DIR>::run(x);
    } else {
        fft_phase_a<N, DIR>(x, buf, tw, tau);
        line_sync<P::TPL>();
        fft_phase_b<N, DIR>(x, buf, tau);
        line_sync<P::TPL>();
        fft_phase_c<N, DIR>(x, buf, tw, tau);
        line_sync<P::TPL>();
        fft_phase_d<N, DIR>(x, buf, tw, tau);
        line_sync<P::TPL>();
    }
}
#endif

}  // namespace nsc
