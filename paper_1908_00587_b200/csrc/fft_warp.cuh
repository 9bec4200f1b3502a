// fft_warp.cuh -- two-pass fp64 FFTs of length N = NA x 32 (NA = 24: N = 768, NA = 12: N = 384) for one warp,
// and of length 1536 = 2 x 768 for a pair of warps.
//
// The long workloads (BASELINE.json configs[3]: 768 x 768 physical grid per radial node, configs[2]: 384 x 384)
// spend their time in these transforms.  With 24 complex values per thread the generic
// three-pass plan of fft.cuh exchanges every line twice through shared memory and is bound by the shared-memory
// crossbar (128 B/clk/SM), not by the DFMA pipe.  Here a line crosses shared memory ONCE, and a warp always
// carries 24 x 32 values: one line of 768 or LPW = 2 lines of 384.
//
//   "S" (spectral-side) layout : 32 lanes x 24 values; register t of lane tau holds index tau + 32 (t % NA) of
//                                line t / NA
//   "P" (physical-side) layout : 24 lanes x 32 values; lane a holds line a / NA, register e holds index
//                                (a % NA) + NA p(e),  p(e) = (e >> 3) + 4 (e & 7)  (register order left by the
//                                radix-32 butterfly; a static permutation, never materialised)
//
//   s2p :  S -> P     n = 32 n1 + tau,  k = k1 + NA k2
//          pass A  lane tau: DFT-NA over n1 per line (Good-Thomas 3 x 2^q, no inner twiddles), times W_N^(tau k1)
//          exchange through a [24][33] complex matrix (row = (line, k1) = a, column = tau; stride 33 keeps
//          both the column-wise 16-byte stores and the row-wise 16-byte loads conflict free)
//          pass B  lane a < 24: DFT-32 over tau (4 x 8 with W_32 constants)
//   p2s :  P -> S     n = k1 + NA n2,  k = 32 k1' + tau      (the mirror image)
//
// Lanes 24..31 idle through the radix-32 halves (they recompute lane 23's butterfly and store nothing).
// X[k] = sum_n x[n] exp(DIR 2 pi i n k / N), unnormalised.
#pragma once
#include "fft.cuh"

namespace nsc {
namespace fw {

constexpr int NB = 32;            // radix of the pass on the P side = lanes on the S side
constexpr int NV = 24;            // values per lane on the S side = lanes on the P side
constexpr int XS = 33;            // row stride (complex) of the exchange matrix and the twiddle table
constexpr int XBUF = NV * XS;     // complex elements of one exchange matrix (12 672 bytes)

NSC_HD int p_of(int e) { return (e >> 3) + 4 * (e & 7); }

template <int NA_> struct WGeo {
    static constexpr int NA = NA_;            // radix of the pass on the S side
    static constexpr int N = NA * NB;         // line length
    static constexpr int LPW = NV / NA;       // lines per warp
    static constexpr int NMAX = N / 3;        // largest mode count of the 3/2 rule
    // index within its line of register e of lane a (P layout), of register t of lane tau (S layout)
    static NSC_HD int p_idx(int e, int a) { return (a % NA) + NA * p_of(e); }
    static NSC_HD int s_idx(int t, int tau) { return tau + NB * (t % NA); }
    // S-layout slot tt = t % NA can hold a non-zero spectral bin when the mode count is <= NMAX:
    // bins 0..NMAX (tt <= NMAX / 32) and bins N - NMAX..N - 1 (tt >= NA - NMAX / 32)
    static NSC_HD bool slot_pos(int tt) { return tt <= NMAX / NB; }
    static NSC_HD bool slot_neg(int tt) { return tt >= NA - NMAX / NB; }
    static NSC_HD bool slot_live(int tt) { return slot_pos(tt) || slot_neg(tt); }
};

// cos / sin of 2 pi e / 32, correctly rounded
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr double cos32(int e) {
    e &= 31;
    if (e > 16) e = 32 - e;          // cos is even
    bool neg = false;
    if (e > 8) {
        e = 16 - e;                  // cos(pi - x) = -cos(x)
        neg = true;
    }
    double c = e == 0   ? 1.0
               : e == 1 ? 0.98078528040323044912618223613424
               : e == 2 ? 0.92387953251128675612818318939679
               : e == 3 ? 0.83146961230254523707878837761791
               : e == 4 ? 0.70710678118654752440084436210485
               : e == 5 ? 0.55557023301960222474283081394853
               : e == 6 ? 0.38268343236508977172845998403040
               : e == 7 ? 0.19509032201612826784828486847702
                        : 0.0;
    return neg ? -c : c;
}
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr double sin32(int e) { return cos32(e - 8); }

// a * exp(DIR 2 pi i E / 32)
template <int DIR, int E> NSC_HD cd mul_w32(cd a) {
    constexpr int e = ((DIR > 0 ? E : -E) % 32 + 32) % 32;
    if constexpr (e == 0) {
        return a;
    } else if constexpr (e == 8) {
        return mul_i(a);
    } else if constexpr (e == 16) {
        return mk(-a.x, -a.y);
    } else if constexpr (e == 24) {
        return mul_mi(a);
    } else if constexpr (e % 8 == 4) {
        constexpr double h = 0.70710678118654752440084436210485;
        // (+-1 +- i) / sqrt2
        if constexpr (e == 4) return mk(h * (a.x - a.y), h * (a.x + a.y));
        if constexpr (e == 12) return mk(-h * (a.x + a.y), h * (a.x - a.y));
        if constexpr (e == 20) return mk(h * (a.y - a.x), -h * (a.x + a.y));
        return mk(h * (a.x + a.y), h * (a.y - a.x));     // e == 28
    } else {
        constexpr double c = cos32(e), s = sin32(e);
        return mk(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

template <int DIR, int NBI, int KA> struct TwRow32 {
    static NSC_HD void run(cd* x) {
        if constexpr (NBI < 8) {
            x[NBI + 8 * KA] = mul_w32<DIR, NBI * KA>(x[NBI + 8 * KA]);
            TwRow32<DIR, NBI + 1, KA>::run(x);
        }
    }
};

// DFT-32, natural register order in (x[n]), permuted order out: x[8 ka + kb] = X[ka + 4 kb]
template <int DIR> NSC_HD void dft32_nat_in(cd* x) {
#pragma unroll
    for (int nb = 0; nb < 8; ++nb) dft4<DIR>(x[nb], x[nb + 8], x[nb + 16], x[nb + 24]);
    TwRow32<DIR, 1, 1>::run(x);
    TwRow32<DIR, 1, 2>::run(x);
    TwRow32<DIR, 1, 3>::run(x);
#pragma unroll
    for (int ka = 0; ka < 4; ++ka) dft8<DIR>(x + 8 * ka);
}

// DFT-32, permuted register order in (x[8 na + nb] = sample na + 4 nb), natural order out (x[k] = X[k])
template <int DIR> NSC_HD void dft32_perm_in(cd* x) {
#pragma unroll
    for (int na = 0; na < 4; ++na) dft8<DIR>(x + 8 * na);
    // x[8 na + kb] *= W_32^(na kb): the same table as above with the roles (ka, nb) -> (na, kb)
    TwRow32<DIR, 1, 1>::run(x);
    TwRow32<DIR, 1, 2>::run(x);
    TwRow32<DIR, 1, 3>::run(x);
#pragma unroll
    for (int kb = 0; kb < 8; ++kb) dft4<DIR>(x[kb], x[kb + 8], x[kb + 16], x[kb + 24]);
}

// the LPW transforms of length NA of the S side, in place
template <int NA, int DIR> NSC_HD void dft_s(cd* x) {
#pragma unroll
    for (int l = 0; l < NV / NA; ++l) Dft<NA, DIR>::run(x + NA * l);
}

// ---------------------------------------------------------------- phases of the two transforms
// tw[t * XS + n2] = exp(-2 pi i (t % NA) n2 / N), t < 24, n2 < 32  (plan.cu: one table per length)

// s2p, lane tau < 32: x[0..23] (S layout) -> DFT-NA, twiddle, store column tau of the matrix
template <int NA, int DIR> NSC_HD void s2p_front(cd* x, cd* buf, const cd* tw, int tau) {
    dft_s<NA, DIR>(x);
#pragma unroll
    for (int t = 1; t < NV; ++t) {
        if (t % NA == 0) continue;
        cd w = tw[t * XS + tau];
        if (DIR > 0) w = conj(w);
        x[t] = x[t] * w;
    }
#pragma unroll
    for (int t = 0; t < NV; ++t) buf[t * XS + tau] = x[t];
}
// s2p, lane a < 24 (callers pass a = min(tau, 23)): load row a, DFT-32 -> x[0..31] (P layout)
template <int DIR> NSC_HD void s2p_back(cd* x, const cd* buf, int a) {
#pragma unroll
    for (int n2 = 0; n2 < NB; ++n2) x[n2] = buf[a * XS + n2];
    dft32_nat_in<DIR>(x);
}

// p2s, lane a < 24: x[0..31] (P layout) -> DFT-32, twiddle, store row a  (store iff `active`)
template <int DIR> NSC_HD void p2s_front(cd* x, cd* buf, const cd* tw, int a, bool active) {
    dft32_perm_in<DIR>(x);
#pragma unroll
    for (int k2 = 1; k2 < NB; ++k2) {
        cd w = tw[a * XS + k2];
        if (DIR > 0) w = conj(w);
        x[k2] = x[k2] * w;
    }
    if (active)
#pragma unroll
        for (int k2 = 0; k2 < NB; ++k2) buf[a * XS + k2] = x[k2];
}
// p2s, lane tau < 32: load column tau, DFT-NA -> x[0..23] (S layout)
template <int NA, int DIR> NSC_HD void p2s_back(cd* x, const cd* buf, int tau) {
#pragma unroll
    for (int t = 0; t < NV; ++t) x[t] = buf[t * XS + tau];
    dft_s<NA, DIR>(x);
}

#ifdef __CUDACC__
// Whole transforms for one warp; x has 32 elements.  `buf` is the warp's private exchange matrix.
template <int NA, int DIR> __device__ __forceinline__ void s2p(cd* x, cd* buf, const cd* tw, int tau) {
    __syncwarp();                      // every lane has finished reading buf (previous transform)
    s2p_front<NA, DIR>(x, buf, tw, tau);
    __syncwarp();
    s2p_back<DIR>(x, buf, tau < NV ? tau : NV - 1);
}
template <int NA, int DIR> __device__ __forceinline__ void p2s(cd* x, cd* buf, const cd* tw, int tau) {
    __syncwarp();
    p2s_front<DIR>(x, buf, tw, tau < NV ? tau : NV - 1, tau < NV);
    __syncwarp();
    p2s_back<NA, DIR>(x, buf, tau);
}

// ---------------------------------------------------------------- length 1536 = 2 x 768 on a warp pair
// Warp h (= 0, 1) of a pair holds the samples of parity h in the S layout (register t of lane tau: index
// h + 2 (tau + 32 t)) and, on the P side, the half h of the line (lane a, register e: index a + 24 p(e) + 768 h).
// s2p_pair: each warp transforms its decimated sequence (E, O), then X[k'] = E + W^k' O, X[k' + 768] = E - W^k' O
// (decimation in time); p2s_pair is the mirror image (decimation in frequency: sums to the even outputs, twiddled
// differences to the odd ones).  The halves meet through the warps' exchange matrices (row a, column e) under a
// named barrier of the 64 threads of the pair.  twc[k'] = exp(-2 pi i k' / 1536), k' < 768.
constexpr int NPAIR = 1536;
__device__ __forceinline__ void pair_sync(int pair) { asm volatile("bar.sync %0, 64;" ::"r"(1 + pair) : "memory"); }

template <int DIR>
__device__ __forceinline__ void s2p_pair(cd* x, cd* buf, const cd* pbuf, const cd* tw, const cd* twc, int tau, int h,
                                         int pair) {
    const int a = tau < NV ? tau : NV - 1;
    pair_sync(pair);                   // the partner has finished reading my matrix (previous combine)
    s2p<24, DIR>(x, buf, tw, tau);
    if (h == 1) {
#pragma unroll
        for (int e = 0; e < NB; ++e) {
            cd w = twc[a + NV * p_of(e)];
            if (DIR > 0) w = conj(w);
            x[e] = x[e] * w;
        }
    }
    __syncwarp();                      // every lane has read its row of the matrix
    if (tau < NV)
#pragma unroll
        for (int e = 0; e < NB; ++e) buf[a * XS + e] = x[e];
    pair_sync(pair);
#pragma unroll
    for (int e = 0; e < NB; ++e) {
        const cd y = pbuf[a * XS + e];
        x[e] = h == 0 ? x[e] + y : y - x[e];
    }
}

template <int DIR>
__device__ __forceinline__ void p2s_pair(cd* x, cd* buf, const cd* pbuf, const cd* tw, const cd* twc, int tau, int h,
                                         int pair) {
    const int a = tau < NV ? tau : NV - 1;
    pair_sync(pair);                   // both matrices are free
    if (tau < NV)
#pragma unroll
        for (int e = 0; e < NB; ++e) buf[a * XS + e] = x[e];
    pair_sync(pair);
#pragma unroll
    for (int e = 0; e < NB; ++e) {
        const cd y = pbuf[a * XS + e];
        if (h == 0) {
            x[e] = x[e] + y;
        } else {
            cd w = twc[a + NV * p_of(e)];
            if (DIR > 0) w = conj(w);
            x[e] = (y - x[e]) * w;
        }
    }
    pair_sync(pair);                   // the partner has read my matrix: the transform may overwrite it
    p2s<24, DIR>(x, buf, tw, tau);
}

// cooperative copy of the [24][33] twiddle matrix (global, plan.cu) into shared memory
__device__ __forceinline__ void load_twiddles(cd* tw_s, const cd* tw_g) {
    for (int i = threadIdx.x; i < XBUF; i += blockDim.x) tw_s[i] = tw_g[i];
}
#endif

}  // namespace fw
}  // namespace nsc
