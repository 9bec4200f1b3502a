// nonlinear_v2.cuh -- transform kernels of the nonlinear term for the long line lengths 768 = 24 x 32 and
// 384 = 12 x 32 (BASELINE.json configs[3]: 3/2-padded 768 x 768 grid per radial node, the headline workload;
// configs[2]: 384 x 384, heated).  Same steps N1-N6 and the same intermediate layout as nonlinear_kernels.cuh;
// what changes:
//
//   * the two-pass NA x 32 transform of fft_warp.cuh: one shared-memory exchange per line instead of two,
//     conflict-free, one warp per 768-line (or per two 384-lines) and only warp-level barriers inside a transform;
//   * k_dr     the radial derivative D1 f (N1) is taken once per evaluation by a marching kernel
//              (one thread per (m, k) column, nine levels in registers), so that no transform
//              kernel re-reads nine radial neighbours per line;
//   * k_zinv2  4 (8) adjacent m-lines per CTA; the transposed [z][m] stores go through a swizzled
//              shared-memory tile and leave as full 64-byte (128-byte) segments;
//   * k_theta2 one (j, z) point-line (two for length 384) per warp, the 12 (15 with temperature) real
//              physical-space lines exist only in registers; the three velocity lines and one parked line live
//              in a lane-private scratch in Tensor Memory (tcgen05.st / tcgen05.ld, 256 columns per warp: TMEM
//              as a 256 KB lane-private register spill space next to the 64 K registers); optionally the
//              per-level maxima of |u_r|, |u_theta|, |u_z| for the CFL rate of the step-size controller;
//   * k_zfwd2  cp.async double-buffered [z][4 m] ([z][8 m]) tiles, forward transform, truncation, scaling,
//              buoyancy.
#pragma once
#include <cstdint>
#include "fft_warp.cuh"
#include "nonlinear_v2_args.h"

namespace nsc {


// ------------------------------------------------------------------------------------------ k_dr
// out[j] = sum_l D1[j][l] f[s0(j) + l],  s0(j) = clamp(j - 4, 0, N_r - 9)   (O2, R3)
// One thread per (mode, field) marches over j; the rows of f arrive by cp.async in a 16-row
// shared-memory ring up to seven rows ahead of the stencil (column threadIdx.x of the ring is private).
constexpr int DR_TB = 128;  // modes per block
constexpr int DR_PRE = 12;  // rows requested up front; row j + DR_PRE is requested after row j is done, so the
                            // ring holds rows j - 3 .. j + 12 (16 rows) when row j + 1 starts
template <int R> struct DrRow { static constexpr int value = R; };
#define NSC_DR_ROWS16(F, j0)                                                                              \
    F(DrRow<0>{}, (j0) + 0); F(DrRow<1>{}, (j0) + 1); F(DrRow<2>{}, (j0) + 2); F(DrRow<3>{}, (j0) + 3);     \
    F(DrRow<4>{}, (j0) + 4); F(DrRow<5>{}, (j0) + 5); F(DrRow<6>{}, (j0) + 6); F(DrRow<7>{}, (j0) + 7);     \
    F(DrRow<8>{}, (j0) + 8); F(DrRow<9>{}, (j0) + 9); F(DrRow<10>{}, (j0) + 10); F(DrRow<11>{}, (j0) + 11); \
    F(DrRow<12>{}, (j0) + 12); F(DrRow<13>{}, (j0) + 13); F(DrRow<14>{}, (j0) + 14); F(DrRow<15>{}, (j0) + 15)

__global__ void __launch_bounds__(DR_TB) k_dr(DrArgs a) {
    __shared__ __align__(16) cd ring[16][DR_TB];
    const int tx = threadIdx.x;
    const size_t col0 = (size_t)blockIdx.x * DR_TB + tx;
    const bool valid = col0 < a.ncols;
    const size_t col = valid ? col0 : a.ncols - 1;
    const int fi = blockIdx.y;
    const cd* src = (fi == 0 ? a.f[0] : fi == 1 ? a.f[1] : fi == 2 ? a.f[2] : a.f[3]) + col;
    cd* dst = (fi == 0 ? a.out[0] : fi == 1 ? a.out[1] : fi == 2 ? a.out[2] : a.out[3]) + col;
    const int N = a.N_r;
    auto issue = [&](int row) {
        if (row < N) {
            const uint32_t d = (uint32_t)__cvta_generic_to_shared(&ring[row & 15][tx]);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src + (size_t)row * a.plane) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
#pragma unroll
    for (int r = 0; r < DR_PRE; ++r) issue(r);
    // register copy of the ring: row r lives in w[r & 15]; the march is unrolled by 16 so that every index is
    // a compile-time constant; each row enters the registers once (one shared-memory read per result)
    cd w[16];
    asm volatile("cp.async.wait_group %0;" ::"n"(DR_PRE - NPT) : "memory");     // rows 0 .. 8
#pragma unroll
    for (int r = 0; r < NPT; ++r) w[r] = ring[r][tx];
    auto row = [&](auto tag, int j) {
        constexpr int R = decltype(tag)::value;
        if (j >= N) return;
        const double* d = a.D1 + j * NPT;
        cd acc = mk(0.0, 0.0);
        if (j > N - 1 - NPT / 2) {
            // last rows: stencil rows N - 9 .. N - 1 (all loaded), ring position not static: from shared memory
            asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
            for (int l = 0; l < NPT; ++l) {
                const double c = __ldg(d + l);
                const cd v = ring[(N - NPT + l) & 15][tx];
                acc.x = fma(c, v.x, acc.x);
                acc.y = fma(c, v.y, acc.y);
            }
        } else {
            if (j > NPT / 2) {                          // row j + 4 enters the window
                asm volatile("cp.async.wait_group %0;" ::"n"(DR_PRE - 1 - NPT / 2) : "memory");
                w[(R + NPT / 2) & 15] = ring[(R + NPT / 2) & 15][tx];
            }
            // first rows (j <= 4): rows 0 .. 8 = w[0 .. 8]; interior: rows j - 4 .. j + 4
#pragma unroll
            for (int l = 0; l < NPT; ++l) {
                const double c = __ldg(d + l);
                const cd v = (R <= NPT / 2) ? ((j <= NPT / 2) ? w[l] : w[(R - NPT / 2 + l) & 15]) : w[(R - NPT / 2 + l) & 15];
                acc.x = fma(c, v.x, acc.x);
                acc.y = fma(c, v.y, acc.y);
            }
        }
        if (valid) dst[(size_t)j * a.plane] = acc;
        issue(DR_PRE + j);
    };
    for (int j0 = 0; j0 < N; j0 += 16) {
        NSC_DR_ROWS16(row, j0);
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------ z kernels
constexpr int Z2_WARPS = 4;
constexpr int Z2_THREADS = Z2_WARPS * 32;

template <int NA> struct Z2Cfg {
    using G = fw::WGeo<NA>;
    static constexpr int LPW = G::LPW;                           // spectral lines per warp
    static constexpr int MT = Z2_WARPS * LPW;                    // m-lines per work item: 4 (768) or 8 (384)
    static constexpr int LINE = (2 * G::NMAX + 1 + 7) / 8 * 8;   // staged spectral line (>= 2 K + 1): 520 / 264
    static constexpr int TILE = G::N * MT;                       // complex elements of the [N][MT] tile (3072)
    static constexpr int NIT = TILE / Z2_THREADS;                // tile elements per thread (24)
    static constexpr size_t SMEM_INV = sizeof(cd) * (size_t)(fw::XBUF * (1 + Z2_WARPS) + LINE * LPW * Z2_WARPS);
    static constexpr size_t SMEM_FWD = sizeof(cd) * (size_t)(fw::XBUF * (1 + Z2_WARPS) + TILE);
    static_assert(TILE <= fw::XBUF * Z2_WARPS, "the tile overlays the exchange matrices");
};

// swizzle of the m_local index of row z of a [N][MT] tile: positions (in 16-byte chunks) z MT + (ml ^ swz(z)) are
// conflict free both for lanes walking z (transform side) and for lanes walking (z, m_local) row-major (global side)
template <int MT> __device__ __forceinline__ int swz(int z) { return MT == 4 ? ((z >> 1) & 3) : (z & 7); }
template <int MT> __device__ __forceinline__ int tile_pos(int z, int ml) { return z * MT + (ml ^ swz<MT>(z)); }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------ k_zinv2
// work item = (field, level, tile of MT adjacent m); two or three inverse transforms per line:
// q = 1 (i kappa f), q = 0 (f), [q = 2 (D1 f)].  Each warp stages its spectral line(s) in a private
// shared-memory buffer filled by cp.async one transform ahead (f for two transforms, then D1 f,
// then the next item's f), so no line waits in registers; the transforms share one copy of
// the code (instruction cache).
template <int NA>
__global__ void __launch_bounds__(Z2_THREADS, 2) k_zinv2(Nl2Args A) {
    using namespace fw;
    using G = WGeo<NA>;
    using C = Z2Cfg<NA>;
    constexpr int N = G::N, LPW = C::LPW, MT = C::MT;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    cd* tile = tw + XBUF;                               // [N][MT] tile, overlays the 4 matrices
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    cd* buf = tile + warp * XBUF;
    cd* line = tw + XBUF * (1 + Z2_WARPS) + warp * (LPW * C::LINE);
    load_twiddles(tw, A.tw_z);
    const int mtiles = a.MP / MT;
    const size_t plane = (size_t)a.M1 * a.NK;
    const size_t qstride = (size_t)N * a.MP;
    const double taud = (double)tau;
    const int NKc = a.NK;

    // requests this warp's spectral line(s) of item `it` from `base` (a field or its radial derivative)
    auto fetch = [&](const cd* base, int it) {
        const int mt = it % mtiles, r = it / mtiles;
        const int jl = r % a.nj;
#pragma unroll
        for (int l = 0; l < LPW; ++l) {
            const int m = mt * MT + warp * LPW + l;
            if (m < a.M1) {
                const cd* src = base + (size_t)(a.j0 + jl) * plane + (size_t)m * NKc;
                for (int i = tau; i < NKc; i += 32) cp_async16(line + l * C::LINE + i, src + i);
            }
        }
    };
    auto field_of = [&](int it) { return (it / mtiles) / a.nj; };
    // without radial-derivative input (A.dr[0] null) only i kappa f and f are transformed: D1 is then
    // applied to the z-transformed f by k_dr on the work array (D1 and the z transform commute)
    const int ns = A.dr[0] ? 3 : 2;
    int item = blockIdx.x;
    if (item < A.nitems) fetch(a.f[field_of(item)], item);
    __syncthreads();                                    // twiddles

    for (; item < A.nitems; item += gridDim.x) {
        const int mt = item % mtiles, r = item / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
#pragma unroll 1
        for (int s = 0; s < ns; ++s) {
            const int q = (s == 0) ? 1 : (s == 1 ? 0 : 2);
            cd x[32];
            if (s != 1) {
                cp_async_commit_wait_all();
                __syncwarp();
            }
            // v' = (am + i bm k) v: (am, bm) = (0, alpha) for d/dz = i kappa, (1, 0) otherwise (no branch per slot)
            const double am = (s == 0) ? 0.0 : 1.0, bm = (s == 0) ? A.alpha : 0.0;
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                const int l = t / NA, tt = t % NA;
                cd v = mk(0.0, 0.0);
                if (G::slot_live(tt)) {
                    const bool pos = G::slot_pos(tt);
                    const int bin = tau + 32 * tt;
                    const bool vm = (mt * MT + warp * LPW + l) < a.M1;
                    const bool ok = vm && (pos ? (bin <= a.K) : (bin >= N - a.K));
                    const int kk = pos ? bin + a.K : bin - N + a.K;
                    const cd g = ok ? line[l * C::LINE + kk] : mk(0.0, 0.0);
                    const double kd = bm * (pos ? taud + (double)(32 * tt) : taud + (double)(32 * tt - N));
                    v = mk(fma(-kd, g.y, am * g.x), fma(kd, g.x, am * g.y));
                }
                x[t] = v;
            }
            if (s >= 1) {                               // the staged line is consumed: request the next one
                __syncwarp();
                if (s == 1 && ns == 3) {
                    fetch(A.dr[fi], item);
                } else {
                    const int nxt = item + gridDim.x;
                    if (nxt < A.nitems) fetch(a.f[field_of(nxt)], nxt);
                }
            }
            s2p<NA, +1>(x, buf, tw, tau);
            // P-layout result of this warp's line(s) -> tile -> [z][m] work array in MT * 16-byte segments
            __syncthreads();                            // all warps left their exchange matrices
            if (tau < NV) {
                const int ml = warp * LPW + tau / NA;
#pragma unroll
                for (int e = 0; e < 32; ++e) tile[tile_pos<MT>(G::p_idx(e, tau), ml)] = x[e];
            }
            __syncthreads();
            cd* dst = a.zbuf + ((size_t)jl * 3 * a.nf + (3 * fi + q)) * qstride + mt * MT;
            // all shared-memory reads first, then all stores (the transform's registers are free here): no
            // store has to release its source registers before the next read can issue
            {
                cd v[C::NIT];
#pragma unroll
                for (int it = 0; it < C::NIT; ++it) v[it] = tile[threadIdx.x + it * Z2_THREADS];
                // id = threadIdx.x + 128 it: z = id / MT = z0 + (128 / MT) it, c = id % MT = c0; swz(z) = swz(z0)
                const int z0 = threadIdx.x / MT, c0 = threadIdx.x % MT;
                cd* d0 = dst + (size_t)z0 * a.MP + (c0 ^ swz<MT>(z0));
#pragma unroll
                for (int it = 0; it < C::NIT; ++it) d0[(size_t)((Z2_THREADS / MT) * it) * a.MP] = v[it];
            }
            __syncthreads();                            // tile free again
        }
    }
    cp_async_commit_wait_all();
}

// ------------------------------------------------------------------------------------------ k_zfwd2
// work item = (field, level, tile of MT adjacent m).  The [N][MT] tile of theta-transformed
// products arrives by cp.async (MT * 16-byte segments) while the previous item is being transformed.
template <int NA>
__global__ void __launch_bounds__(Z2_THREADS, 2) k_zfwd2(Nl2Args A) {
    using namespace fw;
    using G = WGeo<NA>;
    using C = Z2Cfg<NA>;
    constexpr int N = G::N, LPW = C::LPW, MT = C::MT;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    cd* buf = tw + XBUF + warp * XBUF;
    cd* tile = tw + XBUF * (1 + Z2_WARPS);
    load_twiddles(tw, A.tw_z);
    const int a23 = tau < NV ? tau : NV - 1;
    const int mtiles = a.MP / MT;
    const size_t qstride = (size_t)N * a.MP;

    auto fetch = [&](int it) {
        const int mt = it % mtiles, r = it / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
        const cd* src = a.tbuf + ((size_t)jl * a.nf + fi) * qstride + mt * MT;
#pragma unroll 4
        for (int k = 0; k < C::NIT; ++k) {
            const int id = threadIdx.x + k * Z2_THREADS;
            const int z = id / MT, c = id % MT;
            cp_async16(tile + id, src + (size_t)z * a.MP + (c ^ swz<MT>(z)));
        }
    };
    int item = blockIdx.x;
    if (item < A.nitems) fetch(item);
    for (; item < A.nitems; item += gridDim.x) {
        const int mt = item % mtiles, r = item / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
        const int j = a.j0 + jl;
        cp_async_commit_wait_all();
        __syncthreads();                                 // the tile (and, first time, tw) is complete
        cd x[32];
        {
            const int ml = warp * LPW + a23 / NA;
#pragma unroll
            for (int e = 0; e < 32; ++e) x[e] = tile[tile_pos<MT>(G::p_idx(e, a23), ml)];
        }
        __syncthreads();                                 // every warp holds its line(s): the tile is free
        if (item + (int)gridDim.x < A.nitems) fetch(item + gridDim.x);
        p2s<NA, -1>(x, buf, tw, tau);
        const bool add_buoy = (fi == 2) && (a.buoy != 0.0);
#pragma unroll
        for (int l = 0; l < LPW; ++l) {
            const int m = mt * MT + warp * LPW + l;
            if (m < a.M1) {
                const size_t off = ((size_t)j * a.M1 + m) * a.NK;
                cd* dst = a.out[fi] + off;
                const cd* Th = a.f[add_buoy ? 3 : 0] + off;
#pragma unroll
                for (int tt = 0; tt < NA; ++tt) {
                    if (G::slot_live(tt)) {
                        const bool pos = G::slot_pos(tt);
                        const int bin = tau + 32 * tt;
                        if (pos ? (bin <= a.K) : (bin >= N - a.K)) {
                            const int kk = pos ? bin + a.K : bin - N + a.K;
                            cd v = a.scale * x[l * NA + tt];
                            if (add_buoy) {
                                const cd th = Th[kk];
                                v.x = fma(a.buoy, th.x, v.x);
                                v.y = fma(a.buoy, th.y, v.y);
                            }
                            dst[kk] = v;
                        }
                    }
                }
            }
        }
    }
    cp_async_commit_wait_all();
}

// ------------------------------------------------------------------------------------------ scratch
// Lane-private scratch of k_theta2: T2_NSLOT lines of 32 doubles per lane in Tensor Memory.  A CTA of 8 warps owns
// all 512 columns of its SM's TMEM; warp w may touch the 32 lanes of its quadrant (w & 3) only, so warps w and
// w + 4 share lanes and split the columns: 256 columns = 128 doubles per thread = 4 slots of 32.  tcgen05.st / .ld
// with shape 32x32b move one 32-bit column per register per lane; x16 = 8 doubles per instruction.
constexpr int T2_NSLOT = 4;            // U_r, U_theta / r, U_z, one parked line
constexpr int T2_WARPS = 8;

struct TmemScratch {
    uint32_t base;        // TMEM address (lane << 16 | column) of this warp's slot 0
    __device__ __forceinline__ void st8(uint32_t addr, const double* v) const {
        asm volatile(
            "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, "
            "%14, %15, %16};" ::"r"(addr),
            "r"(__double2loint(v[0])), "r"(__double2hiint(v[0])), "r"(__double2loint(v[1])),
            "r"(__double2hiint(v[1])), "r"(__double2loint(v[2])), "r"(__double2hiint(v[2])),
            "r"(__double2loint(v[3])), "r"(__double2hiint(v[3])), "r"(__double2loint(v[4])),
            "r"(__double2hiint(v[4])), "r"(__double2loint(v[5])), "r"(__double2hiint(v[5])),
            "r"(__double2loint(v[6])), "r"(__double2hiint(v[6])), "r"(__double2loint(v[7])),
            "r"(__double2hiint(v[7]))
            : "memory");
    }
    // asynchronous: the 16 raw registers are valid only after wait_ld()
    __device__ __forceinline__ void ld8_raw(uint32_t addr, uint32_t* r) const {
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, "
            "%14, %15}, [%16];"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
              "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
            : "r"(addr)
            : "memory");
    }
    // the registers of every ld8_raw issued so far are valid after this
    __device__ __forceinline__ void wait_ld() const { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
};

// chunked access (8 doubles = elements 8 c .. 8 c + 7 of a slot); split form: sc_ld8_raw (issue) ... sc_wait_ld
// ... sc_unpack8 (use), so that several loads share one wait
struct Raw8 {
    uint32_t r[16];
};
__device__ __forceinline__ void sc_st8(const TmemScratch& s, int slot, int c, const double* v) {
    s.st8(s.base + slot * 64 + c * 16, v);
}
__device__ __forceinline__ void sc_fence(const TmemScratch&) {
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void sc_ld8_raw(const TmemScratch& s, int slot, int c, Raw8& q) {
    s.ld8_raw(s.base + slot * 64 + c * 16, q.r);
}
__device__ __forceinline__ void sc_wait_ld(const TmemScratch& s) { s.wait_ld(); }
__device__ __forceinline__ void sc_unpack8(const Raw8& q, double* v) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __hiloint2double((int)q.r[2 * i + 1], (int)q.r[2 * i]);
}

template <int NA> struct T2Cfg {
    using G = fw::WGeo<NA>;
    static constexpr int LPW = G::LPW;                            // point-lines per warp
    static constexpr int STAGE = (G::NMAX + 1 + 7) / 8 * 8;       // staged half-spectral line (>= M + 1): 264 / 136
    // twiddles + one exchange matrix and one staged line pair per point-line per warp; more than half of the SM's
    // shared memory, so exactly one CTA (the owner of all 512 TMEM columns) is resident per SM
    static constexpr size_t SMEM = sizeof(cd) * ((size_t)fw::XBUF * (1 + T2_WARPS) + (size_t)2 * STAGE * LPW * T2_WARPS);
};

// ------------------------------------------------------------------------------------------ k_theta2
// Z[i] = G_X(i) + i G_Y(i) in the S layout, G(m) = mult * line[m] (0 <= m <= M), G(-m) = conj G(m),
// Im G(0) dropped (R6); mult = 1 or i n_m (d/dtheta, N1).  Slots without a retained mode are zero padding.
// One copy of the code serves all inverse transforms of a point-line, which keeps the kernel inside the instruction
// cache.  dx / dy select the d/dtheta multiplier i n of the X / Y half; the transforms without a derivative take the
// short branch (uniform per warp), the others blend (1, 0) / (0, n) multipliers arithmetically (no selects).
// X, Y: the LPW staged lines of each half, STAGE apart.
template <int NA>
__device__ __forceinline__ void load_pair_rt(cd* x, const cd* X, const cd* Y, bool dx, bool dy, int M, int tau,
                                             double taud, double kth0) {
    using G = fw::WGeo<NA>;
    constexpr int N = G::N, STAGE = T2Cfg<NA>::STAGE;
    if (!(dx || dy)) {
#pragma unroll
        for (int t = 0; t < fw::NV; ++t) {
            const int l = t / NA, tt = t % NA;
            if (!G::slot_live(tt)) {
                x[t] = mk(0.0, 0.0);
            } else if (G::slot_pos(tt)) {
                const int m = tau + 32 * tt;
                const bool ok = m <= M;
                cd gx = ok ? X[l * STAGE + m] : mk(0.0, 0.0);
                cd gy = ok ? Y[l * STAGE + m] : mk(0.0, 0.0);
                if (tt == 0 && tau == 0) {
                    gx.y = 0.0;
                    gy.y = 0.0;
                }
                x[t] = mk(gx.x - gy.y, gx.y + gy.x);
            } else {
                const int m = N - 32 * tt - tau;
                const bool ok = m <= M;
                const cd gx = ok ? X[l * STAGE + m] : mk(0.0, 0.0);
                const cd gy = ok ? Y[l * STAGE + m] : mk(0.0, 0.0);
                x[t] = mk(gx.x + gy.y, gy.x - gx.y);
            }
        }
    } else {
        // g' = (a + i b n) g with (a, b) = (1, 0) plain or (0, 1) derivative
        const double ax = dx ? 0.0 : 1.0, bx = dx ? kth0 : 0.0;
        const double ay = dy ? 0.0 : 1.0, by = dy ? kth0 : 0.0;
#pragma unroll
        for (int t = 0; t < fw::NV; ++t) {
            const int l = t / NA, tt = t % NA;
            if (!G::slot_live(tt)) {
                x[t] = mk(0.0, 0.0);
            } else if (G::slot_pos(tt)) {
                const int m = tau + 32 * tt;
                const bool ok = m <= M;
                cd gx = ok ? X[l * STAGE + m] : mk(0.0, 0.0);
                cd gy = ok ? Y[l * STAGE + m] : mk(0.0, 0.0);
                if (tt == 0 && tau == 0) {
                    gx.y = 0.0;
                    gy.y = 0.0;
                }
                const double mr = taud + (double)(32 * tt);
                const double bxn = bx * mr, byn = by * mr;
                const cd hx = mk(fma(-bxn, gx.y, ax * gx.x), fma(bxn, gx.x, ax * gx.y));
                const cd hy = mk(fma(-byn, gy.y, ay * gy.x), fma(byn, gy.x, ay * gy.y));
                x[t] = mk(hx.x - hy.y, hx.y + hy.x);
            } else {
                const int m = N - 32 * tt - tau;
                const bool ok = m <= M;
                const cd gx = ok ? X[l * STAGE + m] : mk(0.0, 0.0);
                const cd gy = ok ? Y[l * STAGE + m] : mk(0.0, 0.0);
                const double mr = (double)(N - 32 * tt) - taud;
                const double bxn = bx * mr, byn = by * mr;
                const cd hx = mk(fma(-bxn, gx.y, ax * gx.x), fma(bxn, gx.x, ax * gx.y));
                const cd hy = mk(fma(-byn, gy.y, ay * gy.x), fma(byn, gy.x, ay * gy.y));
                x[t] = mk(hx.x + hy.y, hy.x - hx.y);
            }
        }
    }
}

// Splits the forward transform Z (S layout) of a packed real pair (a + i b) into the Hermitian half
// lines A[m] = (Z[m] + conj Z[N-m]) / 2, B[m] = (Z[m] - conj Z[N-m]) / (2 i), m <= M (N5 truncation).
// Z[N-m] of lane tau, slot tt sits in lane (32 - tau) & 31, slot NA - 1 - tt (lane 0: its own slot (NA - tt) % NA).
// outA / outB: line l of the warp at outA + l * lstep.
template <int NA>
__device__ __forceinline__ void store_pair_rt(const cd* x, cd* outA, cd* outB, size_t lstep, bool has_b, int M, int tau) {
    using G = fw::WGeo<NA>;
    constexpr int TTMAX = G::NMAX / 32;                  // the last positive slot: only lane 0 (m = NMAX) can be kept
    const int src = (32 - tau) & 31;
#pragma unroll
    for (int l = 0; l < G::LPW; ++l) {
#pragma unroll
        for (int tt = 0; tt <= TTMAX; ++tt) {
            cd pz;
            if (tt == TTMAX) {
                pz = x[l * NA + NA - tt];
            } else {
                pz.x = __shfl_sync(0xffffffffu, x[l * NA + NA - 1 - tt].x, src);
                pz.y = __shfl_sync(0xffffffffu, x[l * NA + NA - 1 - tt].y, src);
                if (tau == 0) pz = x[l * NA + (NA - tt) % NA];
            }
            const int m = tau + 32 * tt;
            if (m <= M) {
                const cd zm = conj(pz);
                outA[l * lstep + m] = 0.5 * (x[l * NA + tt] + zm);
                if (has_b) outB[l * lstep + m] = 0.5 * mul_mi(x[l * NA + tt] - zm);
            }
        }
    }
}

// The inverse transforms of a point-line as a table: work array index q = 3 field + kind (kind 0 f, 1 d_z f,
// 2 d_r f) of the X and Y halves of the packed pair; d/dtheta flags: X for t = 2, 5, Y for t = 3, 6.
//   t : 0 (u_r, u_th)  1 (u_z, dr u_r)  2 (dth u_r, dz u_r)  3 (dr u_th, dth u_th)  4 (dz u_th, dr u_z)
//       5 (dth u_z, dz u_z)  6 (dr T, dth T)  7 (dz T, -)      [6, 7 with temperature only]
__device__ __forceinline__ int t2_qx(int t) { return (int)((0xAB645060u >> (4 * t)) & 15u); }
__device__ __forceinline__ int t2_qy(int t) { return (int)((0xA9783123u >> (4 * t)) & 15u); }

// The physical-space stage (N4) of inverse transform t of a point-line, shared by k_theta2 and k_theta3: x holds the
// transformed pair in the P layout (32 points per lane); slots of the lane-private scratch: 0 U_r, 1 U_theta / r,
// 2 U_z, 3 a parked line; acc carries partial sums from one transform to the next.  After t = 4 and after the last
// transform x holds the pair to be transformed forward.  cfl_j: the three maxima of the point-line's radial level.
template <int NF, bool CFL>
__device__ __forceinline__ void theta_products(int t, cd* x, double* acc, const TmemScratch& sc, double ri, double rj,
                                               unsigned long long* cfl_j, int tau) {
    // physical-space stage (N4): slots 0 U_r, 1 U_theta / r, 2 U_z, 3 parked line
    if (t == 0) {
        if constexpr (CFL) {                            // per-level maxima for the CFL rate (step-size control)
            double m0 = 0.0, m1 = 0.0;
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                m0 = fmax(m0, fabs(x[e].x));
                m1 = fmax(m1, fabs(x[e].y));
            }
            line_atomic_max<32>(cfl_j, m0, tau);
            line_atomic_max<32>(cfl_j + 1, m1, tau);
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t0[8], t1[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                t0[i] = x[8 * c + i].x;
                t1[i] = x[8 * c + i].y * ri;
            }
            sc_st8(sc, 0, c, t0);
            sc_st8(sc, 1, c, t1);
        }
    } else if (t == 1) {                               // acc = U_r d_r u_r
        if constexpr (CFL) {
            double m2 = 0.0;
#pragma unroll
            for (int e = 0; e < 32; ++e) m2 = fmax(m2, fabs(x[e].x));
            line_atomic_max<32>(cfl_j + 2, m2, tau);
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t0[8], t2[8];
            Raw8 q0;
            sc_ld8_raw(sc, 0, c, q0);
            sc_wait_ld(sc);
            sc_unpack8(q0, t0);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                t2[i] = x[8 * c + i].x;
                acc[8 * c + i] = t0[i] * x[8 * c + i].y;
            }
            sc_st8(sc, 2, c, t2);
        }
    } else if (t == 2) {                               // N_r = -(u.grad u_r - u_theta^2 / r) -> slot 3
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t0[8], t1[8], t2[8];
            Raw8 q0;
            Raw8 q1;
            sc_ld8_raw(sc, 1, c, q0);
            sc_ld8_raw(sc, 2, c, q1);
            sc_wait_ld(sc);
            sc_unpack8(q0, t1);
            sc_unpack8(q1, t2);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                double s = fma(t1[i], x[8 * c + i].x, acc[8 * c + i]);
                s = fma(t2[i], x[8 * c + i].y, s);
                s = fma(-(t1[i] * rj), t1[i], s);
                t0[i] = -s;
            }
            sc_st8(sc, 3, c, t0);
        }
    } else if (t == 3 || t == 6) {                     // acc = U_r d_r f + (U_th / r) d_th f,  f = u_th or T
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t0[8], t1[8];
            Raw8 q0;
            Raw8 q1;
            sc_ld8_raw(sc, 0, c, q0);
            sc_ld8_raw(sc, 1, c, q1);
            sc_wait_ld(sc);
            sc_unpack8(q0, t0);
            sc_unpack8(q1, t1);
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[8 * c + i] = fma(t1[i], x[8 * c + i].y, t0[i] * x[8 * c + i].x);
        }
    } else if (t == 4) {                               // N_theta; x <- (N_r, N_theta); slot 3 <- U_r d_r u_z
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t0[8], t1[8], t2[8], t3[8];
            Raw8 q0;
            Raw8 q1;
            Raw8 q2;
            Raw8 q3;
            sc_ld8_raw(sc, 0, c, q0);
            sc_ld8_raw(sc, 1, c, q1);
            sc_ld8_raw(sc, 2, c, q2);
            sc_ld8_raw(sc, 3, c, q3);
            sc_wait_ld(sc);
            sc_unpack8(q0, t0);
            sc_unpack8(q1, t1);
            sc_unpack8(q2, t2);
            sc_unpack8(q3, t3);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                double s = fma(t2[i], x[8 * c + i].x, acc[8 * c + i]);
                s = fma(t0[i], t1[i], s);
                t2[i] = t0[i] * x[8 * c + i].y;
                x[8 * c + i] = mk(t3[i], -s);
            }
            sc_st8(sc, 3, c, t2);
        }
    } else if (t == 5) {                               // N_z = -(u.grad u_z)  (buoyancy: k_zfwd)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t0[8], t1[8], t2[8];
            Raw8 q0;
            Raw8 q1;
            Raw8 q2;
            sc_ld8_raw(sc, 1, c, q0);
            sc_ld8_raw(sc, 2, c, q1);
            sc_ld8_raw(sc, 3, c, q2);
            sc_wait_ld(sc);
            sc_unpack8(q0, t1);
            sc_unpack8(q1, t2);
            sc_unpack8(q2, t0);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                double s = fma(t1[i], x[8 * c + i].x, t0[i]);
                s = fma(t2[i], x[8 * c + i].y, s);
                if (NF == 3)
                    x[8 * c + i] = mk(-s, 0.0);
                else
                    t0[i] = -s;
            }
            if (NF == 4) sc_st8(sc, 3, c, t0);         // N_z parked until N_T is known
        }
    } else {                                           // t == 7: N_T = -(u.grad T); x <- (N_z, N_T)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double t2[8], t3[8];
            Raw8 q2;
            Raw8 q3;
            sc_ld8_raw(sc, 2, c, q2);
            sc_ld8_raw(sc, 3, c, q3);
            sc_wait_ld(sc);
            sc_unpack8(q2, t2);
            sc_unpack8(q3, t3);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const double s = fma(t2[i], x[8 * c + i].x, acc[8 * c + i]);
                x[8 * c + i] = mk(t3[i], -s);
            }
        }
    }
}

// CFL: also gather the per-level maxima of |u_r|, |u_theta|, |u_z| (a.cfl); an instantiation of its own, because
// that code, even when skipped, lengthens the transform loop beyond the instruction cache (4 % slower).
template <int NA, int NF, bool CFL>
__global__ void __launch_bounds__(T2_WARPS * 32, 1) k_theta2(Nl2Args A) {
    using namespace fw;
    using G = WGeo<NA>;
    using Cfg = T2Cfg<NA>;
    constexpr int LPW = Cfg::LPW, STAGE = Cfg::STAGE;
    constexpr int NT = NF == 3 ? 6 : 8;                  // inverse transforms per point-line
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tmem_base_s;
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    cd* buf = tw + XBUF * (1 + warp);
    load_twiddles(tw, A.tw_t);
    TmemScratch sc;
    if (warp == 0) {
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&tmem_base_s);
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(dst) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    sc.base = tmem_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 256);
    const int M = a.M;
    const double taud = (double)tau, kth0 = A.ktheta0;
    const size_t qstride = (size_t)a.Nz * a.MP;
    const int nlines = a.nj * a.Nz;                      // even; the LPW lines of a warp share their radial level
    const int lstride = gridDim.x * T2_WARPS * LPW;
    // this warp's staged line pairs (X then Y, LPW lines each) of the next inverse transform, filled by cp.async
    cd* stX = tw + XBUF * (1 + T2_WARPS) + 2 * STAGE * LPW * warp;
    cd* stY = stX + STAGE * LPW;
    auto stage = [&](int ln, int t) {
        const size_t off = ((size_t)(ln / a.Nz) * 3 * a.nf * a.Nz + ln % a.Nz) * a.MP;     // line ln of q = 0; ln + 1: + MP
        const cd* X = a.zbuf + (size_t)t2_qx(t) * qstride + off;
        const cd* Y = a.zbuf + (size_t)t2_qy(t) * qstride + off;
#pragma unroll
        for (int l = 0; l < LPW; ++l)
            for (int i = tau; i <= M; i += 32) {
                cp_async16(stX + l * STAGE + i, X + (size_t)l * a.MP + i);
                cp_async16(stY + l * STAGE + i, Y + (size_t)l * a.MP + i);
            }
    };
    int line = (blockIdx.x * T2_WARPS + warp) * LPW;
    if (line < nlines) stage(line, 0);
    for (; line < nlines; line += lstride) {
        const int jl = line / a.Nz;
        const size_t loff = ((size_t)jl * a.nf * a.Nz + line % a.Nz) * a.MP;   // line (j, z) of q = 0 in tbuf
        const double ri = a.rinv[a.j0 + jl];
        const double rj = 1.0 / ri;
        cd x[32];
        double acc[32];
#pragma unroll 1
        for (int t = 0; t < NT; ++t) {
            cp_async_commit_wait_all();
            __syncwarp();
            load_pair_rt<NA>(x, stX, stY, t == 2 || t == 5, t == 3 || t == 6, M, tau, taud, kth0);
            __syncwarp();                                      // the staged pair is consumed: request the next one
            if (t < NT - 1)
                stage(line, t + 1);
            else if (line + lstride < nlines)
                stage(line + lstride, 0);
            s2p<NA, +1>(x, buf, tw, tau);
            sc_fence(sc);
            theta_products<NF, CFL>(t, x, acc, sc, ri, rj, a.cfl + 3 * (a.j0 + jl), tau);
            if (t == 4 || t == NT - 1) {                       // N5: forward transform, truncation m <= M
                p2s<NA, -1>(x, buf, tw, tau);
                cd* O = a.tbuf + (size_t)(t == 4 ? 0 : 2) * qstride + loff;
                store_pair_rt<NA>(x, O, O + qstride, (size_t)a.MP, t == 4 || NF == 4, M, tau);
            }
        }
    }
    cp_async_commit_wait_all();
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base_s) : "memory");
}

}  // namespace nsc
