// nonlinear_v2.cuh -- transform kernels of the nonlinear term specialised for line length 768
// (BASELINE.json configs[3], the headline workload: 3/2-padded 768 x 768 grid per radial node).
// Same steps N1-N6 and the same intermediate layout as nonlinear_kernels.cuh; what changes:
//
//   * the two-pass 24 x 32 transform of fft768.cuh: one shared-memory exchange per line instead of
//     two, conflict-free, one warp per line and only warp-level barriers inside a transform;
//   * k_dr     the radial derivative D1 f (N1) is taken once per evaluation by a marching kernel
//              (one thread per (m, k) column, nine levels in registers), so that no transform
//              kernel re-reads nine radial neighbours per line;
//   * k_zinv2  four adjacent m-lines per CTA; the transposed [z][m] stores go through a swizzled
//              shared-memory tile and leave as full 64-byte segments;
//   * k_theta2 one (j, z) point-line per warp, the 12 real physical-space lines exist only in
//              registers; the three velocity lines and one parked line live in a lane-private
//              scratch -- Tensor Memory (tcgen05.st / tcgen05.ld, 256 columns per warp: TMEM as
//              a 256 KB lane-private register spill space next to the 64 K registers) or shared
//              memory (fallback variant);
//   * k_zfwd2  cp.async double-buffered [z][4 m] tiles, forward transform, truncation, scaling,
//              buoyancy.
#pragma once
#include <cstdint>
#include "fft768.cuh"
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

// ------------------------------------------------------------------------------------------

// swizzled position (in 16-byte chunks) of (z, m_local) in a [768][4] tile: conflict free both for
// lanes walking z (transform side) and for lanes walking (z, m_local) row-major (global side)
__device__ __forceinline__ int tile4(int z, int ml) { return z * 4 + (ml ^ ((z >> 1) & 3)); }

// axial mode index kk = k + K of padded-line index i (i <= K or i >= 768 - K), and k as a double
struct ZBin {
    int kk;
    double kd;
    bool ok;
};
__device__ __forceinline__ ZBin z_bin(int i, int K) {
    ZBin b;
    if (i <= K) {
        b.kk = i + K;
        b.kd = (double)i;
        b.ok = true;
    } else if (i >= f768::N - K) {
        b.kk = i - f768::N + K;
        b.kd = (double)(i - f768::N);
        b.ok = true;
    } else {
        b.kk = 0;
        b.kd = 0.0;
        b.ok = false;
    }
    return b;
}

// S-layout slots that can hold non-zero spectral data when the mode count is <= 256 = 768 / 3:
// t = 0..8 (bins 0..287) and t = 16..23 (bins 512..767); t = 9..15 is always zero padding.
#define NSC_S_SLOTS(OP) OP(0) OP(1) OP(2) OP(3) OP(4) OP(5) OP(6) OP(7) OP(8) OP(16) OP(17) OP(18) OP(19) OP(20) OP(21) OP(22) OP(23)

constexpr int Z2_WARPS = 4;
constexpr int Z2_THREADS = Z2_WARPS * 32;
constexpr size_t Z2_SMEM_X = sizeof(cd) * (size_t)(f768::XBUF * (1 + Z2_WARPS));
constexpr size_t Z2_TILE = (size_t)f768::N * Z2_WARPS;                 // complex elements of one tile
constexpr size_t Z2_SMEM_FWD = Z2_SMEM_X + sizeof(cd) * Z2_TILE;     // + the second tile buffer

// ------------------------------------------------------------------------------------------ k_zinv2
// work item = (field, level, tile of 4 adjacent m); three inverse transforms per line:
// q = 1 (i kappa f), q = 0 (f), q = 2 (D1 f).  Each warp stages its spectral line in a private
// shared-memory buffer filled by cp.async one transform ahead (f for two transforms, then D1 f,
// then the next item's f), so no line waits in registers; the three transforms share one copy of
// the code (instruction cache).
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

constexpr int Z2_LINE = 520;      // complex elements of a staged spectral line (>= 2 K + 1 = 513)
constexpr size_t Z2_SMEM_INV = sizeof(cd) * (size_t)(f768::XBUF * (1 + Z2_WARPS) + Z2_LINE * Z2_WARPS);

__global__ void __launch_bounds__(Z2_THREADS, 2) k_zinv2(Nl2Args A) {
    using namespace f768;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    cd* tile = tw + XBUF;                               // [768][4] tile, overlays the 4 matrices
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    cd* buf = tile + warp * XBUF;
    cd* line = tw + XBUF * (1 + Z2_WARPS) + warp * Z2_LINE;
    load_twiddles(tw, A.tw768);
    const int mtiles = a.MP / 4;
    const size_t plane = (size_t)a.M1 * a.NK;
    const size_t qstride = (size_t)N * a.MP;
    const double taud = (double)tau;
    const int NKc = a.NK;

    // requests this warp's spectral line of item `it` from `base` (a field or its radial derivative)
    auto fetch = [&](const cd* base, int it) {
        const int mt = it % mtiles, r = it / mtiles;
        const int jl = r % a.nj;
        const int m = mt * 4 + warp;
        if (m < a.M1) {
            const cd* src = base + (size_t)(a.j0 + jl) * plane + (size_t)m * NKc;
            for (int i = tau; i < NKc; i += 32) cp_async16(line + i, src + i);
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
        const bool vm = (mt * 4 + warp) < a.M1;
#pragma unroll 1
        for (int s = 0; s < ns; ++s) {
            const int q = (s == 0) ? 1 : (s == 1 ? 0 : 2);
            cd x[32];
            if (s != 1) {
                cp_async_commit_wait_all();
                __syncwarp();
            }
            const double mult = (s == 0) ? A.alpha : 0.0;
            {
#define NSC_SET(T)                                                                              \
    {                                                                                           \
        const int kk = (T <= 8) ? tau + 32 * T + a.K : tau + 32 * T - N + a.K;                  \
        const bool ok = vm && ((T <= 8) ? (tau + 32 * T <= a.K) : (tau + 32 * T >= N - a.K));   \
        cd v = ok ? line[kk] : mk(0.0, 0.0);                                                    \
        if (s == 0) {                                                                           \
            const double kd = (T <= 8) ? taud + (double)(32 * T) : taud + (double)(32 * T - N); \
            v = (mult * kd) * mul_i(v);                                                         \
        }                                                                                       \
        x[T] = v;                                                                               \
    }
                NSC_S_SLOTS(NSC_SET)
#undef NSC_SET
#pragma unroll
                for (int t = 9; t < 16; ++t) x[t] = mk(0.0, 0.0);
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
            s2p<+1>(x, buf, tw, tau);
            // P-layout result of this warp's line -> tile -> [z][m] work array in 64-byte segments
            __syncthreads();                            // all warps left their exchange matrices
            if (tau < NA) {
#pragma unroll
                for (int e = 0; e < 32; ++e) tile[tile4(p_idx(e, tau), warp)] = x[e];
            }
            __syncthreads();
            cd* dst = a.zbuf + ((size_t)jl * 3 * a.nf + (3 * fi + q)) * qstride + mt * 4;
            // all shared-memory reads first, then all stores (the transform's registers are free here): no
            // store has to release its source registers before the next read can issue
            {
                constexpr int NIT = (N * 4) / Z2_THREADS;       // 24
                cd v[NIT];
#pragma unroll
                for (int it = 0; it < NIT; ++it) v[it] = tile[threadIdx.x + it * Z2_THREADS];
                // id = threadIdx.x + 128 it: z = id >> 2 = (threadIdx.x >> 2) + 32 it, c = id & 3 = threadIdx.x & 3
                const int z0 = threadIdx.x >> 2, c0 = threadIdx.x & 3;
                cd* d0 = dst + (size_t)z0 * a.MP + (c0 ^ ((z0 >> 1) & 3));  // (z >> 1) & 3 is the same for z0 + 32 it
#pragma unroll
                for (int it = 0; it < NIT; ++it) d0[(size_t)(32 * it) * a.MP] = v[it];
            }
            __syncthreads();                            // tile free again
        }
    }
    cp_async_commit_wait_all();
}

// ------------------------------------------------------------------------------------------ k_zfwd2
// work item = (field, level, tile of 4 adjacent m).  The [768][4] tile of theta-transformed
// products arrives by cp.async (64-byte segments) while the previous item is being transformed.

__global__ void __launch_bounds__(Z2_THREADS, 2) k_zfwd2(Nl2Args A) {
    using namespace f768;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    cd* buf = tw + XBUF + warp * XBUF;
    cd* tile = tw + XBUF * (1 + Z2_WARPS);
    load_twiddles(tw, A.tw768);
    const int a23 = tau < NA ? tau : NA - 1;
    const int mtiles = a.MP / 4;
    const size_t qstride = (size_t)N * a.MP;

    auto fetch = [&](int it) {
        const int mt = it % mtiles, r = it / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
        const cd* src = a.tbuf + ((size_t)jl * a.nf + fi) * qstride + mt * 4;
#pragma unroll 4
        for (int k = 0; k < (N * 4) / Z2_THREADS; ++k) {
            const int id = threadIdx.x + k * Z2_THREADS;
            const int z = id >> 2, c = id & 3;
            cp_async16(tile + id, src + (size_t)z * a.MP + (c ^ ((z >> 1) & 3)));
        }
    };
    int item = blockIdx.x;
    if (item < A.nitems) fetch(item);
    for (; item < A.nitems; item += gridDim.x) {
        const int mt = item % mtiles, r = item / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
        const int j = a.j0 + jl, m = mt * 4 + warp;
        cp_async_commit_wait_all();
        __syncthreads();                                 // the tile (and, first time, tw) is complete
        cd x[32];
#pragma unroll
        for (int e = 0; e < 32; ++e) x[e] = tile[tile4(p_idx(e, a23), warp)];
        __syncthreads();                                 // every warp holds its line: the tile is free
        if (item + (int)gridDim.x < A.nitems) fetch(item + gridDim.x);
        p2s<-1>(x, buf, tw, tau);
        if (m < a.M1) {
            const size_t off = ((size_t)j * a.M1 + m) * a.NK;
            cd* dst = a.out[fi] + off;
            const bool add_buoy = (fi == 2) && (a.buoy != 0.0);
            const cd* Th = a.f[add_buoy ? 3 : 0] + off;
#define NSC_ST(T)                                          \
    {                                                      \
        ZBin zb = z_bin(tau + 32 * T, a.K);                \
        if (zb.ok) {                                       \
            cd v = a.scale * x[T];                         \
            if (add_buoy) {                                \
                cd th = Th[zb.kk];                         \
                v.x = fma(a.buoy, th.x, v.x);              \
                v.y = fma(a.buoy, th.y, v.y);              \
            }                                              \
            dst[zb.kk] = v;                                \
        }                                                  \
    }
            NSC_S_SLOTS(NSC_ST)
#undef NSC_ST
        }
    }
    cp_async_commit_wait_all();
}

// ------------------------------------------------------------------------------------------ scratch
// Lane-private scratch of k_theta2: NSLOT lines of 32 doubles per lane.  Two implementations with
// the same interface: st(slot, v[32]) / ld(slot, v[32]), both warp-collective.
constexpr int T2_NSLOT = 4;            // U_r, U_theta / r, U_z, one parked line

// (1) Tensor Memory.  A CTA of 8 warps owns all 512 columns of its SM's TMEM; warp w may touch the
// 32 lanes of its quadrant (w & 3) only, so warps w and w + 4 share lanes and split the columns:
// 256 columns = 128 doubles per thread = 4 slots of 32.  tcgen05.st / .ld with shape 32x32b move one
// 32-bit column per register per lane; x16 = 8 doubles per instruction.
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
    __device__ __forceinline__ void ld8(uint32_t addr, double* v) const {
        uint32_t r[16];
        ld8_raw(addr, r);
        wait_ld();
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = __hiloint2double((int)r[2 * i + 1], (int)r[2 * i]);
    }
    // the registers of every ld8 issued so far are valid after this
    __device__ __forceinline__ void wait_ld() const { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ void st(int slot, const double* v) const {
#pragma unroll
        for (int c = 0; c < 4; ++c) st8(base + slot * 64 + c * 16, v + 8 * c);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    __device__ __forceinline__ void ld(int slot, double* v) const {
#pragma unroll
        for (int c = 0; c < 4; ++c) ld8(base + slot * 64 + c * 16, v + 8 * c);
    }
};

// (2) shared memory: [slot][e][24 lanes] doubles per warp (lanes >= 24 hold nothing)
struct SmemScratch {
    double* base;         // this warp's block of T2_NSLOT * 32 * 24 doubles, already offset by the lane
    bool active;
    __device__ __forceinline__ void st(int slot, const double* v) const {
        if (active)
#pragma unroll
            for (int e = 0; e < 32; ++e) base[(slot * 32 + e) * f768::NA] = v[e];
    }
    __device__ __forceinline__ void ld(int slot, double* v) const {
#pragma unroll
        for (int e = 0; e < 32; ++e) v[e] = base[(slot * 32 + e) * f768::NA];
    }
};

template <bool TMEM> struct T2Cfg;
constexpr int T2_STAGE = 264;      // complex elements of one staged half-spectral line (>= M + 1 = 257)
template <> struct T2Cfg<true> {
    static constexpr int WARPS = 8;
    using Scratch = TmemScratch;
    // twiddles + one exchange matrix and one staged line pair per warp; more than half of the SM's
    // shared memory, so exactly one CTA (the owner of all 512 TMEM columns) is resident per SM
    static constexpr size_t SMEM = sizeof(cd) * ((size_t)f768::XBUF * (1 + WARPS) + (size_t)2 * T2_STAGE * WARPS);
};
template <> struct T2Cfg<false> {
    static constexpr int WARPS = 5;
    using Scratch = SmemScratch;
    static constexpr size_t SMEM = sizeof(cd) * ((size_t)f768::XBUF * (1 + WARPS) + (size_t)2 * T2_STAGE * WARPS) +
                                   sizeof(double) * (size_t)WARPS * T2_NSLOT * 32 * f768::NA;
};

// chunked access (8 doubles = elements 8 c .. 8 c + 7 of a slot)
__device__ __forceinline__ void sc_st8(const TmemScratch& s, int slot, int c, const double* v) {
    s.st8(s.base + slot * 64 + c * 16, v);
}
__device__ __forceinline__ void sc_ld8(const TmemScratch& s, int slot, int c, double* v) {
    s.ld8(s.base + slot * 64 + c * 16, v);
}
__device__ __forceinline__ void sc_fence(const TmemScratch&) {
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void sc_st8(const SmemScratch& s, int slot, int c, const double* v) {
    if (s.active)
#pragma unroll
        for (int i = 0; i < 8; ++i) s.base[(slot * 32 + c * 8 + i) * f768::NA] = v[i];
}
__device__ __forceinline__ void sc_ld8(const SmemScratch& s, int slot, int c, double* v) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = s.base[(slot * 32 + c * 8 + i) * f768::NA];
}
__device__ __forceinline__ void sc_fence(const SmemScratch&) {}
// split form: sc_ld8_raw (issue) ... sc_wait_ld ... sc_unpack8 (use), so that several loads share one wait
struct Raw8 {
    uint32_t r[16];
};
__device__ __forceinline__ void sc_ld8_raw(const TmemScratch& s, int slot, int c, Raw8& q) {
    s.ld8_raw(s.base + slot * 64 + c * 16, q.r);
}
__device__ __forceinline__ void sc_ld8_raw(const SmemScratch& s, int slot, int c, Raw8& q) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const double v = s.base[(slot * 32 + c * 8 + i) * f768::NA];
        q.r[2 * i] = (uint32_t)__double2loint(v);
        q.r[2 * i + 1] = (uint32_t)__double2hiint(v);
    }
}
__device__ __forceinline__ void sc_wait_ld(const TmemScratch& s) { s.wait_ld(); }
__device__ __forceinline__ void sc_wait_ld(const SmemScratch&) {}
__device__ __forceinline__ void sc_unpack8(const Raw8& q, double* v) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __hiloint2double((int)q.r[2 * i + 1], (int)q.r[2 * i]);
}

// ------------------------------------------------------------------------------------------ k_theta2
// Z[i] = G_X(i) + i G_Y(i) in the S layout, G(m) = mult * line[m] (0 <= m <= M), G(-m) = conj G(m),
// Im G(0) dropped (R6); mult = 1 or i n_m (d/dtheta, N1).  Slots t = 9..15 are zero padding.
template <bool DX, bool DY, bool HAS_Y>
__device__ __forceinline__ void load_pair768(cd* x, const cd* X, const cd* Y, int M, int tau, double taud,
                                             double kth0) {
#define NSC_POS(T)                                                    \
    {                                                                 \
        const int m = tau + 32 * T;                                   \
        const bool ok = m <= M;                                       \
        cd gx = ok ? X[m] : mk(0.0, 0.0);                             \
        cd gy = (HAS_Y && ok) ? Y[m] : mk(0.0, 0.0);                  \
        const double n = kth0 * (taud + (double)(32 * T));            \
        if (DX) gx = n * mul_i(gx);                                   \
        if (DY) gy = n * mul_i(gy);                                   \
        if (T == 0 && tau == 0) {                                     \
            gx.y = 0.0;                                               \
            gy.y = 0.0;                                               \
        }                                                             \
        x[T] = mk(gx.x - gy.y, gx.y + gy.x);                          \
    }
#define NSC_NEG(T)                                                    \
    {                                                                 \
        const int m = f768::N - 32 * T - tau;                         \
        const bool ok = m <= M;                                       \
        cd gx = ok ? X[m] : mk(0.0, 0.0);                             \
        cd gy = (HAS_Y && ok) ? Y[m] : mk(0.0, 0.0);                  \
        const double n = kth0 * ((double)(f768::N - 32 * T) - taud);  \
        if (DX) gx = n * mul_i(gx);                                   \
        if (DY) gy = n * mul_i(gy);                                   \
        x[T] = mk(gx.x + gy.y, gy.x - gx.y);                          \
    }
    NSC_POS(0) NSC_POS(1) NSC_POS(2) NSC_POS(3) NSC_POS(4) NSC_POS(5) NSC_POS(6) NSC_POS(7) NSC_POS(8)
#pragma unroll
    for (int t = 9; t < 16; ++t) x[t] = mk(0.0, 0.0);
    NSC_NEG(16) NSC_NEG(17) NSC_NEG(18) NSC_NEG(19) NSC_NEG(20) NSC_NEG(21) NSC_NEG(22) NSC_NEG(23)
#undef NSC_POS
#undef NSC_NEG
}

// Splits the forward transform Z (S layout) of a packed real pair (a + i b) into the Hermitian half
// lines A[m] = (Z[m] + conj Z[N-m]) / 2, B[m] = (Z[m] - conj Z[N-m]) / (2 i), m <= M (N5 truncation).
// Z[N-m] of lane tau, slot T sits in lane (32 - tau) & 31, slot 23 - T (lane 0: its own slot 24 - T).
template <bool HAS_B>
__device__ __forceinline__ void store_pair768(const cd* x, cd* outA, cd* outB, int M, int tau) {
    const int src = (32 - tau) & 31;
#define NSC_OUT(T)                                                                 \
    {                                                                              \
        cd pz;                                                                     \
        if (T == 8) {                                                              \
            pz = x[16];                                                            \
        } else {                                                                   \
            pz.x = __shfl_sync(0xffffffffu, x[23 - T].x, src);                     \
            pz.y = __shfl_sync(0xffffffffu, x[23 - T].y, src);                     \
            if (tau == 0) pz = (T == 0) ? x[0] : x[(24 - T) % 24];                 \
        }                                                                          \
        const int m = tau + 32 * T;                                                \
        if (m <= M) {                                                              \
            const cd zm = conj(pz);                                                \
            outA[m] = 0.5 * (x[T] + zm);                                           \
            if (HAS_B) outB[m] = 0.5 * mul_mi(x[T] - zm);                          \
        }                                                                          \
    }
    NSC_OUT(0) NSC_OUT(1) NSC_OUT(2) NSC_OUT(3) NSC_OUT(4) NSC_OUT(5) NSC_OUT(6) NSC_OUT(7) NSC_OUT(8)
#undef NSC_OUT
}

__device__ __forceinline__ void store_pair768_rt(const cd* x, cd* outA, cd* outB, bool HAS_B, int M, int tau) {
    const int src = (32 - tau) & 31;
#define NSC_OUT(T)                                                                 \
    {                                                                              \
        cd pz;                                                                     \
        if (T == 8) {                                                              \
            pz = x[16];                                                            \
        } else {                                                                   \
            pz.x = __shfl_sync(0xffffffffu, x[23 - T].x, src);                     \
            pz.y = __shfl_sync(0xffffffffu, x[23 - T].y, src);                     \
            if (tau == 0) pz = (T == 0) ? x[0] : x[(24 - T) % 24];                 \
        }                                                                          \
        const int m = tau + 32 * T;                                                \
        if (m <= M) {                                                              \
            const cd zm = conj(pz);                                                \
            outA[m] = 0.5 * (x[T] + zm);                                           \
            if (HAS_B) outB[m] = 0.5 * mul_mi(x[T] - zm);                          \
        }                                                                          \
    }
    NSC_OUT(0) NSC_OUT(1) NSC_OUT(2) NSC_OUT(3) NSC_OUT(4) NSC_OUT(5) NSC_OUT(6) NSC_OUT(7) NSC_OUT(8)
#undef NSC_OUT
}

__device__ __forceinline__ void prefetch_l2(const void* p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// run-time variant of load_pair768: one copy of the code serves all six inverse transforms of a
// point-line, which keeps the kernel inside the instruction cache.  dx / dy select the d/dtheta
// multiplier i n of the X / Y half; the four transforms without a derivative take the short branch
// (uniform per warp), the other two blend (1, 0) / (0, n) multipliers arithmetically (no selects).
__device__ __forceinline__ void load_pair768_rt(cd* x, const cd* X, const cd* Y, bool dx, bool dy, int M, int tau,
                                                double taud, double kth0) {
    if (!(dx || dy)) {
#define NSC_POS(T)                                                    \
    {                                                                 \
        const int m = tau + 32 * T;                                   \
        const bool ok = m <= M;                                       \
        cd gx = ok ? X[m] : mk(0.0, 0.0);                             \
        cd gy = ok ? Y[m] : mk(0.0, 0.0);                             \
        if (T == 0 && tau == 0) {                                     \
            gx.y = 0.0;                                               \
            gy.y = 0.0;                                               \
        }                                                             \
        x[T] = mk(gx.x - gy.y, gx.y + gy.x);                          \
    }
#define NSC_NEG(T)                                                    \
    {                                                                 \
        const int m = f768::N - 32 * T - tau;                         \
        const bool ok = m <= M;                                       \
        const cd gx = ok ? X[m] : mk(0.0, 0.0);                       \
        const cd gy = ok ? Y[m] : mk(0.0, 0.0);                       \
        x[T] = mk(gx.x + gy.y, gy.x - gx.y);                          \
    }
        NSC_POS(0) NSC_POS(1) NSC_POS(2) NSC_POS(3) NSC_POS(4) NSC_POS(5) NSC_POS(6) NSC_POS(7) NSC_POS(8)
        NSC_NEG(16) NSC_NEG(17) NSC_NEG(18) NSC_NEG(19) NSC_NEG(20) NSC_NEG(21) NSC_NEG(22) NSC_NEG(23)
#undef NSC_POS
#undef NSC_NEG
    } else {
        // g' = (a + i b n) g with (a, b) = (1, 0) plain or (0, 1) derivative
        const double ax = dx ? 0.0 : 1.0, bx = dx ? kth0 : 0.0;
        const double ay = dy ? 0.0 : 1.0, by = dy ? kth0 : 0.0;
#define NSC_POS(T)                                                    \
    {                                                                 \
        const int m = tau + 32 * T;                                   \
        const bool ok = m <= M;                                       \
        cd gx = ok ? X[m] : mk(0.0, 0.0);                             \
        cd gy = ok ? Y[m] : mk(0.0, 0.0);                             \
        if (T == 0 && tau == 0) {                                     \
            gx.y = 0.0;                                               \
            gy.y = 0.0;                                               \
        }                                                             \
        const double mr = taud + (double)(32 * T);                    \
        const double bxn = bx * mr, byn = by * mr;                    \
        const cd hx = mk(fma(-bxn, gx.y, ax * gx.x), fma(bxn, gx.x, ax * gx.y)); \
        const cd hy = mk(fma(-byn, gy.y, ay * gy.x), fma(byn, gy.x, ay * gy.y)); \
        x[T] = mk(hx.x - hy.y, hx.y + hy.x);                          \
    }
#define NSC_NEG(T)                                                    \
    {                                                                 \
        const int m = f768::N - 32 * T - tau;                         \
        const bool ok = m <= M;                                       \
        const cd gx = ok ? X[m] : mk(0.0, 0.0);                       \
        const cd gy = ok ? Y[m] : mk(0.0, 0.0);                       \
        const double mr = (double)(f768::N - 32 * T) - taud;          \
        const double bxn = bx * mr, byn = by * mr;                    \
        const cd hx = mk(fma(-bxn, gx.y, ax * gx.x), fma(bxn, gx.x, ax * gx.y)); \
        const cd hy = mk(fma(-byn, gy.y, ay * gy.x), fma(byn, gy.x, ay * gy.y)); \
        x[T] = mk(hx.x + hy.y, hy.x - hx.y);                          \
    }
        NSC_POS(0) NSC_POS(1) NSC_POS(2) NSC_POS(3) NSC_POS(4) NSC_POS(5) NSC_POS(6) NSC_POS(7) NSC_POS(8)
        NSC_NEG(16) NSC_NEG(17) NSC_NEG(18) NSC_NEG(19) NSC_NEG(20) NSC_NEG(21) NSC_NEG(22) NSC_NEG(23)
#undef NSC_POS
#undef NSC_NEG
    }
#pragma unroll
    for (int t = 9; t < 16; ++t) x[t] = mk(0.0, 0.0);
}

// The six inverse transforms of a point-line as a table: work array index q = 3 field + kind
// (kind 0 f, 1 d_z f, 2 d_r f) of the X and Y halves of the packed pair, d/dtheta flags.
//   t : 0 (u_r, u_th)  1 (u_z, dr u_r)  2 (dth u_r, dz u_r)  3 (dr u_th, dth u_th)  4 (dz u_th, dr u_z)  5 (dth u_z, dz u_z)
__device__ __forceinline__ int t2_qx(int t) { return (0x645060 >> (4 * t)) & 15; }
__device__ __forceinline__ int t2_qy(int t) { return (0x783123 >> (4 * t)) & 15; }

template <bool TMEM>
__global__ void __launch_bounds__(T2Cfg<TMEM>::WARPS * 32, 1) k_theta2(Nl2Args A) {
    using namespace f768;
    using Cfg = T2Cfg<TMEM>;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tmem_base_s;
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    cd* buf = tw + XBUF * (1 + warp);
    const int a23 = tau < NA ? tau : NA - 1;
    load_twiddles(tw, A.tw768);
    typename Cfg::Scratch sc;
    if constexpr (TMEM) {
        if (warp == 0) {
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&tmem_base_s);
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(dst) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        sc.base = tmem_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 256);
    } else {
        double* sb = reinterpret_cast<double*>(tw + XBUF * (1 + Cfg::WARPS) + 2 * T2_STAGE * Cfg::WARPS);
        sc.base = sb + (size_t)warp * T2_NSLOT * 32 * NA + a23;
        sc.active = tau < NA;
        __syncthreads();
    }
    const int M = a.M;
    const double taud = (double)tau, kth0 = A.ktheta0;
    const size_t qstride = (size_t)a.Nz * a.MP;
    const int nlines = a.nj * a.Nz;
    const int lstride = gridDim.x * Cfg::WARPS;
    // this warp's staged line pair (X, Y) of the next inverse transform, filled by cp.async
    cd* stX = tw + XBUF * (1 + Cfg::WARPS) + 2 * T2_STAGE * warp;
    cd* stY = stX + T2_STAGE;
    auto stage = [&](int ln, int t) {
        const size_t off = ((size_t)(ln / a.Nz) * 3 * a.nf * a.Nz + ln % a.Nz) * a.MP;
        const cd* X = a.zbuf + (size_t)t2_qx(t) * qstride + off;
        const cd* Y = a.zbuf + (size_t)t2_qy(t) * qstride + off;
        for (int i = tau; i <= M; i += 32) {
            cp_async16(stX + i, X + i);
            cp_async16(stY + i, Y + i);
        }
    };
    int line = blockIdx.x * Cfg::WARPS + warp;
    if (line < nlines) stage(line, 0);
    for (; line < nlines; line += lstride) {
        const int jl = line / a.Nz;
        const size_t loff = ((size_t)jl * a.nf * a.Nz + line % a.Nz) * a.MP;   // line (j, z) of q = 0 in tbuf
        const double ri = a.rinv[a.j0 + jl];
        const double rj = 1.0 / ri;
        cd x[32];
        double acc[32];
#pragma unroll 1
        for (int t = 0; t < 6; ++t) {
            cp_async_commit_wait_all();
            __syncwarp();
            load_pair768_rt(x, stX, stY, t == 2 || t == 5, t == 3, M, tau, taud, kth0);
            __syncwarp();                                      // the staged pair is consumed: request the next one
            if (t < 5)
                stage(line, t + 1);
            else if (line + lstride < nlines)
                stage(line + lstride, 0);
            s2p<+1>(x, buf, tw, tau);
            sc_fence(sc);
            // physical-space stage (N4): slots 0 U_r, 1 U_theta / r, 2 U_z, 3 parked line
            if (t == 0) {
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
            } else if (t == 3) {                               // acc = U_r d_r u_th + (U_th / r) d_th u_th
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
            } else {                                           // N_z = -(u.grad u_z)  (buoyancy: k_zfwd)
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
                        x[8 * c + i] = mk(-s, 0.0);
                    }
                }
            }
            if (t >= 4) {                                      // N5: forward transform, truncation m <= M
                p2s<-1>(x, buf, tw, tau);
                cd* O = a.tbuf + (size_t)(t == 4 ? 0 : 2) * qstride + loff;
                store_pair768_rt(x, O, O + qstride, t == 4, M, tau);
            }
        }
    }
    cp_async_commit_wait_all();
    if constexpr (TMEM) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (warp == 0)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base_s) : "memory");
    }
}

}  // namespace nsc
