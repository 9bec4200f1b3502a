// nonlinear_v3.cuh -- transform kernels of the nonlinear term for the line length 1536 = 2 x 768 (BASELINE.json
// configs[4]: N_r = 512, 513 x 1025 modes, the problem size of the paper's Fig. 1).  No split
// N = N1 x N2 of 1536 keeps both sides of a two-pass warp transform at <= 32 values per lane, so a line is carried by
// a PAIR of warps: each transforms one of the two decimated sequences with the 24 x 32 machinery of fft_warp.cuh and
// one radix-2 step across the pair (s2p_pair / p2s_pair) completes the transform.  Steps N1-N6, work-array layouts and
// the order of operations are those of nonlinear_v2.cuh; what changes are the index maps
//     S layout : register tt of lane tau of warp h  <->  bin  h + 2 tau + 64 tt     (live slots: tt <= 8, tt >= 16)
//     P layout : register e of lane a of warp h     <->  point a + 24 p(e) + 768 h
// and that a CTA of 8 warps serves 4 lines at a time.
#pragma once
#include "nonlinear_v2.cuh"

namespace nsc {

constexpr int P3_WARPS = 8;
constexpr int P3_THREADS = P3_WARPS * 32;
constexpr int P3_PAIRS = P3_WARPS / 2;
constexpr int P3_N = fw::NPAIR;                       // 1536
constexpr int P3_NC = P3_N / 2;                       // combine twiddles
constexpr int P3_LINE = 1032;                         // staged spectral line (>= 2 K + 1 = 1025)
constexpr int P3_STAGE = 520;                         // staged half-spectral line (>= M + 1 = 513)
constexpr int P3_TILE = P3_N * P3_PAIRS;              // [1536][4] tile (6144 complex)
constexpr int P3_NIT = P3_TILE / P3_THREADS;          // 24
constexpr size_t P3_SMEM_INV = sizeof(cd) * (size_t)(fw::XBUF * (1 + P3_WARPS) + P3_NC + P3_LINE * P3_PAIRS);
constexpr size_t P3_SMEM_FWD = sizeof(cd) * (size_t)(fw::XBUF * (1 + P3_WARPS) + P3_NC + P3_TILE);
constexpr size_t P3_SMEM_THETA = sizeof(cd) * (size_t)(fw::XBUF * (1 + P3_WARPS) + P3_NC + 2 * P3_STAGE * P3_PAIRS);
static_assert(P3_TILE <= fw::XBUF * P3_WARPS, "the tile overlays the exchange matrices");

__device__ __forceinline__ bool p3_live(int tt) { return tt <= 8 || tt >= 16; }

// ------------------------------------------------------------------------------------------ k_zinv3
// work item = (field, level, tile of 4 adjacent m); each warp pair takes one m-line
__global__ void __launch_bounds__(P3_THREADS, 1) k_zinv3(Nl2Args A) {
    using namespace fw;
    constexpr int N = P3_N, MT = P3_PAIRS;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    cd* tile = tw + XBUF;                               // [1536][4] tile, overlays the 8 matrices
    cd* twc = tw + XBUF * (1 + P3_WARPS);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    const int h = warp & 1, pair = warp >> 1;
    cd* buf = tile + warp * XBUF;
    const cd* pbuf = tile + (warp ^ 1) * XBUF;
    cd* line = twc + P3_NC + pair * P3_LINE;
    load_twiddles(tw, A.tw_z);
    for (int i = threadIdx.x; i < P3_NC; i += blockDim.x) twc[i] = A.tw_cz[i];
    const int mtiles = a.MP / MT;
    const size_t plane = (size_t)a.M1 * a.NK;
    const size_t qstride = (size_t)N * a.MP;
    const int NKc = a.NK;
    const int l64 = (h << 5) | tau;                     // lane index within the pair

    auto fetch = [&](const cd* base, int it) {
        const int mt = it % mtiles, r = it / mtiles;
        const int jl = r % a.nj;
        const int m = mt * MT + pair;
        if (m < a.M1) {
            const cd* src = base + (size_t)(a.j0 + jl) * plane + (size_t)m * NKc;
            for (int i = l64; i < NKc; i += 64) cp_async16(line + i, src + i);
        }
    };
    auto field_of = [&](int it) { return (it / mtiles) / a.nj; };
    const int ns = A.dr[0] ? 3 : 2;
    int item = blockIdx.x;
    if (item < A.nitems) fetch(a.f[field_of(item)], item);
    __syncthreads();                                    // twiddles

    for (; item < A.nitems; item += gridDim.x) {
        const int mt = item % mtiles, r = item / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
        const bool vm = (mt * MT + pair) < a.M1;
#pragma unroll 1
        for (int s = 0; s < ns; ++s) {
            const int q = (s == 0) ? 1 : (s == 1 ? 0 : 2);
            cd x[32];
            if (s != 1) {
                cp_async_commit_wait_all();
                pair_sync(pair);                        // the staged line is complete (both warps copied halves)
            }
            const double am = (s == 0) ? 0.0 : 1.0, bm = (s == 0) ? A.alpha : 0.0;
#pragma unroll
            for (int tt = 0; tt < NV; ++tt) {
                cd v = mk(0.0, 0.0);
                if (p3_live(tt)) {
                    const bool pos = tt <= 8;
                    const int bin = h + 2 * tau + 64 * tt;
                    const bool ok = vm && (pos ? (bin <= a.K) : (bin >= N - a.K));
                    const int kk = pos ? bin + a.K : bin - N + a.K;
                    const cd g = ok ? line[kk] : mk(0.0, 0.0);
                    const double kd = bm * (double)(pos ? bin : bin - N);
                    v = mk(fma(-kd, g.y, am * g.x), fma(kd, g.x, am * g.y));
                }
                x[tt] = v;
            }
            if (s >= 1) {                               // the staged line is consumed by both warps: request the next one
                pair_sync(pair);
                if (s == 1 && ns == 3) {
                    fetch(A.dr[fi], item);
                } else {
                    const int nxt = item + gridDim.x;
                    if (nxt < A.nitems) fetch(a.f[field_of(nxt)], nxt);
                }
            }
            s2p_pair<+1>(x, buf, pbuf, tw, twc, tau, h, pair);
            __syncthreads();                            // all warps left their exchange matrices
            if (tau < NV) {
#pragma unroll
                for (int e = 0; e < 32; ++e) tile[tile_pos<MT>(tau + NV * p_of(e) + P3_NC * h, pair)] = x[e];
            }
            __syncthreads();
            cd* dst = a.zbuf + ((size_t)jl * 3 * a.nf + (3 * fi + q)) * qstride + mt * MT;
            {
                cd v[P3_NIT];
#pragma unroll
                for (int it = 0; it < P3_NIT; ++it) v[it] = tile[threadIdx.x + it * P3_THREADS];
                const int z0 = threadIdx.x / MT, c0 = threadIdx.x % MT;
                cd* d0 = dst + (size_t)z0 * a.MP + (c0 ^ swz<MT>(z0));
#pragma unroll
                for (int it = 0; it < P3_NIT; ++it) d0[(size_t)((P3_THREADS / MT) * it) * a.MP] = v[it];
            }
            __syncthreads();                            // tile free again
        }
    }
    cp_async_commit_wait_all();
}

// ------------------------------------------------------------------------------------------ k_zfwd3
__global__ void __launch_bounds__(P3_THREADS, 1) k_zfwd3(Nl2Args A) {
    using namespace fw;
    constexpr int N = P3_N, MT = P3_PAIRS;
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    const int h = warp & 1, pair = warp >> 1;
    cd* buf = tw + XBUF + warp * XBUF;
    const cd* pbuf = tw + XBUF + (warp ^ 1) * XBUF;
    cd* twc = tw + XBUF * (1 + P3_WARPS);
    cd* tile = twc + P3_NC;
    load_twiddles(tw, A.tw_z);
    for (int i = threadIdx.x; i < P3_NC; i += blockDim.x) twc[i] = A.tw_cz[i];
    const int a23 = tau < NV ? tau : NV - 1;
    const int mtiles = a.MP / MT;
    const size_t qstride = (size_t)N * a.MP;

    auto fetch = [&](int it) {
        const int mt = it % mtiles, r = it / mtiles;
        const int jl = r % a.nj, fi = r / a.nj;
        const cd* src = a.tbuf + ((size_t)jl * a.nf + fi) * qstride + mt * MT;
#pragma unroll 4
        for (int k = 0; k < P3_NIT; ++k) {
            const int id = threadIdx.x + k * P3_THREADS;
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
        __syncthreads();                                 // the tile (and, first time, the twiddles) is complete
        cd x[32];
#pragma unroll
        for (int e = 0; e < 32; ++e) x[e] = tile[tile_pos<MT>(a23 + NV * p_of(e) + P3_NC * h, pair)];
        __syncthreads();                                 // every warp holds its half line: the tile is free
        if (item + (int)gridDim.x < A.nitems) fetch(item + gridDim.x);
        p2s_pair<-1>(x, buf, pbuf, tw, twc, tau, h, pair);
        const bool add_buoy = (fi == 2) && (a.buoy != 0.0);
        const int m = mt * MT + pair;
        if (m < a.M1) {
            const size_t off = ((size_t)j * a.M1 + m) * a.NK;
            cd* dst = a.out[fi] + off;
            const cd* Th = a.f[add_buoy ? 3 : 0] + off;
#pragma unroll
            for (int tt = 0; tt < NV; ++tt) {
                if (p3_live(tt)) {
                    const bool pos = tt <= 8;
                    const int bin = h + 2 * tau + 64 * tt;
                    if (pos ? (bin <= a.K) : (bin >= N - a.K)) {
                        const int kk = pos ? bin + a.K : bin - N + a.K;
                        cd v = a.scale * x[tt];
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
    cp_async_commit_wait_all();
}

// ------------------------------------------------------------------------------------------ k_theta3
// load_pair_rt / store_pair_rt of nonlinear_v2.cuh with the bin map of a warp pair: slot tt of lane tau of warp h
// holds bin h + 2 tau + 64 tt.
__device__ __forceinline__ void load_pair_rt3(cd* x, const cd* X, const cd* Y, bool dx, bool dy, int M, int tau, int h,
                                              double kth0) {
    constexpr int N = P3_N;
    // g' = (a + i b n) g with (a, b) = (1, 0) plain or (0, 1) derivative
    const double ax = dx ? 0.0 : 1.0, bx = dx ? kth0 : 0.0;
    const double ay = dy ? 0.0 : 1.0, by = dy ? kth0 : 0.0;
#pragma unroll
    for (int tt = 0; tt < fw::NV; ++tt) {
        if (!p3_live(tt)) {
            x[tt] = mk(0.0, 0.0);
        } else if (tt <= 8) {
            const int m = h + 2 * tau + 64 * tt;
            const bool ok = m <= M;
            cd gx = ok ? X[m] : mk(0.0, 0.0);
            cd gy = ok ? Y[m] : mk(0.0, 0.0);
            if (tt == 0 && m == 0) {
                gx.y = 0.0;
                gy.y = 0.0;
            }
            const double mr = (double)m;
            const double bxn = bx * mr, byn = by * mr;
            const cd hx = mk(fma(-bxn, gx.y, ax * gx.x), fma(bxn, gx.x, ax * gx.y));
            const cd hy = mk(fma(-byn, gy.y, ay * gy.x), fma(byn, gy.x, ay * gy.y));
            x[tt] = mk(hx.x - hy.y, hx.y + hy.x);
        } else {
            const int m = N - (h + 2 * tau + 64 * tt);
            const bool ok = m <= M;
            const cd gx = ok ? X[m] : mk(0.0, 0.0);
            const cd gy = ok ? Y[m] : mk(0.0, 0.0);
            const double mr = (double)m;
            const double bxn = bx * mr, byn = by * mr;
            const cd hx = mk(fma(-bxn, gx.y, ax * gx.x), fma(bxn, gx.x, ax * gx.y));
            const cd hy = mk(fma(-byn, gy.y, ay * gy.x), fma(byn, gy.x, ay * gy.y));
            x[tt] = mk(hx.x + hy.y, hy.x - hx.y);
        }
    }
}

// Z[N - m] of bin m = h + 2 tau + 64 tt lies in the same warp (N is even): warp 0 as in the length-768 case (slot
// 23 - tt of lane (32 - tau) & 31, lane 0: its own slot (24 - tt) % 24); warp 1: slot 23 - tt of lane 31 - tau.
__device__ __forceinline__ void store_pair_rt3(const cd* x, cd* outA, cd* outB, bool has_b, int M, int tau, int h) {
    const int src = h == 0 ? ((32 - tau) & 31) : (31 - tau);
#pragma unroll
    for (int tt = 0; tt <= 8; ++tt) {
        cd pz;
        if (tt == 8) {
            pz = x[16];                                  // only bin 512 (h = 0, tau = 0) can be kept: its partner is bin 1024
        } else {
            pz.x = __shfl_sync(0xffffffffu, x[23 - tt].x, src);
            pz.y = __shfl_sync(0xffffffffu, x[23 - tt].y, src);
            if (h == 0 && tau == 0) pz = x[(24 - tt) % 24];
        }
        const int m = h + 2 * tau + 64 * tt;
        if (m <= M) {
            const cd zm = conj(pz);
            outA[m] = 0.5 * (x[tt] + zm);
            if (has_b) outB[m] = 0.5 * mul_mi(x[tt] - zm);
        }
    }
}

template <int NF, bool CFL>
__global__ void __launch_bounds__(P3_THREADS, 1) k_theta3(Nl2Args A) {
    using namespace fw;
    constexpr int NT = NF == 3 ? 6 : 8;                  // inverse transforms per point-line
    const NlArgs& a = A.b;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tmem_base_s;
    cd* tw = reinterpret_cast<cd*>(smem_raw);
    const int warp = threadIdx.x >> 5, tau = threadIdx.x & 31;
    const int h = warp & 1, pair = warp >> 1;
    cd* buf = tw + XBUF * (1 + warp);
    const cd* pbuf = tw + XBUF * (1 + (warp ^ 1));
    cd* twc = tw + XBUF * (1 + P3_WARPS);
    load_twiddles(tw, A.tw_t);
    for (int i = threadIdx.x; i < P3_NC; i += blockDim.x) twc[i] = A.tw_ct[i];
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
    const double kth0 = A.ktheta0;
    const size_t qstride = (size_t)a.Nz * a.MP;
    const int nlines = a.nj * a.Nz;
    const int lstride = gridDim.x * P3_PAIRS;
    const int l64 = (h << 5) | tau;
    // the pair's staged line pair (X, Y) of the next inverse transform, filled by cp.async of both warps
    cd* stX = twc + P3_NC + 2 * P3_STAGE * pair;
    cd* stY = stX + P3_STAGE;
    auto stage = [&](int ln, int t) {
        const size_t off = ((size_t)(ln / a.Nz) * 3 * a.nf * a.Nz + ln % a.Nz) * a.MP;
        const cd* X = a.zbuf + (size_t)t2_qx(t) * qstride + off;
        const cd* Y = a.zbuf + (size_t)t2_qy(t) * qstride + off;
        for (int i = l64; i <= M; i += 64) {
            cp_async16(stX + i, X + i);
            cp_async16(stY + i, Y + i);
        }
    };
    int line = blockIdx.x * P3_PAIRS + pair;
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
            pair_sync(pair);                                   // both halves of the staged pair have arrived
            load_pair_rt3(x, stX, stY, t == 2 || t == 5, t == 3 || t == 6, M, tau, h, kth0);
            pair_sync(pair);                                   // consumed by both warps: request the next one
            if (t < NT - 1)
                stage(line, t + 1);
            else if (line + lstride < nlines)
                stage(line + lstride, 0);
            s2p_pair<+1>(x, buf, pbuf, tw, twc, tau, h, pair);
            sc_fence(sc);
            theta_products<NF, CFL>(t, x, acc, sc, ri, rj, a.cfl + 3 * (a.j0 + jl), tau);
            if (t == 4 || t == NT - 1) {                       // N5: forward transform, truncation m <= M
                p2s_pair<-1>(x, buf, pbuf, tw, twc, tau, h, pair);
                cd* O = a.tbuf + (size_t)(t == 4 ? 0 : 2) * qstride + loff;
                store_pair_rt3(x, O, O + qstride, t == 4 || NF == 4, M, tau, h);
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
