// nsc_internal.h -- context, device tables and kernel-launcher prototypes shared by the
// translation units of libnsc.so.  Not part of the ABI (that is include/nsc.h).
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <vector>
#include "../../include/nsc.h"
#include "fft.cuh"

namespace nsc {

constexpr int NPT = 9;        // finite-difference stencil length (default nine points)
constexpr int QW = 17;        // stored width of a Poisson-operator row, Q = (D1 + 1/r) G~
constexpr int MAXF = 4;       // u_r, u_theta, u_z, T

// Variable-band LU factors of one family of per-mode matrices, pair-major ("pair" = (m, |k|)):
// entry e of row j of pair p lives at  L[(offL[j] + e) * P + p],  U[(offU[j] + e) * P + p];
// U row = [1/pivot, upper entries...].
struct BandFactors {
    double* L = nullptr;
    double* U = nullptr;
    size_t nL = 0, nU = 0;    // entries per pair
};

// Row envelope of a banded matrix family: columns lo[j]..hi[j]; nl = j - lo, nu = hi - j.
struct BandShape {
    int* lo = nullptr;        // device [N_r]
    int* hi = nullptr;
    int* offL = nullptr;      // device [N_r] prefix sums of nl
    int* offU = nullptr;      // device [N_r] prefix sums of (nu + 1)
    size_t nL = 0, nU = 0;
    std::vector<int> h_lo, h_hi, h_offL, h_offU;
};

struct Tables {               // all device pointers
    double* D1 = nullptr;     // [N_r][9]   d/dr weights on the stencil s0[j]..s0[j]+8
    double* L0 = nullptr;     // [N_r][9]   d2/dr2 + (1/r) d/dr
    int* s0 = nullptr;        // [N_r]      first stencil node
    double* Q = nullptr;      // [N_r][17]  (D1 + 1/r) G~ on columns q0[j]..q0[j]+16
    int* q0 = nullptr;        // [N_r]
    double* rinv = nullptr;   // [N_r]      1 / r_j
    double* nm = nullptr;     // [M+1]      n = m k_theta0
    double* kap = nullptr;    // [2K+1]     kappa = k alpha
    cd* tw_t = nullptr;       // [N_theta]  exp(-2 pi i t / N_theta)
    cd* tw_z = nullptr;       // [N_z]
    cd* tw_wz = nullptr;      // [24][33]   twiddle matrix of fft_warp.cuh for N_z (if its length is 768 or 384)
    cd* tw_wt = nullptr;      // [24][33]   ... for N_theta
    cd* tw_c1536 = nullptr;   // [768]      exp(-2 pi i k / 1536): combine twiddles of the warp-pair transform (length 1536)
};

}  // namespace nsc

constexpr int NSC_MAX_SLICES = 8;

struct nsc_ctx {
    nsc_params p{};
    int N_r = 0, M = 0, K = 0, M1 = 0, NK = 0, MP = 0, Nt = 0, Nz = 0, nf = 3, JC = 0;
    bool heated = false;
    size_t F = 0;                         // complex elements per spectral field
    int P = 0;                            // pairs (m, |k|): (M+1)(K+1)
    cudaStream_t stream = nullptr;
    int dev = -1;                         // ordinal of the device the context was created on
    std::vector<double> r;                // radial nodes (host copy)
    nsc::Tables t;
    nsc::cd* state[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // u_r, u_theta, u_z, T, p
    nsc::cd* W[nsc::MAXF] = {nullptr, nullptr, nullptr, nullptr};        // sub-step work / predictor state
    nsc::cd* G = nullptr;                 // divergence / phi
    nsc::cd* DP = nullptr;                // D1 p of the state (fused linear path)
    // iterated corrector (nsc_step_iterated), allocated on first use: ping-pong iterates, pressure of the pass
    nsc::cd* itA[nsc::MAXF] = {nullptr, nullptr, nullptr, nullptr};
    nsc::cd* itB[nsc::MAXF] = {nullptr, nullptr, nullptr, nullptr};
    nsc::cd* itP = nullptr;
    nsc::cd* itDP = nullptr;
    double* it_acc = nullptr;
    double* diag = nullptr;               // device scratch of the diagnostics (4 doubles)
    nsc::cd* N0[nsc::MAXF] = {nullptr, nullptr, nullptr, nullptr};
    nsc::cd* N1[nsc::MAXF] = {nullptr, nullptr, nullptr, nullptr};
    nsc::cd* zbuf = nullptr;              // [JC][3 nf][N_z][MP]  z-transformed f, dz f, dr f
    nsc::cd* tbuf = nullptr;              // [JC][nf][N_z][MP]    theta-transformed products
    nsc::cd* DR[nsc::MAXF] = {nullptr, nullptr, nullptr, nullptr};       // D1 f (warp z pipeline in several chunks)
    int z_na = 0;                         // z transforms by k_dr + k_zinv2 / k_zfwd2 of fft_warp.cuh: 24 (768), 12 (384), 48 (1536, warp pairs), 0 no
    int t_na = 0;                         // theta transforms by k_theta2: 24, 12, 0 no
    unsigned long long* cfl_max = nullptr;    // [N_r][3] per-level maxima of |u| (k_theta2 / k_theta), step-size control
    bool want_cfl = false;                // the next launch_nonlinear accumulates them
    nsc::BandShape shH, shP;              // Helmholtz (9-wide rows) / Poisson (17-wide rows) envelopes
    nsc::BandFactors facH[4];             // u_+, u_-, u_z, T
    nsc::BandFactors facP;
    bool facT_shared = false;             // T shares the u_z factors (Pr == 1)
    double fac_dt = 0.0;                  // dt the Helmholtz factors were built for (0: none)
    bool facP_ready = false;
    // CUDA graph of one nsc_step (nsc_params.no_graph disables)
    bool use_graph = true;
    cudaGraphExec_t graph_exec = nullptr;
    double graph_dt = 0.0;
    cudaStream_t graph_stream = nullptr;
    long long graph_gen = -1, ptr_gen = 0, graph_launches = 0, graph_replays = 0;
    int n_slices = 2;                                 // mode slices of the linear stage (nsc_params.linear_slices)
    cudaStream_t slice_stream[NSC_MAX_SLICES] = {};   // their streams
    cudaEvent_t slice_ev[NSC_MAX_SLICES + 1] = {};    // [0] fork, [1 + s] join of slice s
    // NEXT-2 window (nsc_set_window): the nonlinear term is evaluated at the radial levels [wj0, wj1) only, the
    // sub-step for the Fourier modes [we0, we1) only (flat index m (2K+1) + k + K); default: everything
    int wj0 = 0, wj1 = 0;
    long long we0 = 0, we1 = 0;
    // asynchronous device-to-host copies of the state (nsc_get_state_host_async): snapshot + private copy stream
    nsc::cd* snap[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_snap = nullptr, ev_copied = nullptr;
    bool down_ready = false;              // snapshot set, stream and both events exist (set last by the first-use set-up)
    // asynchronous host-to-device copies (nsc_set_state_host_async): staging set + private upload stream
    nsc::cd* stage_in[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaStream_t up_stream = nullptr;
    cudaEvent_t ev_uploaded = nullptr, ev_staged_used = nullptr;
    bool up_ready = false;                // likewise for the staging set
    bool have_state = false;
    std::string err;
    long long launches = 0;
    long long dev_bytes = 0;
    std::vector<void*> allocs;
    // optional per-kernel event timing (nsc_set_profiling)
    struct ProfRec { int id; cudaEvent_t a, b; };
    bool profiling = false;
    std::vector<ProfRec> prof;
    std::vector<cudaEvent_t> ev_pool;
};

namespace nsc {

// plan.cu
int build_plan(nsc_ctx* c);

// nonlinear.cu : N(f[0..nf-1]) -> out[0..nf-1]   (steps N1-N6)
int launch_nonlinear(nsc_ctx* c, cd* const* f, cd* const* out);
// out = D1 f (radial derivative of one spectral field, all rows)
int launch_radial_derivative(nsc_ctx* c, const cd* f, cd* out);

// linear.cu
int ensure_factors(nsc_ctx* c, double dt);
// one implicit sub-step from c->state with explicit term w0*E0 + w1*E1 (E1 may be null);
// result (u, T) -> dst[0..nf-1]; new pressure -> p_dst (may be null: discarded)
int launch_substep(nsc_ctx* c, cd* const* E0, double w0, cd* const* E1, double w1, double dt,
                   cd* const* dst, cd* p_dst, cd* DP_dst = nullptr);
// d_acc[0] = sum |b - a|^2, d_acc[1] = sum |b|^2 over the nf fields (device doubles)
int launch_diff_norm(nsc_ctx* c, cd* const* a, cd* const* b, double* d_acc);
// diagnostics (NEXT-3): d_out[4] = Nu_i, Nu_o (heat), Nu_w_i, Nu_w_o (torque); d_acc = field value at (r_j, theta, z)
int launch_nusselt(nsc_ctx* c, double* d_out);
int launch_probe(nsc_ctx* c, const cd* field, int j, double theta, double z, double* d_acc);

// event brackets around a kernel launch (no-ops unless profiling is on); every launch site uses
// them, and they also count the launch.
void prof_begin(nsc_ctx* c, int kernel_id);
void prof_end(nsc_ctx* c);

// Makes `dev` the calling thread's current device for the lifetime of the guard and puts the caller's device back
// afterwards (entry points that must run on a given device whatever is current).  ok() is false if that failed.
class DeviceGuard {
    int prev_ = -1;
    bool ok_ = false;
public:
    explicit DeviceGuard(int dev) {
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess) return;
        if (cur == dev) {
            ok_ = true;
        } else if (cudaSetDevice(dev) == cudaSuccess) {
            ok_ = true;
            prev_ = cur;
        }
    }
    ~DeviceGuard() {
        if (prev_ >= 0) cudaSetDevice(prev_);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
    bool ok() const { return ok_; }
};

int fail(nsc_ctx* c, int code, const std::string& msg);
int cuda_fail(nsc_ctx* c, cudaError_t e, const char* what);

}  // namespace nsc

#define NSC_CUDA(c, call)                                                  \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) return nsc::cuda_fail((c), e__, #call);    \
    } while (0)
