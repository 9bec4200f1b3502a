// api.cu -- the C ABI of include/nsc.h: argument checks, allocation, and the composition of
// one predictor-corrector step (O7) from the kernels of nonlinear.cu
// and linear.cu.  No arithmetic of the method happens on the host after nsc_create.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>
#include <vector>
#include "nsc_internal.h"

namespace nsc {

bool fft_length_supported(int n);
int warp_na(int n, int modes);

static thread_local std::string g_create_err;

int fail(nsc_ctx* c, int code, const std::string& msg) {
    if (c)
        c->err = msg;
    else
        g_create_err = msg;
    return code;
}

int cuda_fail(nsc_ctx* c, cudaError_t e, const char* what) {
    std::string m = std::string(what) + ": " + cudaGetErrorString(e);
    fail(c, NSC_ECUDA, m);
    return e == cudaErrorMemoryAllocation ? NSC_ENOMEM : NSC_ECUDA;
}

static int dev_alloc(nsc_ctx* c, cd** dst, size_t elems, bool zero) {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, elems * sizeof(cd));
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaMalloc(field)");
    c->allocs.push_back(p);
    c->dev_bytes += (long long)(elems * sizeof(cd));
    if (zero) {
        e = cudaMemset(p, 0, elems * sizeof(cd));
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaMemset(field)");
    }
    *dst = (cd*)p;
    return NSC_OK;
}

static cudaEvent_t get_event(nsc_ctx* c) {
    if (!c->ev_pool.empty()) {
        cudaEvent_t e = c->ev_pool.back();
        c->ev_pool.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}

void prof_begin(nsc_ctx* c, int kernel_id) {
    c->launches += 1;
    if (!c->profiling) return;
    nsc_ctx::ProfRec r{kernel_id, get_event(c), get_event(c)};
    cudaEventRecord(r.a, c->stream);
    c->prof.push_back(r);
}

void prof_end(nsc_ctx* c) {
    if (!c->profiling) return;
    cudaEventRecord(c->prof.back().b, c->stream);
}

static const char* kKernelNames[NSC_NKERN] = {"k_zinv", "k_theta", "k_zfwd", "k_rhs_fwd", "k_bwd_div",
                                              "k_diff_norm", "k_nusselt / k_probe", "k_poisson_fwd", "k_poisson_bwd_correct",
                                              "k_factor", "k_dr"};

}  // namespace nsc

using namespace nsc;

extern "C" {

int nsc_create_ex(nsc_ctx** out, const nsc_params* pp) {
    if (!out || !pp) return fail(nullptr, NSC_EINVAL, "nsc_create: NULL argument");
    nsc_params p = *pp;
    if (p.N_r < NPT) return fail(nullptr, NSC_EINVAL, "nsc_create: N_r must be >= 9");
    if (p.M_theta < 1 || p.M_theta > 512 || p.K_z < 1 || p.K_z > 512)
        return fail(nullptr, NSC_EINVAL, "nsc_create: M_theta and K_z must be in [1, 512]");
    if (!(p.eta > 0.0 && p.eta < 1.0)) return fail(nullptr, NSC_EINVAL, "nsc_create: eta must be in (0, 1)");
    if (!(p.alpha > 0.0)) return fail(nullptr, NSC_EINVAL, "nsc_create: alpha must be > 0");
    if (p.k_theta0 < 1) return fail(nullptr, NSC_EINVAL, "nsc_create: k_theta0 must be >= 1");
    if (p.Ra != 0.0 && !(p.Pr > 0.0)) return fail(nullptr, NSC_EINVAL, "nsc_create: Pr must be > 0 when Ra != 0");
    if (p.radial_grid != 0 && p.radial_grid != 1) return fail(nullptr, NSC_EINVAL, "nsc_create: radial_grid must be 0 or 1");
    // default physical grid: the shortest supported transform length (3 * 2^p, 12..1536) that holds the 3/2 rule
    auto default_len = [](int modes) {
        int n = 12;
        while (n < 3 * modes) n *= 2;
        return n;
    };
    if (p.n_theta_phys == 0) p.n_theta_phys = default_len(p.M_theta);
    if (p.n_z_phys == 0) p.n_z_phys = default_len(p.K_z);
    if (p.n_theta_phys < 3 * p.M_theta || p.n_z_phys < 3 * p.K_z || !fft_length_supported(p.n_theta_phys) ||
        !fft_length_supported(p.n_z_phys))
        return fail(nullptr, NSC_EINVAL, "nsc_create: unsupported physical grid size");
    if (p.c == 0.0) p.c = 0.5;
    if (!(p.c > 0.0 && p.c <= 1.0)) return fail(nullptr, NSC_EINVAL, "nsc_create: c must be in (0, 1]");
    if (p.Ra == 0.0) p.Pr = 1.0;

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, NSC_ECUDA, "nsc_create: no CUDA device (there is no CPU fallback)");
    }
    if (p.device >= 0) {
        e = cudaSetDevice(p.device);
        if (e != cudaSuccess) return fail(nullptr, NSC_ECUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e));
    }
    nsc_ctx* c = new (std::nothrow) nsc_ctx();
    if (!c) return fail(nullptr, NSC_ENOMEM, "nsc_create: out of host memory");
    c->p = p;
    cudaGetDevice(&c->dev);
    c->N_r = p.N_r;
    c->M = p.M_theta;
    c->K = p.K_z;
    c->M1 = c->M + 1;
    c->NK = 2 * c->K + 1;
    c->MP = (c->M1 + 7) / 8 * 8;
    c->Nt = p.n_theta_phys;
    c->Nz = p.n_z_phys;
    c->heated = p.Ra != 0.0;
    c->nf = c->heated ? 4 : 3;
    c->F = (size_t)c->N_r * c->M1 * c->NK;
    c->wj1 = c->N_r;
    c->we1 = (long long)c->M1 * c->NK;
    c->P = c->M1 * (c->K + 1);
    // radial chunk of the transform pipeline: work arrays of ~2 GiB unless told otherwise
    // default: the whole radius at once when the work arrays stay below an eighth of the device memory
    // (cfg 4: 10 GB), else chunks of ~2 GiB
    const size_t per_level = (size_t)4 * c->nf * c->Nz * c->MP * sizeof(cd);
    size_t mem_free = 0, mem_total = 0;
    cudaMemGetInfo(&mem_free, &mem_total);
    int jc = p.radial_chunk > 0 ? p.radial_chunk
             : (per_level * (size_t)p.N_r <= mem_total / 8 ? p.N_r : (int)(((size_t)2 << 30) / per_level));
    if (jc < 1) jc = 1;
    if (jc > c->N_r) jc = c->N_r;
    c->JC = jc;

    // warp-transform pipeline for the lengths 768 and 384 (nonlinear_v2.cuh)
    c->z_na = warp_na(c->Nz, c->K);
    c->t_na = warp_na(c->Nt, c->M);
    int rc = build_plan(c);
    if (!rc && c->z_na && c->JC < c->N_r)     // D1 f arrays of the multi-chunk transform pipeline
        for (int i = 0; i < c->nf && !rc; ++i) rc = dev_alloc(c, &c->DR[i], c->F, false);
    if (!rc) {
        for (int i = 0; i < 5 && !rc; ++i)
            if (i != 3 || c->heated) rc = dev_alloc(c, &c->state[i], c->F, true);
        for (int i = 0; i < c->nf && !rc; ++i) rc = dev_alloc(c, &c->W[i], c->F, false);
        for (int i = 0; i < c->nf && !rc; ++i) rc = dev_alloc(c, &c->N0[i], c->F, false);
        for (int i = 0; i < c->nf && !rc; ++i) rc = dev_alloc(c, &c->N1[i], c->F, false);
        if (!rc) rc = dev_alloc(c, &c->G, c->F, false);
        if (!rc) rc = dev_alloc(c, &c->DP, c->F, true);
        if (!rc) rc = dev_alloc(c, &c->zbuf, (size_t)3 * c->nf * c->JC * c->Nz * c->MP, true);
        if (!rc) rc = dev_alloc(c, &c->tbuf, (size_t)c->nf * c->JC * c->Nz * c->MP, true);
    }
    c->use_graph = p.no_graph == 0;
    c->n_slices = p.linear_slices > 0 ? p.linear_slices : 2;
    if (c->n_slices < 1) c->n_slices = 1;
    if (c->n_slices > NSC_MAX_SLICES) c->n_slices = NSC_MAX_SLICES;
    for (int i = 0; i < c->n_slices && !rc && c->n_slices > 1; ++i)
        if (cudaStreamCreateWithFlags(&c->slice_stream[i], cudaStreamNonBlocking) != cudaSuccess) rc = fail(c, NSC_ECUDA, "cudaStreamCreate");
    for (int i = 0; i <= c->n_slices && !rc; ++i)
        if (cudaEventCreateWithFlags(&c->slice_ev[i], cudaEventDisableTiming) != cudaSuccess) rc = fail(c, NSC_ECUDA, "cudaEventCreate");
    if (!rc) {
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) rc = cuda_fail(c, e, "nsc_create: cudaDeviceSynchronize");
    }
    if (rc) {
        g_create_err = c->err;
        nsc_destroy(c);
        return rc;
    }
    *out = c;
    return NSC_OK;
}

int nsc_create(nsc_ctx** out, int N_r, int M_theta, int K_z, double eta, double alpha, int k_theta0, double Re_i,
               double Re_o, double Ra, double Pr, int radial_grid) {
    nsc_params p;
    memset(&p, 0, sizeof(p));
    p.N_r = N_r;
    p.M_theta = M_theta;
    p.K_z = K_z;
    p.eta = eta;
    p.alpha = alpha;
    p.k_theta0 = k_theta0;
    p.Re_i = Re_i;
    p.Re_o = Re_o;
    p.Ra = Ra;
    p.Pr = Pr;
    p.radial_grid = radial_grid;
    p.device = -1;
    return nsc_create_ex(out, &p);
}

int nsc_destroy(nsc_ctx* c) {
    if (!c) return NSC_OK;
    cudaDeviceSynchronize();
    for (void* p : c->allocs) cudaFree(p);
    for (auto& r : c->prof) {
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    for (cudaStream_t s : c->slice_stream)
        if (s) cudaStreamDestroy(s);
    for (cudaEvent_t e : c->slice_ev)
        if (e) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->up_stream) cudaStreamDestroy(c->up_stream);
    if (c->ev_uploaded) cudaEventDestroy(c->ev_uploaded);
    if (c->ev_staged_used) cudaEventDestroy(c->ev_staged_used);
    if (c->ev_snap) cudaEventDestroy(c->ev_snap);
    if (c->ev_copied) cudaEventDestroy(c->ev_copied);
    cudaGetLastError();
    delete c;
    return NSC_OK;
}

int nsc_set_stream(nsc_ctx* c, void* s) {
    if (!c) return NSC_EINVAL;
    c->stream = (cudaStream_t)s;
    return NSC_OK;
}

int nsc_get_grid(const nsc_ctx* c, double* h_r) {
    if (!c || !h_r) return NSC_EINVAL;
    memcpy(h_r, c->r.data(), sizeof(double) * c->N_r);
    return NSC_OK;
}

static int copy_state(nsc_ctx* c, const void* const* src, void* const* dst, cudaMemcpyKind kind, bool set) {
    for (int i = 0; i < 5; ++i) {
        if (i == 3 && !c->heated) continue;
        const size_t bytes = c->F * sizeof(cd);
        if (set) {
            if (src[i])
                NSC_CUDA(c, cudaMemcpyAsync(c->state[i], src[i], bytes, kind, c->stream));
            else if (i == 4)
                NSC_CUDA(c, cudaMemsetAsync(c->state[4], 0, bytes, c->stream));
            else
                return fail(c, NSC_EINVAL, "nsc_set_state: required field pointer is NULL");
        } else if (dst[i]) {
            NSC_CUDA(c, cudaMemcpyAsync(dst[i], c->state[i], bytes, kind, c->stream));
        }
    }
    return NSC_OK;
}

// derived arrays of a new state: D1 p for the fused linear path
static int after_set_state(nsc_ctx* c) {
    if (c->DP) {
        int rc = launch_radial_derivative(c, c->state[4], c->DP);
        if (rc) return rc;
    }
    c->have_state = true;
    return NSC_OK;
}

int nsc_set_state(nsc_ctx* c, const void* ur, const void* uth, const void* uz, const void* T, const void* p) {
    if (!c) return NSC_EINVAL;
    const void* src[5] = {ur, uth, uz, T, p};
    int rc = copy_state(c, src, nullptr, cudaMemcpyDeviceToDevice, true);
    if (!rc) rc = after_set_state(c);
    return rc;
}

int nsc_get_state(nsc_ctx* c, void* ur, void* uth, void* uz, void* T, void* p) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_get_state before nsc_set_state");
    void* dst[5] = {ur, uth, uz, T, p};
    return copy_state(c, nullptr, dst, cudaMemcpyDeviceToDevice, false);
}

int nsc_set_state_host(nsc_ctx* c, const void* ur, const void* uth, const void* uz, const void* T, const void* p) {
    if (!c) return NSC_EINVAL;
    const void* src[5] = {ur, uth, uz, T, p};
    int rc = copy_state(c, src, nullptr, cudaMemcpyHostToDevice, true);
    if (rc) return rc;
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    return after_set_state(c);
}

int nsc_get_state_host(nsc_ctx* c, void* ur, void* uth, void* uz, void* T, void* p) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_get_state_host before nsc_set_state");
    void* dst[5] = {ur, uth, uz, T, p};
    int rc = copy_state(c, nullptr, dst, cudaMemcpyDeviceToHost, false);
    if (rc) return rc;
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    return NSC_OK;
}

// First-use set-up shared by the two double-buffered transfers: one buffer set of the state's size, a private stream
// and two events, the second of which is recorded once on `first_on` so that the first wait finds it signalled.
// `*ready` is set last.  A call that failed halfway leaves what it created in place (owned by the context, released by
// nsc_destroy); the next call creates only what is still missing instead of allocating everything again or running
// with null events.
static int transfer_setup(nsc_ctx* c, cd** bufs, cudaStream_t* priv, cudaEvent_t* ev_a, cudaEvent_t* ev_b,
                          bool first_on_private, bool* ready) {
    if (*ready) return NSC_OK;
    int rc;
    for (int i = 0; i < 5; ++i)
        if ((i != 3 || c->heated) && !bufs[i] && (rc = dev_alloc(c, &bufs[i], c->F, false))) return rc;
    if (!*priv) NSC_CUDA(c, cudaStreamCreateWithFlags(priv, cudaStreamNonBlocking));
    if (!*ev_a) NSC_CUDA(c, cudaEventCreateWithFlags(ev_a, cudaEventDisableTiming));
    if (!*ev_b) NSC_CUDA(c, cudaEventCreateWithFlags(ev_b, cudaEventDisableTiming));
    NSC_CUDA(c, cudaEventRecord(*ev_b, first_on_private ? *priv : c->stream));
    *ready = true;
    return NSC_OK;
}

// Double-buffered read-out: the state is snapshot on the context's stream (device to device), the snapshot leaves for
// the host on a private stream, and the call returns; the next step and the next host-to-device copy overlap with it.
int nsc_get_state_host_async(nsc_ctx* c, void* ur, void* uth, void* uz, void* T, void* p) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_get_state_host_async before nsc_set_state");
    if (T && !c->heated)
        return fail(c, NSC_EINVAL, "nsc_get_state_host_async: a temperature buffer was given, but the context has no temperature field (Ra = 0)");
    void* dst[5] = {ur, uth, uz, T, p};
    int rc = transfer_setup(c, c->snap, &c->copy_stream, &c->ev_snap, &c->ev_copied, true, &c->down_ready);
    if (rc) return rc;
    const size_t bytes = c->F * sizeof(cd);
    NSC_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_copied, 0));        // the previous snapshot has left
    for (int i = 0; i < 5; ++i)
        if (dst[i] && c->snap[i]) NSC_CUDA(c, cudaMemcpyAsync(c->snap[i], c->state[i], bytes, cudaMemcpyDeviceToDevice, c->stream));
    NSC_CUDA(c, cudaEventRecord(c->ev_snap, c->stream));
    NSC_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev_snap, 0));
    for (int i = 0; i < 5; ++i)
        if (dst[i] && c->snap[i]) NSC_CUDA(c, cudaMemcpyAsync(dst[i], c->snap[i], bytes, cudaMemcpyDeviceToHost, c->copy_stream));
    NSC_CUDA(c, cudaEventRecord(c->ev_copied, c->copy_stream));
    return NSC_OK;
}

// Double-buffered read-in: the host buffers are copied into a staging set on a private stream (overlapping whatever
// the context's stream is doing with the current state), then the context's stream takes the staging set over as the
// new state (device to device) and derives D1 p.
int nsc_set_state_host_async(nsc_ctx* c, const void* ur, const void* uth, const void* uz, const void* T, const void* p) {
    if (!c) return NSC_EINVAL;
    const void* src[5] = {ur, uth, uz, T, p};
    for (int i = 0; i < 3 + (c->heated ? 1 : 0); ++i)
        if (!src[i]) return fail(c, NSC_EINVAL, "nsc_set_state_host_async: required field pointer is NULL");
    int rc = transfer_setup(c, c->stage_in, &c->up_stream, &c->ev_uploaded, &c->ev_staged_used, false, &c->up_ready);
    if (rc) return rc;
    const size_t bytes = c->F * sizeof(cd);
    NSC_CUDA(c, cudaStreamWaitEvent(c->up_stream, c->ev_staged_used, 0));     // the previous staging set has been taken over
    for (int i = 0; i < 5; ++i) {
        if (i == 3 && !c->heated) continue;
        if (src[i])
            NSC_CUDA(c, cudaMemcpyAsync(c->stage_in[i], src[i], bytes, cudaMemcpyHostToDevice, c->up_stream));
        else
            NSC_CUDA(c, cudaMemsetAsync(c->stage_in[i], 0, bytes, c->up_stream));  // p = 0
    }
    NSC_CUDA(c, cudaEventRecord(c->ev_uploaded, c->up_stream));
    NSC_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_uploaded, 0));
    for (int i = 0; i < 5; ++i)
        if (i != 3 || c->heated)
            NSC_CUDA(c, cudaMemcpyAsync(c->state[i], c->stage_in[i], bytes, cudaMemcpyDeviceToDevice, c->stream));
    NSC_CUDA(c, cudaEventRecord(c->ev_staged_used, c->stream));
    return after_set_state(c);
}

int nsc_host_copies_wait(nsc_ctx* c) {
    if (!c) return NSC_EINVAL;
    if (c->up_ready) NSC_CUDA(c, cudaStreamSynchronize(c->up_stream));
    if (c->down_ready) NSC_CUDA(c, cudaStreamSynchronize(c->copy_stream));
    return NSC_OK;
}

int nsc_nonlinear(nsc_ctx* c, void* Nr, void* Nth, void* Nz, void* NT) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_nonlinear before nsc_set_state");
    if (!Nr || !Nth || !Nz || (c->heated && !NT)) return fail(c, NSC_EINVAL, "nsc_nonlinear: NULL output pointer");
    cd* out[MAXF] = {(cd*)Nr, (cd*)Nth, (cd*)Nz, (cd*)NT};
    return launch_nonlinear(c, c->state, out);
}

int nsc_substep(nsc_ctx* c, const void* Er, const void* Eth, const void* Ez, const void* ET, double dt) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_substep before nsc_set_state");
    if (!(dt > 0.0)) return fail(c, NSC_EINVAL, "nsc_substep: dt must be > 0");
    if (!Er || !Eth || !Ez || (c->heated && !ET)) return fail(c, NSC_EINVAL, "nsc_substep: NULL explicit-term pointer");
    cd* E[MAXF] = {(cd*)Er, (cd*)Eth, (cd*)Ez, (cd*)ET};
    return launch_substep(c, E, 1.0, nullptr, 0.0, dt, c->state, c->state[4]);
}

// the kernel sequence of one step (R10)
static int step_body(nsc_ctx* c, double dt) {
    int rc;
    // N0 = N(u^n);  u^1 = substep(N0) -> W (its pressure is discarded)
    if ((rc = launch_nonlinear(c, c->state, c->N0))) return rc;
    if ((rc = launch_substep(c, c->N0, 1.0, nullptr, 0.0, dt, c->W, nullptr))) return rc;
    // N1 = N(u^1);  u^{n+1} = substep(c N1 + (1 - c) N0) from (u^n, p^n), in place
    if ((rc = launch_nonlinear(c, c->W, c->N1))) return rc;
    return launch_substep(c, c->N1, c->p.c, c->N0, 1.0 - c->p.c, dt, c->state, c->state[4]);
}

// ---- NEXT-2: the pieces of a step for a slab-decomposed run
int nsc_set_window(nsc_ctx* c, int j0, int nj, long long e0, long long ne) {
    if (!c) return NSC_EINVAL;
    const long long plane = (long long)c->M1 * c->NK;
    if (nj == 0 && ne == 0 && j0 == 0 && e0 == 0) {
        nj = c->N_r;
        ne = plane;
    }
    if (j0 < 0 || nj < 1 || j0 + nj > c->N_r || e0 < 0 || ne < 1 || e0 + ne > plane)
        return fail(c, NSC_EINVAL, "nsc_set_window: levels [j0, j0 + nj) within [0, N_r) and modes [e0, e0 + ne) within [0, (M+1)(2K+1)), both non-empty");
    c->wj0 = j0;
    c->wj1 = j0 + nj;
    c->we0 = e0;
    c->we1 = e0 + ne;
    c->ptr_gen += 1;                                     // a captured step graph covers the old window
    return NSC_OK;
}

int nsc_step_phase(nsc_ctx* c, int phase, double dt) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_step_phase before nsc_set_state");
    if (phase < 0 || phase > 3 || !(dt > 0.0)) return fail(c, NSC_EINVAL, "nsc_step_phase: phase 0..3, dt > 0");
    switch (phase) {
        case 0: return launch_nonlinear(c, c->state, c->N0);
        case 1: return launch_substep(c, c->N0, 1.0, nullptr, 0.0, dt, c->W, nullptr);
        case 2: return launch_nonlinear(c, c->W, c->N1);
        default: return launch_substep(c, c->N1, c->p.c, c->N0, 1.0 - c->p.c, dt, c->state, c->state[4]);
    }
}

int nsc_field_pointers(nsc_ctx* c, int which, void** h_ptrs) {
    if (!c || !h_ptrs || which < 0 || which > 3) return NSC_EINVAL;
    cd* const* src = which == 0 ? c->state : which == 1 ? c->W : which == 2 ? c->N0 : c->N1;
    for (int i = 0; i < MAXF; ++i) h_ptrs[i] = i < c->nf ? (void*)src[i] : nullptr;
    return NSC_OK;
}

static void drop_graph(nsc_ctx* c) {
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    c->graph_exec = nullptr;
}

int nsc_step(nsc_ctx* c, double dt) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_step before nsc_set_state");
    if (!(dt > 0.0)) return fail(c, NSC_EINVAL, "nsc_step: dt must be > 0");
    // The ~44 launches of a step are captured once per (dt, stream, buffer generation) into a CUDA graph and
    // replayed: small configurations are launch-bound.  With per-kernel profiling on (event brackets), or if
    // capture is not possible, the kernels are launched one by one.
    if (c->use_graph && !c->profiling) {
        // set-up kernels stay outside the graph; a no-op unless dt changed since the factors were built (another
        // call, e.g. nsc_substep with its own dt, may have rebuilt them in place since the graph was captured)
        int rc = ensure_factors(c, dt);
        if (rc) return rc;
        const bool stale = !c->graph_exec || c->graph_dt != dt || c->graph_stream != c->stream || c->graph_gen != c->ptr_gen;
        if (stale) {
            drop_graph(c);
            cudaGraph_t g = nullptr;
            const long long l0 = c->launches;
            if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                rc = step_body(c, dt);
                const cudaError_t e = cudaStreamEndCapture(c->stream, &g);
                if (rc == NSC_OK && e == cudaSuccess && g && cudaGraphInstantiate(&c->graph_exec, g, 0) == cudaSuccess) {
                    c->graph_dt = dt;
                    c->graph_stream = c->stream;
                    c->graph_gen = c->ptr_gen;
                    c->graph_launches = c->launches - l0;
                } else {
                    c->graph_exec = nullptr;
                    c->use_graph = false;                // capture works on this stream but the graph does not: plain launches for good
                }
                if (g) cudaGraphDestroy(g);
                cudaGetLastError();
            } else {
                cudaGetLastError();                      // no capture on this stream (legacy default stream): plain launches for this call only
            }
            c->launches = l0;
        }
        if (c->graph_exec) {
            NSC_CUDA(c, cudaGraphLaunch(c->graph_exec, c->stream));
            c->launches += c->graph_launches;
            c->graph_replays += 1;
            return NSC_OK;
        }
    }
    return step_body(c, dt);
}

// ---- NEXT-1: iterated corrector (R16) and step-size control (R17)
static int iter_alloc(nsc_ctx* c) {
    if (c->it_acc) return NSC_OK;                        // first use: ping-pong iterates + pressure of a pass
    int rc;
    for (int i = 0; i < c->nf; ++i) {
        if ((rc = dev_alloc(c, &c->itA[i], c->F, false))) return rc;
        if ((rc = dev_alloc(c, &c->itB[i], c->F, false))) return rc;
    }
    if ((rc = dev_alloc(c, &c->itP, c->F, false))) return rc;
    if ((rc = dev_alloc(c, &c->itDP, c->F, false))) return rc;
    cd* acc = nullptr;
    if ((rc = dev_alloc(c, &acc, 1, true))) return rc;   // one complex = two doubles
    c->it_acc = reinterpret_cast<double*>(acc);
    return NSC_OK;
}

// Predictor and up to max_corr corrector passes from the state, which is left untouched: the newest iterate ends
// in itA, the pressure of its pass in itP / itDP.  have_N0: N0 = N(u^n) is already in c->N0.
static int iterated_core(nsc_ctx* c, double dt, double tol, int max_corr, bool have_N0, int* k_out, double* e_out) {
    int rc;
    // N0 = N(u^n);  u^(1) = substep(N0) -> itA (its pressure is discarded)
    if (!have_N0 && (rc = launch_nonlinear(c, c->state, c->N0))) return rc;
    if ((rc = launch_substep(c, c->N0, 1.0, nullptr, 0.0, dt, c->itA, nullptr))) return rc;
    int k = 0;
    double e = 0.0;
    while (k < max_corr) {
        // u^(k+1) = substep(c N(u^(k)) + (1 - c) N0) from (u^n, p^n) -> itB, pressure of the pass -> itP, itDP
        if ((rc = launch_nonlinear(c, c->itA, c->N1))) return rc;
        if ((rc = launch_substep(c, c->N1, c->p.c, c->N0, 1.0 - c->p.c, dt, c->itB, c->itP, c->itDP))) return rc;
        if ((rc = launch_diff_norm(c, c->itA, c->itB, c->it_acc))) return rc;
        double h[2] = {0.0, 0.0};
        NSC_CUDA(c, cudaMemcpyAsync(h, c->it_acc, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
        NSC_CUDA(c, cudaStreamSynchronize(c->stream));
        ++k;
        e = h[1] > 0.0 ? sqrt(h[0] / h[1]) : 0.0;
        for (int i = 0; i < c->nf; ++i) std::swap(c->itA[i], c->itB[i]);       // itA = newest iterate
        if (e <= tol) break;
    }
    *k_out = k;
    *e_out = e;
    return NSC_OK;
}

// accept: the newest iterate and the pressure of its pass become the state (pointer swaps, no copies)
static void iterated_commit(nsc_ctx* c) {
    for (int i = 0; i < c->nf; ++i) std::swap(c->state[i], c->itA[i]);
    std::swap(c->state[4], c->itP);
    std::swap(c->DP, c->itDP);
    c->ptr_gen += 1;                                     // a captured step graph holds the old pointers
}

int nsc_step_iterated(nsc_ctx* c, double dt, double tol, int max_corr, int* n_corr, double* err) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_step_iterated before nsc_set_state");
    if (!(dt > 0.0)) return fail(c, NSC_EINVAL, "nsc_step_iterated: dt must be > 0");
    if (!(tol >= 0.0) || max_corr < 1) return fail(c, NSC_EINVAL, "nsc_step_iterated: tol must be >= 0 and max_corr >= 1");
    int rc, k = 0;
    double e = 0.0;
    if ((rc = iter_alloc(c))) return rc;
    if ((rc = iterated_core(c, dt, tol, max_corr, false, &k, &e))) return rc;
    iterated_commit(c);
    if (n_corr) *n_corr = k;
    if (err) *err = e;
    return NSC_OK;
}

// step sizes live on the geometric grid (8 + i) / 16 * 2^e, i = 0..7 (R17): the per-mode factors are re-used
static double dt_grid_floor(double x) {
    int e = 0;
    const double m = frexp(x, &e);                       // x = m 2^e, 0.5 <= m < 1
    return ldexp(floor(m * 16.0) / 16.0, e);
}
static double dt_grid_next(double x) {
    int e = 0;
    const double m = frexp(x, &e);
    return ldexp((floor(m * 16.0) + 1.0) / 16.0, e);
}

// N0 = N(u^n) with the per-level maxima of |u| gathered by the theta kernel; *rate = the CFL rate lambda (R17)
static int nonlinear_with_cfl(nsc_ctx* c, double* rate) {
    int rc;
    if (!c->cfl_max) {
        cd* p = nullptr;
        if ((rc = dev_alloc(c, &p, ((size_t)3 * c->N_r + 1) / 2, true))) return rc;     // 3 N_r 64-bit words
        c->cfl_max = reinterpret_cast<unsigned long long*>(p);
    }
    NSC_CUDA(c, cudaMemsetAsync(c->cfl_max, 0, sizeof(unsigned long long) * 3 * c->N_r, c->stream));
    c->want_cfl = true;
    rc = launch_nonlinear(c, c->state, c->N0);
    c->want_cfl = false;
    if (rc) return rc;
    std::vector<double> mx((size_t)3 * c->N_r);          // the bit patterns are those of non-negative doubles
    NSC_CUDA(c, cudaMemcpyAsync(mx.data(), c->cfl_max, sizeof(double) * mx.size(), cudaMemcpyDeviceToHost, c->stream));
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    const int N = c->N_r;
    const double dth = 2.0 * M_PI / ((double)c->p.k_theta0 * (double)c->Nt);
    const double dz = 2.0 * M_PI / (c->p.alpha * (double)c->Nz);
    double lr = 0.0, lt = 0.0, lz = 0.0;
    for (int j = 0; j < N; ++j) {
        const double dl = c->r[j > 0 ? j : 1] - c->r[j > 0 ? j - 1 : 0];
        const double dr = c->r[j < N - 1 ? j + 1 : N - 1] - c->r[j < N - 1 ? j : N - 2];
        lr = fmax(lr, mx[3 * j] / fmin(dl, dr));
        lt = fmax(lt, mx[3 * j + 1] / (c->r[j] * dth));
        lz = fmax(lz, mx[3 * j + 2] / dz);
    }
    *rate = fmax(lr, fmax(lt, lz));
    return NSC_OK;
}

int nsc_cfl_rate(nsc_ctx* c, double* h_rate) {
    if (!c || !h_rate) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_cfl_rate before nsc_set_state");
    return nonlinear_with_cfl(c, h_rate);
}

int nsc_advance(nsc_ctx* c, double t_end, int max_steps, double dt0, double tol, double cfl, int max_corr,
                nsc_advance_info* h_info, double* h_log) {
    if (!c) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_advance before nsc_set_state");
    if (!(t_end > 0.0) || max_steps < 1 || !(dt0 > 0.0) || !(tol >= 0.0) || !(cfl > 0.0) || max_corr < 1)
        return fail(c, NSC_EINVAL, "nsc_advance: t_end, dt0, cfl must be > 0, tol >= 0, max_steps and max_corr >= 1");
    int rc;
    if ((rc = iter_alloc(c))) return rc;
    nsc_advance_info info;
    memset(&info, 0, sizeof(info));
    double t = 0.0, dt_cur = dt_grid_floor(dt0), lam = 0.0;
    bool have_N0 = false;
    int n = 0;
    while (t < t_end && n < max_steps) {
        if (!have_N0) {
            if ((rc = nonlinear_with_cfl(c, &lam))) return rc;
            have_N0 = true;
        }
        double dt = dt_cur;
        if (lam > 0.0) dt = fmin(dt, dt_grid_floor(cfl / lam));
        const bool last = t_end - t <= dt;
        if (last) dt = t_end - t;
        int k = 0;
        double e = 0.0;
        if ((rc = iterated_core(c, dt, tol, max_corr, true, &k, &e))) return rc;
        const bool ok = e <= tol;
        if (h_log) {
            h_log[4 * n] = dt;
            h_log[4 * n + 1] = (double)k;
            h_log[4 * n + 2] = e;
            h_log[4 * n + 3] = ok ? 1.0 : 0.0;
        }
        ++n;
        info.passes += k;
        info.err_last = e;
        info.cfl_rate_last = lam;
        if (ok) {
            iterated_commit(c);
            have_N0 = false;                             // N0 belongs to the old state
            t = last ? t_end : t + dt;
            info.accepted += 1;
            info.dt_last = dt;
            if (info.dt_min == 0.0 || dt < info.dt_min) info.dt_min = dt;
            if (dt > info.dt_max) info.dt_max = dt;
            if (k <= 2 && e <= 0.5 * tol && dt == dt_cur) dt_cur = dt_grid_next(dt_cur);
        } else {
            info.rejected += 1;
            dt_cur = dt_grid_floor(dt / 2.0);            // the state and N0 are untouched: try again
        }
    }
    info.t = t;
    info.dt_next = dt_cur;
    if (h_info) *h_info = info;
    return NSC_OK;
}

// ---- NEXT-3: wave speed
int nsc_mode_coefficient(nsc_ctx* c, int field, int j, int m, int k, double* h_re_im) {
    if (!c || !h_re_im) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_mode_coefficient before nsc_set_state");
    if (field < 0 || field > 4 || (field == 3 && !c->heated) || j < 0 || j >= c->N_r || m < 0 || m > c->M || k < -c->K || k > c->K)
        return fail(c, NSC_EINVAL, "nsc_mode_coefficient: field 0..4 (3 only with temperature), 0 <= j < N_r, 0 <= m <= M, |k| <= K");
    const size_t off = ((size_t)j * c->M1 + m) * c->NK + (size_t)(k + c->K);
    NSC_CUDA(c, cudaMemcpyAsync(h_re_im, c->state[field] + off, sizeof(cd), cudaMemcpyDeviceToHost, c->stream));
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    return NSC_OK;
}

int nsc_wave_speed(nsc_ctx* c, int field, int j, int m, int k, double dt, int n_steps, double* h_speed) {
    if (!c || !h_speed) return NSC_EINVAL;
    if (m < 1 || n_steps < 1) return fail(c, NSC_EINVAL, "nsc_wave_speed: m must be >= 1 and n_steps >= 1");
    double f0[2], f1[2];
    int rc = nsc_mode_coefficient(c, field, j, m, k, f0);
    if (rc) return rc;
    double dphi = 0.0;
    for (int i = 0; i < n_steps; ++i) {
        if ((rc = nsc_step(c, dt))) return rc;
        if ((rc = nsc_mode_coefficient(c, field, j, m, k, f1))) return rc;
        // arg(f1 conj(f0)), in (-pi, pi]
        dphi += atan2(f1[1] * f0[0] - f1[0] * f0[1], f1[0] * f0[0] + f1[1] * f0[1]);
        f0[0] = f1[0];
        f0[1] = f1[1];
    }
    *h_speed = -dphi / ((double)n_steps * dt) / ((double)m * (double)c->p.k_theta0);
    return NSC_OK;
}

static int diag_scratch(nsc_ctx* c) {
    if (c->diag) return NSC_OK;
    cd* p = nullptr;
    int rc = dev_alloc(c, &p, 2, true);                  // two complex = four doubles
    if (!rc) c->diag = reinterpret_cast<double*>(p);
    return rc;
}

int nsc_nusselt(nsc_ctx* c, double* h_out) {
    if (!c || !h_out) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_nusselt before nsc_set_state");
    int rc = diag_scratch(c);
    if (rc) return rc;
    if ((rc = launch_nusselt(c, c->diag))) return rc;
    NSC_CUDA(c, cudaMemcpyAsync(h_out, c->diag, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    return NSC_OK;
}

int nsc_probe(nsc_ctx* c, int field, int j, double theta, double z, double* h_value) {
    if (!c || !h_value) return NSC_EINVAL;
    if (!c->have_state) return fail(c, NSC_ESTATE, "nsc_probe before nsc_set_state");
    if (field < 0 || field > 4 || (field == 3 && !c->heated) || j < 0 || j >= c->N_r)
        return fail(c, NSC_EINVAL, "nsc_probe: field must be 0..4 (3 only with temperature) and 0 <= j < N_r");
    int rc = diag_scratch(c);
    if (rc) return rc;
    if ((rc = launch_probe(c, c->state[field], j, theta, z, c->diag))) return rc;
    NSC_CUDA(c, cudaMemcpyAsync(h_value, c->diag, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    return NSC_OK;
}

int nsc_set_profiling(nsc_ctx* c, int on) {
    if (!c) return NSC_EINVAL;
    c->profiling = on != 0;
    return NSC_OK;
}

int nsc_profile_read(nsc_ctx* c, double* h_ms, long long* h_count) {
    if (!c || !h_ms || !h_count) return NSC_EINVAL;
    NSC_CUDA(c, cudaStreamSynchronize(c->stream));
    for (auto& r : c->prof) {
        float ms = 0.f;
        NSC_CUDA(c, cudaEventElapsedTime(&ms, r.a, r.b));
        h_ms[r.id] += ms;
        h_count[r.id] += 1;
        c->ev_pool.push_back(r.a);
        c->ev_pool.push_back(r.b);
    }
    c->prof.clear();
    return NSC_OK;
}

const char* nsc_kernel_name(int id) { return (id >= 0 && id < NSC_NKERN) ? kKernelNames[id] : ""; }

const char* nsc_last_error(const nsc_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

long long nsc_device_bytes(const nsc_ctx* c) { return c ? c->dev_bytes : 0; }

long long nsc_launch_count(const nsc_ctx* c) { return c ? c->launches : 0; }

long long nsc_graph_replays(const nsc_ctx* c) { return c ? c->graph_replays : 0; }

}  // extern "C"
