/* nsc.h -- C ABI of libnsc.so: one predictor-corrector time step of the nsCouette method
 * (arxiv/paper_1908_00587) for incompressible, optionally heated Taylor-Couette flow,
 * computed entirely by hand-written sm_100a CUDA kernels on one B200.
 *
 * What the library computes (citations: PAPER.md:<line>; BJ = BASELINE.json north_star;
 * R# = reading listed in DESIGN.md):
 *   - Fourier-Galerkin in theta and z, 9-point finite differences on a run-time selectable
 *     radial grid, axially periodic, cylindrical primitive
 *     variables u_r, u_theta, u_z, p, (T);
 *   - the pseudospectral nonlinear term N = -(u.grad)u with the curvature terms, Boussinesq
 *     buoyancy and -(u.grad)T (BJ (a)), 3/2-rule padded (R4, R5);
 *   - the implicit predictor-corrector sub-steps: per Fourier mode banded
 *     Helmholtz solves in u_+- = u_r +- i u_theta, u_z, T and a pressure-Poisson projection
 *     (BJ (b); "linear terms ... independently per Fourier mode").
 *
 * Conventions common to every call
 *   Spectral field  complex128 (re, im interleaved), shape [N_r][M_theta+1][2 K_z+1], the axial
 *                   index fastest; entry (j, m, kk) is radial node j (j = 0 inner wall), azimuthal
 *                   mode m (wavenumber n = m k_theta0), axial mode k = kk - K_z (kappa = k alpha).
 *   Units           gap d = r_o - r_i = 1, time d^2/nu, velocity nu/d, so Re_i, Re_o
 *                   are the wall speeds; T = +1/2 at r_i, -1/2 at r_o (R1).
 *   Pointers        "d_" = DEVICE pointer, "h_" = HOST pointer.  The caller owns every buffer it
 *                   passes; the library owns the context, its copy of the state and all work space.
 *   Streams         all device work is enqueued on the stream given to nsc_set_stream (default:
 *                   the legacy default stream) and is asynchronous; only nsc_create,
 *                   nsc_destroy and the *_host calls synchronise.
 *   Errors          0 on success, a negative NSC_E* code otherwise; nsc_last_error() gives text.
 *                   Nothing throws across the ABI.  There is no CPU fallback: without a CUDA
 *                   device nsc_create fails with NSC_ECUDA.
 *   Temperature     enabled iff Ra != 0 (R13); then the T pointers are required, else ignored.
 */
#ifndef NSC_H
#define NSC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nsc_ctx nsc_ctx;

enum {
    NSC_OK = 0,
    NSC_EINVAL = -1,  /* bad argument (sizes, ranges, NULL where a pointer is required)      */
    NSC_ENOMEM = -2,  /* host or device allocation failed                                       */
    NSC_ECUDA = -3,   /* a CUDA runtime call or kernel launch failed                            */
    NSC_ESTATE = -4   /* call out of order (nsc_step / nsc_nonlinear before nsc_set_state)      */
};

/* Extended creation parameters (nsc_create fills the defaults marked below). */
typedef struct nsc_params {
    int N_r;          /* radial nodes, >= 9 (9-point stencil)                      */
    int M_theta;      /* azimuthal modes m = 0..M_theta, 1 <= M_theta <= 512                       */
    int K_z;          /* axial modes k = -K_z..K_z,     1 <= K_z <= 512                            */
    double eta;       /* radius ratio r_i / r_o, 0 < eta < 1                                      */
    double alpha;     /* axial base wavenumber (domain length 2 pi / alpha), > 0                  */
    int k_theta0;     /* azimuthal base wavenumber, >= 1                                          */
    double Re_i, Re_o;/* inner / outer wall speed (units nu/d)                                    */
    double Ra, Pr;    /* Rayleigh, Prandtl number; Ra == 0 switches temperature off; Pr > 0       */
    int radial_grid;  /* 0 uniform, 1 Chebyshev-Gauss-Lobatto clustering (R2)                     */
    int n_theta_phys; /* physical grid points in theta; 0 => the shortest supported length >= 3 M_theta
                       * (3/2 rule, R4; = 3 M_theta when M_theta is a power of two >= 4)           */
    int n_z_phys;     /* physical grid points in z;     0 => likewise for K_z.  Supported transform
                       * lengths: 3 * 2^p in {12, 24, ..., 1536}; a given length must be >= the 3/2 rule */
    double c;         /* implicitness of the linear terms; 0 => 0.5 (R10)                         */
    int device;       /* CUDA device ordinal; -1 => current device                                */
    int radial_chunk; /* radial nodes per pass of the transform pipeline; 0 => automatic (all N_r
                       * at once when the work arrays fit an eighth of the device memory)         */
    int linear_slices;/* mode slices of the implicit sub-step, each a chain of four sweep kernels on a
                       * stream of its own; 0 => 2, at most 8                    */
    int no_graph;     /* nonzero: nsc_step never captures / replays a CUDA graph (plain launches)     */
} nsc_params;

/* BJ: nsc_create(N_r, M_theta, K_z, eta, alpha, k_theta0, Re_i, Re_o, Ra, Pr, radial-grid type).
 * Builds the plan on the host in extended precision (radial grid, 9-point weights, operator
 * band tables, twiddle tables), uploads it and allocates state and work space.  *out is set
 * only on success.  Synchronises the device. */
int nsc_create(nsc_ctx** out, int N_r, int M_theta, int K_z, double eta, double alpha, int k_theta0,
               double Re_i, double Re_o, double Ra, double Pr, int radial_grid);
int nsc_create_ex(nsc_ctx** out, const nsc_params* p);

/* Frees everything the context owns.  Synchronises.  NULL is a no-op. */
int nsc_destroy(nsc_ctx* ctx);

/* cudaStream_t (as void*) on which all later work of this context is enqueued. */
int nsc_set_stream(nsc_ctx* ctx, void* cuda_stream);

/* Radial nodes r_j, j = 0..N_r-1, written to h_r (host, N_r doubles). */
int nsc_get_grid(const nsc_ctx* ctx, double* h_r);

/* Copies a state into the context (device-to-device on the stream) and derives D1 p of it (one
 * kernel launch; the linear stage keeps the radial pressure gradient as an array, DESIGN.md
 * section 6).  d_T required iff Ra != 0; d_p may be NULL (p = 0).  Each pointer: one spectral
 * field as described above. */
int nsc_set_state(nsc_ctx* ctx, const void* d_ur, const void* d_uth, const void* d_uz,
                  const void* d_T, const void* d_p);
/* Copies the current state out; NULL pointers are skipped. */
int nsc_get_state(nsc_ctx* ctx, void* d_ur, void* d_uth, void* d_uz, void* d_T, void* d_p);
/* The same with HOST buffers (pinned or pageable); the host-to-device / device-to-host copies
 * run on the context's stream and the call returns after they completed. */
int nsc_set_state_host(nsc_ctx* ctx, const void* h_ur, const void* h_uth, const void* h_uz,
                       const void* h_T, const void* h_p);
int nsc_get_state_host(nsc_ctx* ctx, void* h_ur, void* h_uth, void* h_uz, void* h_T, void* h_p);

/* Double-buffered host transfers for loops that feed a state in and take the result out every step (pinned HOST
 * buffers; with pageable memory the copies are not asynchronous).  Both calls return at once.
 *   nsc_set_state_host_async  the host buffers are copied into a staging set on a private stream -- overlapping the work
 *                             the context's stream still does on the current state -- and the context's stream then takes
 *                             the staging set over as the new state (device to device) and derives D1 p; calls enqueued
 *                             afterwards see the new state.  The host buffers may be reused after nsc_host_copies_wait.
 *   nsc_get_state_host_async  the state is snapshot on the context's stream (device to device) and the snapshot is copied
 *                             to the host buffers on a second private stream, so that the next read-in and step overlap
 *                             with the transfer (PCIe carries both directions at the same time).  The host buffers are
 *                             complete after nsc_host_copies_wait.  NULL pointers are skipped; h_T on a context without
 *                             temperature is refused (NSC_EINVAL) instead of being left unwritten without notice.
 * A second call of either kind waits on the device for the first one's staging set / snapshot to be free.  The first
 * calls allocate one staging set and one snapshot of the state and create a private stream and two events each; if that
 * set-up fails halfway the call returns the error, keeps what exists and the next call creates only what is missing. */
int nsc_set_state_host_async(nsc_ctx* ctx, const void* h_ur, const void* h_uth, const void* h_uz,
                             const void* h_T, const void* h_p);
int nsc_get_state_host_async(nsc_ctx* ctx, void* h_ur, void* h_uth, void* h_uz, void* h_T, void* h_p);
int nsc_host_copies_wait(nsc_ctx* ctx);

/* Steps N1-N6 of DESIGN.md (BJ (a)): N(current state), buoyancy included, written to the
 * caller's device buffers (d_NT required iff Ra != 0); the state is unchanged. */
int nsc_nonlinear(nsc_ctx* ctx, void* d_Nr, void* d_Nth, void* d_Nz, void* d_NT);

/* Steps L1-L5 (BJ (b)): one implicit sub-step of size dt from the current state with the explicit
 * term E given by the caller (device buffers, same layout; d_ET required iff Ra != 0):
 *   Helmholtz solves for u_+-, u_z, (T) -> divergence -> pressure Poisson -> correction;
 *   the state (u, T, p) is replaced by the result.  Exposed so that the linear stage can be
 *   checked on its own; nsc_step composes it with nsc_nonlinear internally. */
int nsc_substep(nsc_ctx* ctx, const void* d_Er, const void* d_Eth, const void* d_Ez,
                const void* d_ET, double dt);

/* One predictor-corrector step of size dt > 0 (R10: c = 1/2, one corrector pass):
 *   N0 = N(u^n); u^1 = substep(N0); N1 = N(u^1); u^{n+1} = substep(c N1 + (1-c) N0), both
 *   sub-steps starting from (u^n, T^n, p^n).  The first call with a new dt factors the
 *   per-mode banded matrices (kept until dt changes). */
int nsc_step(nsc_ctx* ctx, double dt);

/* The same step with the corrector iterated to convergence (PAPER.md:46
 * "dynamic control" of the step size; stopping rule = DESIGN.md reading R16):
 *   u^(1) = substep(N0);  u^(k+1) = substep(c N(u^(k)) + (1-c) N0), k = 1, 2, ..., every pass from
 *   (u^n, T^n, p^n); stop after pass k when ||u^(k+1) - u^(k)||_2 / ||u^(k+1)||_2 <= tol (all
 *   fields u_r, u_theta, u_z, (T) concatenated) or k = max_corr >= 1.
 * The newest iterate and the pressure of its pass become the state.  *n_corr (may be NULL) receives
 * k, *err (may be NULL) the last norm: a caller steers dt with them.  max_corr = 1 is nsc_step.
 * Synchronises the stream once per pass (the norm is read back); the first call allocates
 * (2 n_f + 2) more field-sized buffers. */
int nsc_step_iterated(nsc_ctx* ctx, double dt, double tol, int max_corr, int* n_corr, double* err);

/* CFL rate lambda of the current state (reading R17): the largest over the physical
 * grid of |u_r| / dr_j, |u_theta| / (r_j dtheta), |u_z| / dz with dr_j = the smaller radial spacing next to node j,
 * dtheta = 2 pi / (k_theta0 N_theta), dz = 2 pi / (alpha N_z); a step of size dt has CFL number lambda dt.  Runs
 * one nonlinear evaluation (the theta kernel gathers the maxima per radial level).  *h_rate: HOST double.
 * Synchronises the stream. */
int nsc_cfl_rate(nsc_ctx* ctx, double* h_rate);

/* Time integration with dynamic step-size control ("variable time-step size with dynamic control"; the
 * paper's rule is in its ref. [6], not available: DESIGN.md reading R17).  From t = 0, until t = t_end or max_steps
 * attempts:   dt = min(dt_cur, floor(cfl / lambda(u^n)), t_end - t);  the step of nsc_step_iterated(dt, tol, max_corr)
 *   err <= tol : accepted, t += dt;  dt_cur <- next grid value if it took <= 2 passes, err <= tol / 2 and dt == dt_cur
 *   err >  tol : rejected, the state is untouched, dt_cur <- floor(dt / 2), tried again (N(u^n) is not recomputed)
 * with dt_cur starting at floor(dt0); floor / next refer to the grid (8 + i) / 16 * 2^e, i = 0..7, so that the factored
 * per-mode matrices are re-used.  h_info (HOST, may be NULL) receives the summary; h_log (HOST, may be NULL, 4 max_steps
 * doubles) one record (dt, passes, err, accepted 1/0) per attempt.  Synchronises the stream once per corrector pass
 * and once per step (the norm and the maxima are read back). */
typedef struct nsc_advance_info {
    double t;             /* time reached (== t_end unless max_steps ran out)                       */
    double dt_next;       /* the controller's current step size (pass it as dt0 to continue)        */
    double dt_last, dt_min, dt_max;   /* of the accepted steps                                      */
    double err_last;      /* corrector norm of the last attempt                                     */
    double cfl_rate_last; /* lambda of the last state a step started from                           */
    int accepted, rejected, passes;   /* steps accepted / rejected, corrector passes in total       */
} nsc_advance_info;
int nsc_advance(nsc_ctx* ctx, double t_end, int max_steps, double dt0, double tol, double cfl, int max_corr,
                nsc_advance_info* h_info, double* h_log);

/* One Fourier coefficient f^(r_j; m, k) of the current state (field: 0 u_r, 1 u_theta, 2 u_z, 3 T, 4 p), as
 * (re, im) in h_re_im (HOST, 2 doubles).  Synchronises the stream. */
int nsc_mode_coefficient(nsc_ctx* ctx, int field, int j, int m, int k, double* h_re_im);

/* Angular phase speed of that coefficient over n_steps calls of nsc_step(dt) (the
 * CI validation compares "the wave speed of a simulated wavy vortex flow" with an experiment): for
 * f ~ e^{i (n theta - omega t)}, n = m k_theta0 >= 1,  *h_speed = omega / n with
 * omega = - sum_i arg(f_{i+1} conj f_i) / (n_steps dt)  (phase increments per step, each in (-pi, pi]).
 * The state advances by n_steps steps.  Synchronises the stream after every step. */
int nsc_wave_speed(nsc_ctx* ctx, int field, int j, int m, int k, double dt, int n_steps, double* h_speed);

/* The pieces of a step for a slab-decomposed run over several GPUs (modes are
 * independent in the linear terms, radial levels in the nonlinear terms).  Every rank holds a
 * context of the full size and computes only its window; the Python module paper_1908_00587_b200.slabs moves the slabs
 * between the ranks (torch.distributed) directly inside the library's arrays.
 *   nsc_set_window     nsc_nonlinear / phases 0, 2 evaluate the radial levels [j0, j0 + nj) only.  They read the fields at
 *                      the levels the nine-point stencils of the window reach, [s(j0), s(j0 + nj - 1) + 9) with
 *                      s(j) = clamp(j - 4, 0, N_r - 9): four levels beyond the window on either side, and the nine levels
 *                      next to a wall however short the window.  nsc_substep / phases 1, 3 treat the Fourier modes
 *                      [e0, e0 + ne) only (flat index m (2 K_z + 1) + k + K_z).  All four arguments 0: everything (default).
 *   nsc_step_phase     one quarter of nsc_step(dt) on the window: 0  N0 = N(u^n);  1  u^1 = substep(N0) -> predictor buffers;
 *                      2  N1 = N(u^1);  3  u^{n+1} = substep(c N1 + (1 - c) N0), in place.  Outside the window the target
 *                      arrays keep what they held.
 *   nsc_field_pointers DEVICE pointers of the n_f arrays of a buffer set written to h_ptrs (HOST array of 4 pointers, NULL
 *                      for T without temperature): which = 0 state (u_r, u_theta, u_z, T), 1 predictor, 2 N0, 3 N1; each
 *                      array has the layout of a spectral field.  They stay valid until nsc_destroy; nsc_step_iterated
 *                      and nsc_advance exchange the state pointers, so ask again after those. */
int nsc_set_window(nsc_ctx* ctx, int j0, int nj, long long e0, long long ne);
int nsc_step_phase(nsc_ctx* ctx, int phase, double dt);
int nsc_field_pointers(nsc_ctx* ctx, int which, void** h_ptrs);

/* Restart on another resolution ("At every restart, the spatial resolution can be
 * changed using an automated interpolation and mode padding functionality"; reading R18): the state
 * (u, T, p) of `src` is carried onto the radial grid and the mode set of `dst` and becomes the state of `dst`.
 *   radial : degree-8 Lagrange interpolation on the nine source nodes around the source node nearest to each target
 *            node (window start clamp(c - 4, 0, N_r,src - 9)); a target node that coincides with a source node takes
 *            its value exactly;
 *   modes  : coefficients of modes `src` does not hold are zero, modes `dst` does not hold are dropped.
 * `dst` and `src` must be two different contexts on the same device that agree in eta, alpha and k_theta0 (NSC_EINVAL
 * otherwise, checked before anything is touched; the call makes that device current while it runs and puts the caller's
 * current device back); N_r, M_theta, K_z, the grid family, Re_i, Re_o, Ra, Pr may differ.  A temperature field of `src` is dropped if `dst` has none;
 * `dst` with temperature needs `src` with temperature.  `src` is unchanged.  Synchronises both streams. */
int nsc_regrid(nsc_ctx* dst, nsc_ctx* src);

/* Wall diagnostics of the current state (Fig. 3a): transfer at a wall
 * normalised by that of the basic state at the same parameters, from the mean mode (0,0):
 *   h_out[0], h_out[1]  heat-flux Nusselt number at the inner / outer wall, d_r T r ln(eta)  (nan if Ra = 0)
 *   h_out[2], h_out[3]  torque Nusselt number, r^3 d_r(u_theta / r) / (-2 B), B of the Couette profile (nan if B = 0)
 * d_r is the 9-point row of the wall node.  h_out: HOST array of 4 doubles.  Synchronises the stream. */
int nsc_nusselt(nsc_ctx* ctx, double* h_out);

/* Value of a physical field at radial node j and the point (theta, z) (Fig. 3b: u_theta at a
 * fixed probe location): the Fourier series of the state evaluated there.  field: 0 u_r, 1 u_theta, 2 u_z, 3 T,
 * 4 p.  *h_value: HOST double.  Synchronises the stream. */
int nsc_probe(nsc_ctx* ctx, int field, int j, double theta, double z, double* h_value);

/* The probe of nsc_probe without a context and without a single allocation (Fig. 3b: the
 * probe signal is what a run is watched by).
 *
 * For whom: code that reads a probe from a state it holds itself but must not allocate device memory -- a
 * per-step monitoring hook next to a solver that has filled the device on purpose (the N_r = 512 configuration
 * holds 148 of 180 GB; a host framework's pool owns the rest, so a cudaMalloc fails or eats into it), code
 * between a solver's kernels where the device-wide stall of cudaMalloc / cudaFree would be paid every step, or
 * code in a region where its host program bans allocating runtime calls.  nsc_probe cannot serve them: it
 * needs a context, and nsc_create allocates.
 *
 * What it does: the Fourier series of one field at radial node j, evaluated at (theta, z), written to *d_value
 * -- the same sum as nsc_probe, added up in a fixed order (block partials, then the partials in index order),
 * so repeated calls on the same data give the same bits.
 *   d_field     DEVICE, caller's: one spectral field [N_r][M_theta+1][2 K_z+1] complex128 as described at the
 *               top; only level j is read.  k_theta0, alpha: the base wavenumbers the field belongs to.
 *   d_value     DEVICE, caller's: one double, overwritten.
 *   cuda_stream cudaStream_t as void* (NULL: legacy default stream).  The call only enqueues (one 256-byte
 *               memset, one kernel) and returns; *d_value is ready when that stream work has finished.
 *   The device that owns d_field, d_value and the stream must be the calling thread's current device.
 * Memory: nothing is allocated or freed, by this call or by anything it calls (no cudaMalloc / cudaFree, no
 * library routine that allocates).  The block partials and the blocks' arrival counter sit in a fixed array
 * inside the library image, NSC_PROBE_STATIC_SCRATCH_BYTES per GPU that has loaded the library, held until the
 * process exits.
 * Limit: M_theta <= 512 and K_z <= 512 (525 825 modes, what the array is laid out for; also nsc_create's
 * limit).  Anything larger is refused with NSC_EINVAL and a text saying so; nothing is launched.
 * First call on each device: looks up the array's device address (cudaGetSymbolAddress, with that device
 * current; the result is kept) and lets the driver load the kernel.  Make that first call during start-up,
 * before any stream capture is begun on that device.
 * Sharing: every call on a device uses the same array.  It keeps the previous call's contents -- the call
 * clears the counter itself, on `cuda_stream`, before the kernel -- and two calls whose device work overlaps
 * in time (two streams without an event between them, two host threads) race on it and both results are
 * wrong.  Keep the calls of one device on one stream or order them with events.
 * Errors: NSC_EINVAL (NULL pointer, sizes out of range, j outside [0, N_r), k_theta0 < 1, alpha <= 0,
 * non-finite alpha / theta / z) before any CUDA call; NSC_ECUDA if a CUDA call fails.  Text: nsc_last_error(NULL). */
#define NSC_PROBE_STATIC_SCRATCH_BYTES 4608
int nsc_probe_static(const void* d_field, int N_r, int M_theta, int K_z, int k_theta0, double alpha, int j,
                     double theta, double z, double* d_value, void* cuda_stream);

/* Text of the last error of this context ("" if none); valid until the next call on ctx.
 * With ctx == NULL: the text of the last failed nsc_create or nsc_probe_static on this thread. */
const char* nsc_last_error(const nsc_ctx* ctx);

/* Bytes of device memory the context holds (state + work + factors), for reports. */
long long nsc_device_bytes(const nsc_ctx* ctx);

/* Number of kernel launches this context has enqueued so far (for bench.py's gpu_launches). */
long long nsc_launch_count(const nsc_ctx* ctx);

/* Per-kernel device timing (for bench.py's roofline figures).  With profiling on, every kernel
 * launch is bracketed by CUDA events on the context's stream.  nsc_profile_read synchronises the
 * stream, ADDS the elapsed milliseconds and launch counts since the last read to h_ms[id] /
 * h_count[id] (host arrays of NSC_NKERN entries; the caller zeroes them) and forgets the events.
 * Kernel ids are the NSC_K_* constants; nsc_kernel_name gives the kernel's name. */
enum {
    NSC_K_ZINV = 0,      /* N1 + N2: z-derivative, radial derivative, padded inverse z-FFT          */
    NSC_K_THETA = 1,     /* N1 + N3 + N4 + N5: fused theta transforms and physical-space products   */
    NSC_K_ZFWD = 2,      /* N6: forward z-FFT, truncation, scaling, buoyancy                         */
    NSC_K_RHS = 3,       /* L1 + L2 (k_rhs_fwd): right-hand sides + forward substitution, marching up   */
    NSC_K_HELMHOLTZ = 4, /* L2 + L3 (k_bwd_div): back substitution, recombination, divergence, down     */
    NSC_K_RECOMBINE = 5, /* k_diff_norm: convergence norm of the iterated corrector (nsc_step_iterated)  */
    NSC_K_DIV = 6,       /* k_nusselt / k_probe: diagnostics (nsc_nusselt, nsc_probe)                    */
    NSC_K_POISSON = 7,   /* L4 (k_poisson_fwd): forward substitution of the pressure system, up          */
    NSC_K_CORRECT = 8,   /* L4 + L5 (k_poisson_bwd_correct): back substitution + correction, down        */
    NSC_K_FACTOR = 9,    /* set-up: banded LU of the per-mode matrices (once per dt)                 */
    NSC_K_DR = 10,       /* N1: radial derivative of the spectral fields (length-768 pipeline only)  */
    NSC_NKERN = 11
};
int nsc_set_profiling(nsc_ctx* ctx, int on);
int nsc_profile_read(nsc_ctx* ctx, double* h_ms, long long* h_count);
const char* nsc_kernel_name(int id);


/* Number of times nsc_step replayed its captured CUDA graph on this context (0 on the legacy default
 * stream or with profiling on, where the kernels are launched one by one).  For tests and reports. */
long long nsc_graph_replays(const nsc_ctx* ctx);

/* Measured fp64 peak of a device: a register-only
 * kernel on every SM, timed with CUDA events, best of six runs.  kind 0: DFMA only (2 flop each);
 * kind 1: DADD and DMUL alternating (1 flop each).  device: CUDA ordinal, -1 = current.
 * *h_tflops (HOST double) receives TFLOP/s.  Synchronises the device; needs no context.  The calling thread's
 * current device is the same after the call as before it.  NSC_EINVAL for an ordinal the machine does not have,
 * NSC_ECUDA if a CUDA call fails or no positive, finite rate could be measured. */
int nsc_fp64_peak(int kind, int device, double* h_tflops);

#ifdef __cplusplus
}
#endif
#endif /* NSC_H */
