"""Thin binding over the C-ABI library ``libnsc.so`` (include/nsc.h).

Argument marshalling only: every step of the time step runs in the library's CUDA kernels.
PyTorch supplies device memory and streams.  There is no fallback: if ``libnsc.so`` is missing
(run ``python -m paper_1908_00587_b200.build``) or no CUDA device is present, calls raise.

Names follow the header: ``nsc_create`` -> :class:`Context`, ``nsc_set_state``, ``nsc_nonlinear``,
``nsc_substep``, ``nsc_step``, ``nsc_get_state``, ``nsc_destroy``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnsc.so")

EXPORTS = (
    "nsc_create", "nsc_create_ex", "nsc_destroy", "nsc_set_stream", "nsc_get_grid",
    "nsc_set_state", "nsc_get_state", "nsc_set_state_host", "nsc_get_state_host",
    "nsc_nonlinear", "nsc_substep", "nsc_step", "nsc_step_iterated", "nsc_nusselt", "nsc_probe", "nsc_last_error", "nsc_device_bytes",
    "nsc_launch_count", "nsc_set_profiling", "nsc_profile_read", "nsc_kernel_name", "nsc_graph_replays",
    "nsc_fp64_peak", "nsc_cfl_rate", "nsc_advance", "nsc_mode_coefficient", "nsc_wave_speed", "nsc_regrid",
    "nsc_set_window", "nsc_step_phase", "nsc_field_pointers", "nsc_get_state_host_async", "nsc_host_copies_wait",
    "nsc_set_state_host_async", "nsc_probe_static",
)
NSC_NKERN = 11

NSC_OK, NSC_EINVAL, NSC_ENOMEM, NSC_ECUDA, NSC_ESTATE = 0, -1, -2, -3, -4


class NscError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libnsc error {code}: {msg}")
        self.code = code


class nsc_params(C.Structure):
    _fields_ = [
        ("N_r", C.c_int), ("M_theta", C.c_int), ("K_z", C.c_int),
        ("eta", C.c_double), ("alpha", C.c_double), ("k_theta0", C.c_int),
        ("Re_i", C.c_double), ("Re_o", C.c_double), ("Ra", C.c_double), ("Pr", C.c_double),
        ("radial_grid", C.c_int), ("n_theta_phys", C.c_int), ("n_z_phys", C.c_int),
        ("c", C.c_double), ("device", C.c_int), ("radial_chunk", C.c_int),
        ("linear_slices", C.c_int), ("no_graph", C.c_int),
    ]


class nsc_advance_info(C.Structure):
    _fields_ = [("t", C.c_double), ("dt_next", C.c_double), ("dt_last", C.c_double), ("dt_min", C.c_double),
                ("dt_max", C.c_double), ("err_last", C.c_double), ("cfl_rate_last", C.c_double),
                ("accepted", C.c_int), ("rejected", C.c_int), ("passes", C.c_int)]


_lib = None


def load_library() -> C.CDLL:
    """Loads libnsc.so (once) and declares the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_1908_00587_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dbl, i32 = C.c_void_p, C.c_double, C.c_int
    lib.nsc_create.argtypes = [C.POINTER(vp), i32, i32, i32, dbl, dbl, i32, dbl, dbl, dbl, dbl, i32]
    lib.nsc_create_ex.argtypes = [C.POINTER(vp), C.POINTER(nsc_params)]
    lib.nsc_destroy.argtypes = [vp]
    lib.nsc_set_stream.argtypes = [vp, vp]
    lib.nsc_get_grid.argtypes = [vp, C.POINTER(dbl)]
    lib.nsc_set_state.argtypes = [vp] + [vp] * 5
    lib.nsc_get_state.argtypes = [vp] + [vp] * 5
    lib.nsc_set_state_host.argtypes = [vp] + [vp] * 5
    lib.nsc_get_state_host.argtypes = [vp] + [vp] * 5
    lib.nsc_nonlinear.argtypes = [vp] + [vp] * 4
    lib.nsc_substep.argtypes = [vp] + [vp] * 4 + [dbl]
    lib.nsc_step.argtypes = [vp, dbl]
    lib.nsc_nusselt.argtypes = [vp, C.POINTER(dbl)]
    lib.nsc_probe.argtypes = [vp, i32, i32, dbl, dbl, C.POINTER(dbl)]
    lib.nsc_step_iterated.argtypes = [vp, dbl, dbl, i32, C.POINTER(i32), C.POINTER(dbl)]
    lib.nsc_last_error.argtypes = [vp]
    lib.nsc_last_error.restype = C.c_char_p
    lib.nsc_device_bytes.argtypes = [vp]
    lib.nsc_device_bytes.restype = C.c_longlong
    lib.nsc_launch_count.argtypes = [vp]
    lib.nsc_launch_count.restype = C.c_longlong
    lib.nsc_set_profiling.argtypes = [vp, i32]
    lib.nsc_profile_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(C.c_longlong)]
    lib.nsc_kernel_name.argtypes = [i32]
    lib.nsc_kernel_name.restype = C.c_char_p
    lib.nsc_graph_replays.argtypes = [vp]
    lib.nsc_graph_replays.restype = C.c_longlong
    lib.nsc_fp64_peak.argtypes = [i32, i32, C.POINTER(dbl)]
    lib.nsc_cfl_rate.argtypes = [vp, C.POINTER(dbl)]
    lib.nsc_advance.argtypes = [vp, dbl, i32, dbl, dbl, dbl, i32, C.POINTER(nsc_advance_info), C.POINTER(dbl)]
    lib.nsc_mode_coefficient.argtypes = [vp, i32, i32, i32, i32, C.POINTER(dbl)]
    lib.nsc_wave_speed.argtypes = [vp, i32, i32, i32, i32, dbl, i32, C.POINTER(dbl)]
    lib.nsc_regrid.argtypes = [vp, vp]
    lib.nsc_get_state_host_async.argtypes = [vp] + [vp] * 5
    lib.nsc_set_state_host_async.argtypes = [vp] + [vp] * 5
    lib.nsc_host_copies_wait.argtypes = [vp]
    lib.nsc_set_window.argtypes = [vp, i32, i32, C.c_longlong, C.c_longlong]
    lib.nsc_step_phase.argtypes = [vp, i32, dbl]
    lib.nsc_field_pointers.argtypes = [vp, i32, C.POINTER(vp)]
    lib.nsc_probe_static.argtypes = [vp, i32, i32, i32, i32, dbl, i32, dbl, dbl, vp, vp]
    for name in EXPORTS:
        if name not in ("nsc_last_error", "nsc_device_bytes", "nsc_launch_count", "nsc_kernel_name",
                        "nsc_graph_replays"):
            getattr(lib, name).restype = i32
    _lib = lib
    return lib


def _ptr(t):
    """Device (torch.Tensor) or host (numpy.ndarray) complex128 buffer -> void*; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        if t.dtype != np.complex128 or not t.flags["C_CONTIGUOUS"]:
            raise ValueError("host buffers must be C-contiguous complex128")
        return C.c_void_p(t.ctypes.data)
    import torch
    if t.dtype != torch.complex128 or not t.is_contiguous():
        raise ValueError("device buffers must be contiguous complex128")
    return C.c_void_p(t.data_ptr())


def fp64_peak(kind: int = 0, device: int = -1) -> float:
    """nsc_fp64_peak: measured fp64 TFLOP/s of the device (kind 0 DFMA, kind 1 DADD + DMUL)."""
    lib = load_library()
    v = C.c_double(0.0)
    rc = lib.nsc_fp64_peak(kind, device, C.byref(v))
    if rc != NSC_OK:
        raise NscError(rc, "nsc_fp64_peak failed (no CUDA device?)")
    return v.value


def probe_static(field, k_theta0, alpha, j, theta, z, out, stream=None):
    """nsc_probe_static: the value at (r_j, theta, z) of the physical field whose spectral coefficients ``field`` holds
    (a contiguous complex128 CUDA tensor [N_r, M_theta+1, 2 K_z+1] of the caller's), written to ``out`` (a float64 CUDA
    tensor with one element, also the caller's) by work enqueued on ``stream`` (a torch.cuda.Stream; None: torch's
    current stream).  For callers that must not allocate device memory: no context is needed and the library
    allocates nothing -- see include/nsc.h for the size limit (M_theta, K_z <= 512), the first-call set-up and why
    calls that overlap on one GPU must be ordered.  Returns at once; ``out`` is valid once the stream has run."""
    import torch
    lib = load_library()
    if field.dtype != torch.complex128 or not field.is_contiguous() or field.dim() != 3 or not field.is_cuda:
        raise ValueError("field must be a contiguous complex128 CUDA tensor [N_r, M_theta+1, 2 K_z+1]")
    if out.dtype != torch.float64 or out.numel() != 1 or not out.is_cuda:
        raise ValueError("out must be a float64 CUDA tensor with one element")
    N_r, M1, NK = field.shape
    if NK % 2 != 1:
        raise ValueError("the last axis of field holds 2 K_z + 1 axial modes: an odd number")
    s = stream if stream is not None else torch.cuda.current_stream()
    rc = lib.nsc_probe_static(C.c_void_p(field.data_ptr()), N_r, M1 - 1, (NK - 1) // 2, int(k_theta0), float(alpha),
                              int(j), float(theta), float(z), C.c_void_p(out.data_ptr()), C.c_void_p(s.cuda_stream))
    if rc != NSC_OK:
        raise NscError(rc, lib.nsc_last_error(None).decode())


class Context:
    """One Taylor-Couette configuration on one GPU (``nsc_create`` ... ``nsc_destroy``)."""

    def __init__(self, N_r, M, K, eta, alpha, k_theta0, Re_i, Re_o, Ra=0.0, Pr=1.0, grid=1,
                 n_theta=0, n_z=0, c=0.0, device=-1, radial_chunk=0, linear_slices=0, no_graph=0):
        self._lib = load_library()
        self._h = C.c_void_p()
        p = nsc_params(N_r, M, K, eta, alpha, k_theta0, Re_i, Re_o, Ra, Pr, grid, n_theta, n_z, c,
                       device, radial_chunk, linear_slices, no_graph)
        rc = self._lib.nsc_create_ex(C.byref(self._h), C.byref(p))
        if rc != NSC_OK:
            msg = self._lib.nsc_last_error(None).decode()
            self._h = None
            raise NscError(rc, msg)
        self.N_r, self.M, self.K = N_r, M, K
        self.heated = Ra != 0.0
        self.nf = 4 if self.heated else 3
        self.shape = (N_r, M + 1, 2 * K + 1)

    @classmethod
    def from_config(cls, cfg: dict, **over):
        keys = ("N_r", "M", "K", "eta", "alpha", "k_theta0", "Re_i", "Re_o", "Ra", "Pr", "grid")
        kw = {k: cfg[k] for k in keys}
        kw.update(over)
        return cls(**kw)

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc):
        if rc != NSC_OK:
            raise NscError(rc, self._lib.nsc_last_error(self._h).decode())

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.nsc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def set_stream(self, stream=None):
        """Enqueue all later work on ``stream`` (a torch.cuda.Stream; None: torch's current)."""
        import torch
        s = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.nsc_set_stream(self._h, C.c_void_p(s.cuda_stream)))

    def grid(self) -> np.ndarray:
        r = np.empty(self.N_r, np.float64)
        self._check(self._lib.nsc_get_grid(self._h, r.ctypes.data_as(C.POINTER(C.c_double))))
        return r

    def empty(self, n=1):
        import torch
        out = [torch.empty(self.shape, dtype=torch.complex128, device="cuda") for _ in range(n)]
        return out[0] if n == 1 else out

    # ------------------------------------------------------------------ the ABI calls
    def set_state(self, ur, uth, uz, T=None, p=None):
        host = isinstance(ur, np.ndarray)
        fn = self._lib.nsc_set_state_host if host else self._lib.nsc_set_state
        self._check(fn(self._h, _ptr(ur), _ptr(uth), _ptr(uz), _ptr(T), _ptr(p)))

    def get_state(self, ur=None, uth=None, uz=None, T=None, p=None):
        host = any(isinstance(a, np.ndarray) for a in (ur, uth, uz, T, p))
        fn = self._lib.nsc_get_state_host if host else self._lib.nsc_get_state
        self._check(fn(self._h, _ptr(ur), _ptr(uth), _ptr(uz), _ptr(T), _ptr(p)))

    def set_state_host_async(self, ur, uth, uz, T=None, p=None):
        """nsc_set_state_host_async from (pinned) numpy arrays; they may be reused after host_copies_wait()."""
        self._check(self._lib.nsc_set_state_host_async(self._h, _ptr(ur), _ptr(uth), _ptr(uz), _ptr(T), _ptr(p)))

    def get_state_host_async(self, ur=None, uth=None, uz=None, T=None, p=None):
        """nsc_get_state_host_async into (pinned) numpy arrays; complete after host_copies_wait()."""
        for a in (ur, uth, uz, T, p):
            if a is not None and not isinstance(a, np.ndarray):
                raise ValueError("get_state_host_async takes host (numpy) buffers")
        self._check(self._lib.nsc_get_state_host_async(self._h, _ptr(ur), _ptr(uth), _ptr(uz), _ptr(T), _ptr(p)))

    def host_copies_wait(self):
        self._check(self._lib.nsc_host_copies_wait(self._h))

    def nonlinear(self, Nr, Nth, Nz, NT=None):
        self._check(self._lib.nsc_nonlinear(self._h, _ptr(Nr), _ptr(Nth), _ptr(Nz), _ptr(NT)))

    def substep(self, Er, Eth, Ez, ET, dt):
        self._check(self._lib.nsc_substep(self._h, _ptr(Er), _ptr(Eth), _ptr(Ez), _ptr(ET), float(dt)))

    def nusselt(self):
        """nsc_nusselt: (Nu_i, Nu_o, Nu_w_i, Nu_w_o) of the current state."""
        out = (C.c_double * 4)()
        self._check(self._lib.nsc_nusselt(self._h, out))
        return tuple(out)

    def probe(self, field, j, theta, z):
        """nsc_probe: the physical field ``field`` (0 u_r, 1 u_theta, 2 u_z, 3 T, 4 p) at (r_j, theta, z)."""
        v = C.c_double(0.0)
        self._check(self._lib.nsc_probe(self._h, field, j, theta, z, C.byref(v)))
        return v.value

    def step_iterated(self, dt, tol, max_corr):
        """nsc_step_iterated: returns (corrector passes, last convergence norm)."""
        k, err = C.c_int(0), C.c_double(0.0)
        self._check(self._lib.nsc_step_iterated(self._h, dt, tol, max_corr, C.byref(k), C.byref(err)))
        return k.value, err.value

    def cfl_rate(self) -> float:
        v = C.c_double(0.0)
        self._check(self._lib.nsc_cfl_rate(self._h, C.byref(v)))
        return v.value

    def advance(self, t_end, max_steps, dt0, tol, cfl, max_corr):
        """nsc_advance: returns (info dict, log) with log = list of (dt, passes, err, accepted) per attempt."""
        info = nsc_advance_info()
        log = (C.c_double * (4 * max_steps))()
        self._check(self._lib.nsc_advance(self._h, t_end, max_steps, dt0, tol, cfl, max_corr, C.byref(info), log))
        n = info.accepted + info.rejected
        out = [(log[4 * i], int(log[4 * i + 1]), log[4 * i + 2], bool(log[4 * i + 3])) for i in range(n)]
        return {f: getattr(info, f) for f, _ in nsc_advance_info._fields_}, out

    def mode_coefficient(self, field, j, m, k) -> complex:
        v = (C.c_double * 2)()
        self._check(self._lib.nsc_mode_coefficient(self._h, field, j, m, k, v))
        return complex(v[0], v[1])

    def wave_speed(self, field, j, m, k, dt, n_steps) -> float:
        v = C.c_double(0.0)
        self._check(self._lib.nsc_wave_speed(self._h, field, j, m, k, dt, n_steps, C.byref(v)))
        return v.value

    def regrid_from(self, src: "Context"):
        """nsc_regrid: this context's state := src's state interpolated / padded onto this resolution."""
        self._check(self._lib.nsc_regrid(self._h, src._h))

    def set_window(self, j0=0, nj=0, e0=0, ne=0):
        self._check(self._lib.nsc_set_window(self._h, j0, nj, e0, ne))

    def step_phase(self, phase, dt):
        self._check(self._lib.nsc_step_phase(self._h, phase, dt))

    def field_tensors(self, which):
        """nsc_field_pointers as torch views [N_r, (M+1)(2K+1)] (complex128, no copy) of the library's arrays:
        which = 0 state, 1 predictor, 2 N0, 3 N1."""
        import torch
        ptrs = (C.c_void_p * 4)()
        self._check(self._lib.nsc_field_pointers(self._h, which, ptrs))
        n_modes = self.shape[1] * self.shape[2]
        out = []
        for i in range(self.nf):
            iface = {"shape": (self.N_r, n_modes, 2), "typestr": "<f8", "data": (int(ptrs[i]), False), "version": 3}
            holder = type("_DevArray", (), {"__cuda_array_interface__": iface})()
            out.append(torch.view_as_complex(torch.as_tensor(holder, device="cuda")))
        return out

    def step(self, dt):
        self._check(self._lib.nsc_step(self._h, float(dt)))

    def device_bytes(self) -> int:
        return int(self._lib.nsc_device_bytes(self._h))

    def launch_count(self) -> int:
        return int(self._lib.nsc_launch_count(self._h))

    def graph_replays(self) -> int:
        return int(self._lib.nsc_graph_replays(self._h))

    def set_profiling(self, on: bool):
        self._check(self._lib.nsc_set_profiling(self._h, int(bool(on))))

    def profile_read(self) -> dict:
        """{kernel name: (milliseconds, launches)} accumulated since the last read."""
        ms = (C.c_double * NSC_NKERN)()
        cnt = (C.c_longlong * NSC_NKERN)()
        self._check(self._lib.nsc_profile_read(self._h, ms, cnt))
        return {self._lib.nsc_kernel_name(i).decode(): (ms[i], cnt[i]) for i in range(NSC_NKERN)}

    # ------------------------------------------------------------------ conveniences (copies only)
    def state_to_host(self):
        """Current state as numpy arrays [u_r, u_theta, u_z, T or None, p]."""
        out = [np.empty(self.shape, np.complex128) for _ in range(5)]
        if not self.heated:
            out[3] = None
        self.get_state(*out)
        return out

    def nonlinear_to_host(self):
        import torch
        bufs = self.empty(self.nf)
        self.nonlinear(*bufs)
        torch.cuda.synchronize()
        return [b.cpu().numpy() for b in bufs]
