"""Seeded synthetic inputs shaped like the paper's workloads.

This module feeds BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic: no finite differences, no transforms, no solves.  Everything here is
a closed-form expression evaluated on the radial nodes handed in by the caller
(``nsc_get_grid`` on the CUDA side, ``oracle.radial_grid`` on the oracle side).

The five configurations are those of BASELINE.json ``configs`` (index 0..4 = cfg 1..5);
values it leaves open (alpha for cfg 3-5, dt for cfg 2-5, amplitudes) are DESIGN.md
reading R12.  The paper's production fields are not available; these stand in for them.

Perturbation recipe, per Fourier mode (m,k) != (0,0) with x = r - r_i in [0,1] and
T_q the Chebyshev polynomials in 2x-1 (q = 0..2), complex standard-normal a,b,c,d:
    u_r  = A_mk x^2 (1-x)^2 sum_q a_q T_q          (degree 6: u_r = du_r/dr = 0 at walls)
    u_th = A_mk x (1-x)     sum_q b_q T_q
    kappa != 0:  u_z  = -(u_r' + u_r/r + (i n/r) u_th) / (i kappa)
    kappa == 0:  u_z  = A_mk x (1-x) sum_q c_q T_q,   u_th = -r (u_r' + u_r/r) / (i n)
    T'   = A_mk x (1-x) sum_q d_q T_q
with u_r' the exact derivative of the polynomial, so the field is divergence-free
analytically (and discretely to round-off, because a 9-point stencil differentiates a
degree-6 polynomial exactly).  m = 0: k > 0 drawn, k < 0 mirrored by conjugation.
"""
from __future__ import annotations

import math
import numpy as np
from numpy.polynomial import chebyshev as _cheb
from numpy.polynomial import polynomial as _poly

# BASELINE.json configs; alpha/dt/amp where BASELINE.json is silent: DESIGN.md R12.
CONFIGS = [
    dict(name="cfg1", N_r=32, M=8, K=8, eta=0.5, alpha=3.0, k_theta0=1, Re_i=100.0, Re_o=0.0,
         Ra=0.0, Pr=1.0, grid=1, amp=1e-3, band=2, slope_offset=1.0, dt=1e-3),
    dict(name="cfg2", N_r=64, M=32, K=32, eta=0.71, alpha=math.pi, k_theta0=1, Re_i=1000.0, Re_o=0.0,
         Ra=0.0, Pr=1.0, grid=1, amp=1e-2, band=None, slope_offset=1.0, dt=3e-5),
    dict(name="cfg3", N_r=128, M=128, K=128, eta=0.5, alpha=math.pi, k_theta0=2, Re_i=2000.0,
         Re_o=-1000.0, Ra=1e6, Pr=0.7, grid=1, amp=1e-2, band=None, slope_offset=1.0, dt=5e-8),
    dict(name="cfg4", N_r=256, M=256, K=256, eta=0.71, alpha=math.pi, k_theta0=4, Re_i=10000.0,
         Re_o=0.0, Ra=0.0, Pr=1.0, grid=1, amp=1e-2, band=None, slope_offset=0.0, dt=1e-7),
    dict(name="cfg5", N_r=512, M=512, K=512, eta=0.909, alpha=math.pi, k_theta0=8, Re_i=30000.0,
         Re_o=-10000.0, Ra=1e7, Pr=1.0, grid=1, amp=1e-2, band=None, slope_offset=1.0, dt=3e-9),
]
SEED0 = 190800587

PHYS_KEYS = ("N_r", "M", "K", "eta", "alpha", "k_theta0", "Re_i", "Re_o", "Ra", "Pr", "grid")


def config(i: int) -> dict:
    """Config i = 0..4 (cfg 1..5) with its seed."""
    c = dict(CONFIGS[i])
    c["seed"] = SEED0 + i
    return c


def scaled_config(i: int, N_r=None, M=None, K=None) -> dict:
    """A config's physics at a reduced resolution (parity cases the oracle finishes fast)."""
    c = config(i)
    if N_r:
        c["N_r"] = N_r
    if M:
        c["M"] = M
    if K:
        c["K"] = K
    return c


def couette(r, eta, Re_i, Re_o):
    """Circular Couette flow u_theta = A r + B / r (wall speeds Re_i, Re_o)."""
    A = (Re_o - eta * Re_i) / (1 + eta)
    B = eta * (Re_i - eta * Re_o) / ((1 - eta) * (1 - eta ** 2))
    return A * r + B / r


def conductive_T(r, eta):
    """Conductive temperature T_b = ln(r/r_o)/ln(eta) - 1/2: +1/2 inside, -1/2 outside."""
    r_o = 1 / (1 - eta)
    return np.log(r / r_o) / math.log(eta) - 0.5


def axial_base_flow(r, eta, Ra, Pr):
    """Closed-form steady axial flow driven by (Ra/Pr) T_b with no mean pressure gradient:
    (1/r)(r w')' = -(Ra/Pr) T_b,  w(r_i) = w(r_o) = 0."""
    r_i, r_o = eta / (1 - eta), 1 / (1 - eta)
    a = 1 / math.log(eta)
    b = -math.log(r_o) / math.log(eta) - 0.5

    def part(x):
        return -(Ra / Pr) * (a * (x * x / 4 * np.log(x) - x * x / 4) + b * x * x / 4)

    # C1 ln r + C2 from the two wall conditions
    M2 = np.array([[math.log(r_i), 1.0], [math.log(r_o), 1.0]])
    C1, C2 = np.linalg.solve(M2, -np.array([part(r_i), part(r_o)]))
    return part(r) + C1 * np.log(r) + C2


def _radial_basis(x):
    """Values on the nodes of x^2(1-x)^2 T_q, its exact derivative, and x(1-x) T_q, q=0..2."""
    bump2 = _poly.polymul([0, 1, -1], [0, 1, -1])      # x^2 (1-x)^2 as power series in x
    bump1 = np.array([0.0, 1.0, -1.0])                  # x (1-x)
    B2, dB2, B1 = [], [], []
    for q in range(3):
        cq = np.zeros(q + 1)
        cq[q] = 1.0
        # T_q(2x-1) as a power series in x
        tq = _cheb.cheb2poly(cq)
        comp = np.array([0.0])
        lin = np.array([-1.0, 2.0])
        pw = np.array([1.0])
        for coef in tq:
            comp = _poly.polyadd(comp, coef * pw)
            pw = _poly.polymul(pw, lin)
        p2 = _poly.polymul(bump2, comp)
        B2.append(_poly.polyval(x, p2))
        dB2.append(_poly.polyval(x, _poly.polyder(p2)))
        B1.append(_poly.polyval(x, _poly.polymul(bump1, comp)))
    return np.array(B2), np.array(dB2), np.array(B1)     # each [3, N_r]


def make_state(cfg: dict, r: np.ndarray):
    """Initial state (u_r, u_theta, u_z, T or None, p) on the nodes ``r`` for ``cfg``.
    Arrays are complex128 [N_r, M+1, 2K+1], k index = k + K."""
    N_r, M, K = cfg["N_r"], cfg["M"], cfg["K"]
    eta, alpha, kth0 = cfg["eta"], cfg["alpha"], cfg["k_theta0"]
    heated = cfg["Ra"] != 0.0
    rng = np.random.Generator(np.random.PCG64(cfg["seed"]))
    r = np.asarray(r, dtype=np.float64)
    x = r - r[0]
    B2, dB2, B1 = _radial_basis(x)
    shp = (M + 1, 2 * K + 1)

    def cn():
        return rng.standard_normal((3,) + shp) + 1j * rng.standard_normal((3,) + shp)

    a, b, c, d = cn(), cn(), cn(), cn()
    m = np.arange(M + 1)[:, None] * np.ones((1, 2 * K + 1))
    k = np.ones((M + 1, 1)) * np.arange(-K, K + 1)[None, :]
    A = (cfg["slope_offset"] + m * m + k * k)
    A[0, K] = 1.0
    A = A ** (-5.0 / 6.0)
    A[0, K] = 0.0                                        # no perturbation in mode (0,0)
    if cfg.get("band"):
        A = np.where((m <= cfg["band"]) & (np.abs(k) <= cfg["band"]), A, 0.0)
    n = (m * kth0)[None]
    kap = (k * alpha)[None]
    rr = r[:, None, None]
    ur = A[None] * np.einsum("qj,qmk->jmk", B2, a)
    dur = A[None] * np.einsum("qj,qmk->jmk", dB2, a)
    ut = A[None] * np.einsum("qj,qmk->jmk", B1, b)
    uzf = A[None] * np.einsum("qj,qmk->jmk", B1, c)
    Tp = A[None] * np.einsum("qj,qmk->jmk", B1, d)
    kz = (kap != 0.0)
    with np.errstate(divide="ignore", invalid="ignore"):
        uz_div = -(dur + ur / rr + 1j * n / rr * ut) / (1j * kap)
        ut_div = -rr * (dur + ur / rr) / (1j * n)
    uz = np.where(kz, uz_div, uzf)
    ut = np.where(kz, ut, np.where(n != 0, ut_div, 0.0))
    for f in (ur, ut, uz, Tp):
        f[:, 0, K] = 0.0
        f[:, 0, :K] = np.conj(f[:, 0, :K:-1])            # m = 0: k < 0 mirrors k > 0
    # scale: rms(u') = amp * U, via Parseval over (theta, z), plain mean over nodes/components
    w = np.where(np.arange(M + 1) == 0, 1.0, 2.0)[None, :, None]
    ms = sum((w * np.abs(f) ** 2).sum(axis=(1, 2)).mean() for f in (ur, ut, uz)) / 3.0
    U = max(abs(cfg["Re_i"]), abs(cfg["Re_o"]))
    s = cfg["amp"] * U / math.sqrt(ms)
    ur, ut, uz = s * ur, s * ut, s * uz
    ut[:, 0, K] += couette(r, eta, cfg["Re_i"], cfg["Re_o"])
    T = None
    if heated:
        msT = (w * np.abs(Tp) ** 2).sum(axis=(1, 2)).mean()
        T = Tp * (cfg["amp"] / math.sqrt(msT))
        T[:, 0, K] += conductive_T(r, eta)
        uz[:, 0, K] += axial_base_flow(r, eta, cfg["Ra"], cfg["Pr"])
    p = np.zeros((N_r,) + shp, complex)
    return [np.ascontiguousarray(ur), np.ascontiguousarray(ut), np.ascontiguousarray(uz),
            None if T is None else np.ascontiguousarray(T), p]
