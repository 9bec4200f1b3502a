"""Oracle: plain, slow fp64 CPU restatement of one nsCouette predictor-corrector step.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (the package
``paper_1908_00587_b200``) may import this module; only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs do.  It shares no code, table or constant with the CUDA path.

What it restates (citations are PAPER.md:<line>, or
DESIGN.md reading R#):

* PAPER.md:36      cylindrical coordinates, primitive variables (u_r, u_theta, u_z, p, T)
* PAPER.md:42      Fourier-Galerkin in theta and z; 9-point finite differences in r on a
                   radial grid selected at run time
* PAPER.md:44      axial periodicity
* PAPER.md:46      predictor-corrector time integration, implicit linear terms
* PAPER.md:48-50   Boussinesq heat transfer, negative radial temperature gradient, gravity || z
* PAPER.md:64      linear terms solved independently per Fourier mode; nonlinear terms need
                   all modes of a radial node
* PAPER.md:100     the basic state depends on r only (circular Couette flow, conductive T)
* PAPER.md:108     time unit d^2/nu

The paper prints no equations; every numerical choice is a DESIGN.md reading (R1..R15,
taken from SURVEY.md 8(c) S1..S15).  Layout of every spectral field: complex128 array
``[N_r, M+1, 2K+1]``, ``m = 0..M``, ``k index = k + K``, ``j = 0`` at the inner wall.

Transforms are naive O(N^2) sums written as matrix products with explicit root-of-unity
tables (``dft="naive"``).  ``dft="fft"`` swaps those sums for numpy's FFT routines (a
library primitive standing for the same sums; pinned to the naive sums in
tests/test_oracle_transforms.py) so that the large configurations finish.

Linear solves are dense Gaussian elimination with partial pivoting after row
equilibration (LAPACK ``gesv`` through ``numpy.linalg.solve`` on row-scaled matrices).
``solve="c"`` is the same banded elimination written in plain C (oracle/nsc_oracle_sub.c, the whole
sub-step L1-L5 per mode, OpenMP over modes), pinned to both numpy backends.
``solve="banded"`` is the second backend BASELINE.json north_star allows ("dense or banded
Gaussian elimination"): the same matrices held by diagonals and eliminated row by row without
pivoting, vectorised over the Fourier modes, and the radial operators applied through their
9-point rows instead of dense matrices.  It is pinned to the dense backend
(tests/test_oracle_banded.py) and exists so that 20-step runs at the large configurations
finish; plain numpy throughout, so it also runs in ``real=numpy.longdouble`` (SURVEY.md 8(c):
"oracle(double) vs oracle(long double) after 20 steps is reported as the floor"), where the
tables are kept in extended precision instead of being rounded to double.  The sub-step treats
chunks of Fourier modes independently; with the banded backend the chunks are
handed to a thread pool (outer-loop parallelism only, as SURVEY.md section 7 plans for the oracle).

Parity unpinned (defined by the algorithm only): the pressure field,
the O(dt^2) tangential wall slip, and the aliased extreme modes |k| = K, m = M.
"""
from __future__ import annotations

import concurrent.futures
import dataclasses
import os
import numpy as np
import scipy.fft as _fft          # pocketfft, the routines behind numpy.fft, with a ``workers`` argument

LD = np.longdouble


# --------------------------------------------------------------------------------------
# parameters
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class Params:
    """Arguments of ``nsc_create`` (BASELINE.json north_star; "number of
    points, modes ... rotation rates")."""
    N_r: int
    M: int                 # azimuthal modes m = 0..M
    K: int                 # axial modes k = -K..K
    eta: float             # radius ratio r_i / r_o
    alpha: float           # axial base wavenumber, kappa = k * alpha
    k_theta0: int          # azimuthal base wavenumber, n = m * k_theta0
    Re_i: float
    Re_o: float
    Ra: float = 0.0
    Pr: float = 1.0
    grid: int = 1          # 0 uniform, 1 Chebyshev-Gauss-Lobatto (R2)
    n_theta: int = 0       # physical grid; 0 => 3M (R4)
    n_z: int = 0           # physical grid; 0 => 3K (R4)
    c: float = 0.5         # implicitness (R10)

    def __post_init__(self):
        if self.n_theta == 0:
            self.n_theta = 3 * self.M
        if self.n_z == 0:
            self.n_z = 3 * self.K

    @property
    def heated(self) -> bool:      # R13: temperature on iff Ra != 0
        return self.Ra != 0.0


# --------------------------------------------------------------------------------------
# O1 radial grid, O2 finite-difference tables
# --------------------------------------------------------------------------------------
def radial_grid(N_r: int, eta: float, kind: int, dtype=np.float64):
    """O1.  Gap d = r_o - r_i = 1, r_i = eta/(1-eta) (R1; PAPER.md:108 fixes d as length
    unit).  kind 0: uniform; kind 1: Chebyshev-Gauss-Lobatto clustering (R2)."""
    eta = LD(eta)
    r_i = eta / (1 - eta)
    j = np.arange(N_r, dtype=LD)
    if kind == 0:
        r = r_i + j / (N_r - 1)
    elif kind == 1:
        r = r_i + (1 - np.cos(_pi_ld() * j / (N_r - 1))) / 2
    else:
        raise ValueError("radial grid kind must be 0 or 1")
    return r.astype(dtype)


def _pi_ld():
    return LD(4) * np.arctan(LD(1))


def stencil_start(j: int, N_r: int, npt: int = 9) -> int:
    """R3: 9-node window centred inside, shifted (one-sided) at the walls."""
    return min(max(j - npt // 2, 0), N_r - npt)


def fd_tables(r_ld, npt: int = 9):
    """O2.  Dense D1, D2 [N_r, N_r] in long double: derivatives at r_j of the degree-8
    Lagrange basis on the stencil S(j) ("stencil-length ... nine points").

    l != j:  l_l'(x_j)  = prod_{q != l,j}(x_j-x_q) / prod_{q != l}(x_l-x_q)
             l_l''(x_j) = 2 l_l'(x_j) * sum_{q != l,j} 1/(x_j-x_q)
    l == j:  l_j'(x_j)  = s1 = sum_{q != j} 1/(x_j-x_q)
             l_j''(x_j) = s1^2 - sum_{q != j} 1/(x_j-x_q)^2
    """
    r_ld = np.asarray(r_ld, dtype=LD)
    N = len(r_ld)
    D1 = np.zeros((N, N), LD)
    D2 = np.zeros((N, N), LD)
    for j in range(N):
        s = stencil_start(j, N, npt)
        x = r_ld[s:s + npt]
        jl = j - s
        xj = x[jl]
        for a in range(npt):
            l = s + a
            if a == jl:
                inv = [1 / (xj - x[q]) for q in range(npt) if q != jl]
                s1 = sum(inv, LD(0))
                D1[j, l] = s1
                D2[j, l] = s1 * s1 - sum((v * v for v in inv), LD(0))
            else:
                num = LD(1)
                den = LD(1)
                for q in range(npt):
                    if q != a and q != jl:
                        num *= xj - x[q]
                    if q != a:
                        den *= x[a] - x[q]
                w1 = num / den
                D1[j, l] = w1
                D2[j, l] = 2 * w1 * sum((1 / (xj - x[q]) for q in range(npt)
                                         if q != a and q != jl), LD(0))
    return D1, D2


def roots_of_unity(N: int, real=np.float64):
    """exp(2 pi i t / N), t = 0..N-1, evaluated in long double, rounded once (O3)."""
    t = np.arange(N, dtype=LD)
    ang = 2 * _pi_ld() * t / N
    return np.cos(ang).astype(real) + 1j * np.sin(ang).astype(real)


# --------------------------------------------------------------------------------------
# the oracle
# --------------------------------------------------------------------------------------
class Oracle:
    """One Taylor-Couette configuration; methods follow O3..O8 in SURVEY.md 8(c)."""

    def __init__(self, p: Params, dft: str = "naive", solve: str = "dense", real=np.float64):
        if solve not in ("dense", "banded", "c"):
            raise ValueError("solve must be 'dense', 'banded' or 'c'")
        if real is not np.float64 and solve != "banded":
            raise ValueError("extended precision needs solve='banded' (LAPACK and the C backend are double only)")
        self.p = p
        self.dft = dft
        self.solve = solve
        self.band_ops = solve != "dense"                     # radial operators through their 9-point rows
        self.real = real
        self.cplx = np.result_type(real, np.complex64)       # complex128 / clongdouble
        N_r = p.N_r
        r_ld = radial_grid(N_r, p.eta, p.grid, dtype=LD)
        D1, D2 = fd_tables(r_ld)
        inv_r = 1 / r_ld
        L0 = D2 + inv_r[:, None] * D1                        # d2/dr2 + (1/r) d/dr
        Gt = D1.copy()                                       # G~: D1 with wall rows zeroed
        Gt[0, :] = 0
        Gt[-1, :] = 0
        Q = (D1 + np.diag(inv_r)) @ Gt                       # (D1 + 1/r) G~, product in LD
        f64 = real
        self.r = r_ld.astype(f64)
        self.D1, self.D2 = D1.astype(f64), D2.astype(f64)
        self.L0, self.Gt, self.Q = L0.astype(f64), Gt.astype(f64), Q.astype(f64)
        # wavenumbers (BASELINE.json (a): i*m*k_theta0 and i*k*alpha)
        self.n = (np.arange(p.M + 1) * p.k_theta0).astype(f64)          # [M+1]
        self.kappa = (np.arange(-p.K, p.K + 1) * p.alpha).astype(f64)   # [2K+1]
        # O3 root tables, indexed by (m*a mod N_theta), (k*b mod N_z)
        wt = roots_of_unity(p.n_theta, real)
        wz = roots_of_unity(p.n_z, real)
        m = np.arange(p.M + 1)[:, None]
        a = np.arange(p.n_theta)[None, :]
        k = np.arange(-p.K, p.K + 1)[:, None]
        b = np.arange(p.n_z)[None, :]
        self.Et = wt[(m * a) % p.n_theta]                    # [M+1, N_theta]
        self.Ez = wz[(k * b) % p.n_z]                        # [2K+1, N_z]
        self.cm = np.where(np.arange(p.M + 1) == 0, 1.0, 2.0).astype(f64)
        # band form of the radial operators (solve="banded"): row j of D1 / L0 on its stencil S(j)
        self.s0 = np.array([stencil_start(j, N_r) for j in range(N_r)])
        cols = self.s0[:, None] + np.arange(9)[None, :]
        rows = np.arange(N_r)[:, None]
        self.D1_rows = self.D1[rows, cols]                   # [N_r, 9]
        self.L0_rows = self.L0[rows, cols]

    # ---------------------------------------------------------------- O3 transforms
    def to_physical(self, fh):
        """u(theta_a, z_b) = Re[sum_k u^(0,k) e^{2 pi i k b/N_z}]
                             + 2 Re[sum_{m>=1} sum_k u^(m,k) e^{2 pi i (m a/N_theta + k b/N_z)}].
        fh: [..., M+1, 2K+1] -> real [..., N_theta, N_z]."""
        p = self.p
        if self.dft == "fft":
            pad = np.zeros(fh.shape[:-2] + (p.n_theta // 2 + 1, p.n_z), self.cplx)
            kk = np.arange(-p.K, p.K + 1) % p.n_z
            pad[..., :p.M + 1, kk] = fh
            half = _fft.ifft(pad, axis=-1, workers=-1) * p.n_z
            return _fft.irfft(half, n=p.n_theta, axis=-2, workers=-1) * p.n_theta
        half = fh @ self.Ez                                   # sum over k -> [..., M+1, N_z]
        half = half * self.cm[:, None]
        return np.real(np.swapaxes(np.swapaxes(half, -1, -2) @ self.Et, -1, -2))

    def from_physical(self, u):
        """u^(m,k) = 1/(N_theta N_z) sum_{a,b} u(theta_a,z_b) e^{-2 pi i (m a/N_theta + k b/N_z)}
        for 0 <= m <= M, |k| <= K; everything else discarded (truncation).
        u: real [..., N_theta, N_z] -> [..., M+1, 2K+1]."""
        p = self.p
        if self.dft == "fft":
            h = _fft.fft(_fft.rfft(u, axis=-2, workers=-1), axis=-1, workers=-1) / (p.n_theta * p.n_z)
            kk = np.arange(-p.K, p.K + 1) % p.n_z
            return h[..., :p.M + 1, :][..., kk]
        t = np.conj(self.Et) @ u                              # sum over a -> [..., M+1, N_z]
        return (t @ np.conj(self.Ez).T) / (p.n_theta * p.n_z)

    # ---------------------------------------------------------------- O5 operators
    def _rows9(self, rows9, f, js=None):
        """sum_{l in S(j)} rows9[j, l - s0(j)] f_l written out over the nine stencil nodes (banded backend)."""
        js = np.arange(self.p.N_r) if js is None else np.asarray(js)
        out = np.zeros((len(js),) + f.shape[1:], np.result_type(f.dtype, rows9.dtype))
        for l in range(9):
            out += rows9[js, l][:, None, None] * f[self.s0[js] + l]
        return out

    def d_r(self, f):
        """Radial derivative: sum_{l in S(j)} D1[j,l] f_l (N1)."""
        if self.band_ops:
            return self._rows9(self.D1_rows, f)
        return np.einsum("jl,lmk->jmk", self.D1, f)

    def lap(self, f, shift: int):
        """(L0 - diag((n+shift)^2/r^2 + kappa^2)) f.  shift = 0: scalar Laplacian L_s;
        shift = +-1: L_+- acting on u_+- = u_r +- i u_theta (O5)."""
        q = ((self.n[None, :, None] + shift) ** 2 / self.r[:, None, None] ** 2
             + self.kappa[None, None, :] ** 2)
        if self.band_ops:
            return self._rows9(self.L0_rows, f) - q * f
        return np.einsum("jl,lmk->jmk", self.L0, f) - q * f

    def divergence(self, ur, ut, uz):
        """D1 u_r + u_r/r + (i n/r) u_theta + i kappa u_z (O5)."""
        r = self.r[:, None, None]
        return (self.d_r(ur) + ur / r + 1j * self.n[None, :, None] / r * ut
                + 1j * self.kappa[None, None, :] * uz)

    # ---------------------------------------------------------------- O4 nonlinear term
    def nonlinear(self, ur, ut, uz, T=None, nodes=None, workers=1):
        """N = -(u.grad)u with the cylindrical curvature terms, + (Ra/Pr) T^ e_z, and
        N_T = -(u.grad)T (N1..N6; convective form, R7).  Evaluated at every radial node
        (walls included) or at the listed ``nodes`` only (same values; used for sampled
        parity at the large configurations).  Returns [N_r, N_theta, N_z, (N_T)] spectral."""
        p = self.p
        fields = [ur, ut, uz] + ([T] if p.heated else [])
        js = np.arange(p.N_r) if nodes is None else np.asarray(nodes)
        if workers > 1 and len(js) > 16:
            # radial nodes are independent: chunks of 16 nodes on a thread pool, same values
            parts = [js[i:i + 16] for i in range(0, len(js), 16)]
            with concurrent.futures.ThreadPoolExecutor(max_workers=workers) as ex:
                res = list(ex.map(lambda q: self.nonlinear(ur, ut, uz, T, nodes=q), parts))
            return [np.concatenate([r_[i] for r_ in res]) for i in range(len(fields))]
        i_n = 1j * self.n[None, :, None]
        i_k = 1j * self.kappa[None, None, :]
        rj = self.r[js][:, None, None]
        ph, d_r, d_t, d_z = [], [], [], []
        for f in fields:
            fj = f[js]
            ph.append(self.to_physical(fj))
            d_r.append(self.to_physical(self._rows9(self.D1_rows, f, js) if self.band_ops
                                        else np.einsum("jl,lmk->jmk", self.D1[js], f)))
            d_t.append(self.to_physical(i_n * fj))
            d_z.append(self.to_physical(i_k * fj))
        Ur, Ut, Uz = ph[0], ph[1], ph[2]

        def adv(i):
            return Ur * d_r[i] + (Ut / rj) * d_t[i] + Uz * d_z[i]

        Nr = -(adv(0) - Ut * Ut / rj)
        Nt = -(adv(1) + Ur * Ut / rj)
        Nz = -adv(2)
        out = [self.from_physical(Nr), self.from_physical(Nt), self.from_physical(Nz)]
        if p.heated:
            out[2] = out[2] + (p.Ra / p.Pr) * T[js]           # Boussinesq buoyancy (R8)
            out.append(self.from_physical(-adv(3)))
        return out

    # ---------------------------------------------------------------- O6 sub-step
    def _solve_rows(self, A, b):
        """Dense LU with partial pivoting after row equilibration.  A [B,N,N] real,
        b [B,N] complex."""
        s = 1.0 / np.abs(A).max(axis=2)
        return np.linalg.solve(A * s[:, :, None], (b * s)[:, :, None])[:, :, 0]

    # band storage: ab[b, j, d] = A_b[j, j - kl + d], d = 0 .. kl + ku
    @staticmethod
    def _band_pack(A, kl, ku):
        N = A.shape[0]
        ab = np.zeros((N, kl + ku + 1), A.dtype)
        for j in range(N):
            for d in range(kl + ku + 1):
                c = j - kl + d
                if 0 <= c < N:
                    ab[j, d] = A[j, c]
        outside = A.copy()
        for j in range(N):
            outside[j, max(0, j - kl):min(N, j + ku + 1)] = 0
        assert not outside.any(), "matrix does not fit the band"
        return ab

    @staticmethod
    def _solve_banded(ab, b, kl, ku):
        """Gaussian elimination WITHOUT pivoting inside the band, row by row, every step
        vectorised over the batch (BASELINE.json north_star: "dense or banded Gaussian
        elimination").  ab [N, kl+ku+1, B] real (overwritten; batch index last so that every
        vector operation is contiguous), b [N, B] complex (overwritten).  The multiplier of
        (row i, pivot j) is skipped where it is structurally zero: left of the first stored entry
        of row i in the batch-independent pattern."""
        N, W, B = ab.shape
        first = np.array([j - kl + int(np.argmax(np.any(ab[j] != 0, axis=1))) for j in range(N)])
        for j in range(N - 1):
            piv = ab[j, kl]
            for i in range(j + 1, min(j + kl, N - 1) + 1):
                if j < first[i]:
                    continue
                o = kl - (i - j)
                l = ab[i, o] / piv
                ab[i, o:o + ku + 1] -= l[None, :] * ab[j, kl:kl + ku + 1]
                b[i] -= l * b[j]
        for j in range(N - 1, -1, -1):
            acc = b[j]
            for d in range(1, min(ku, N - 1 - j) + 1):
                acc = acc - ab[j, kl + d] * b[j + d]
            b[j] = acc / ab[j, kl]
        return b

    def _helmholtz_banded(self, shift, coef, rhs, im, ik):
        KL = KU = 8
        N_r = self.p.N_r
        if not hasattr(self, "_L0_band"):
            self._L0_band = self._band_pack(self.L0, KL, KU)
        q = ((self.n[im] + shift)[None, :] ** 2 / self.r[:, None] ** 2 + self.kappa[ik][None, :] ** 2)   # [N_r, B]
        ab = np.broadcast_to((-coef * self._L0_band)[:, :, None], (N_r, KL + KU + 1, len(im))).copy()
        ab[:, KL, :] += 1 + coef * q
        for w in (0, N_r - 1):
            ab[w] = 0
            ab[w, KL] = 1
        return self._solve_banded(ab, np.array(rhs.T, dtype=self.cplx), KL, KU).T

    def _poisson_banded(self, g, im, ik):
        KL = KU = 12
        N_r = self.p.N_r
        if not hasattr(self, "_P_band"):
            P0 = self.Q.copy()
            P0[0, :] = self.D1[0]
            P0[-1, :] = self.D1[-1]
            self._P_band = self._band_pack(P0, KL, KU)
        q = self.n[im][None, :] ** 2 / self.r[:, None] ** 2 + self.kappa[ik][None, :] ** 2
        ab = np.broadcast_to(self._P_band[:, :, None], (N_r, KL + KU + 1, len(im))).copy()
        ab[1:-1, KL, :] -= q[1:-1]
        zero = (np.asarray(im) == 0) & (np.asarray(ik) == self.p.K)
        ab[:, :, zero] = 0
        ab[:, KL, zero] = 1                                    # O8: mode (0,0) is not projected
        phi = self._solve_banded(ab, np.array(g.T, dtype=self.cplx), KL, KU).T
        phi[zero] = 0.0
        return phi

    def _helmholtz(self, shift, coef, rhs, im, ik):
        """(I - coef * (L0 - diag((n+shift)^2/r^2 + kappa^2))) x = rhs for the listed
        modes; rows 0 and N_r-1 replaced by identity (Dirichlet, L2)."""
        if self.solve == "banded":
            return self._helmholtz_banded(shift, coef, rhs, im, ik)
        N_r = self.p.N_r
        q = ((self.n[im] + shift)[:, None] ** 2 / self.r[None, :] ** 2
             + self.kappa[ik][:, None] ** 2)                  # [B, N_r]
        A = np.broadcast_to(np.eye(N_r) - coef * self.L0, (len(im), N_r, N_r)).copy()
        idx = np.arange(N_r)
        A[:, idx, idx] += coef * q
        A[:, 0, :] = 0.0
        A[:, 0, 0] = 1.0
        A[:, -1, :] = 0.0
        A[:, -1, -1] = 1.0
        return self._solve_rows(A, rhs)

    def _poisson(self, g, im, ik):
        """P phi = g at interior rows, D1 phi = 0 at the wall rows, with
        P = Q - diag(n^2/r^2 + kappa^2), Q = (D1 + 1/r) G~ (L4, R9)."""
        if self.solve == "banded":
            return self._poisson_banded(g, im, ik)
        N_r = self.p.N_r
        q = self.n[im][:, None] ** 2 / self.r[None, :] ** 2 + self.kappa[ik][:, None] ** 2
        A = np.broadcast_to(self.Q, (len(im), N_r, N_r)).copy()
        idx = np.arange(N_r)
        A[:, idx, idx] -= q
        A[:, 0, :] = self.D1[0]
        A[:, -1, :] = self.D1[-1]
        zero = (np.asarray(im) == 0) & (np.asarray(ik) == self.p.K)
        A[zero] = np.eye(N_r)                                 # O8: mode (0,0) is not projected
        phi = self._solve_rows(A, g)
        phi[zero] = 0.0
        return phi

    def substep(self, state, E, dt, modes=None, chunk=None):
        """One implicit sub-step L1..L5 from ``state`` = (ur, ut, uz, T, p) with explicit
        term E = [E_r, E_theta, E_z, (E_T)].  ``modes``: optional (im, ik) index arrays to
        restrict to sampled modes (returns arrays [N_r, B]); default all modes."""
        p = self.p
        c = p.c
        ur, ut, uz, T, pr = state
        N_r = p.N_r
        if chunk is None:
            chunk = 2048 if self.solve == "dense" else 4096
        full = modes is None
        if full:
            IM, IK = np.meshgrid(np.arange(p.M + 1), np.arange(2 * p.K + 1), indexing="ij")
            IM, IK = IM.ravel(), IK.ravel()
        else:
            IM, IK = (np.asarray(x) for x in modes)
        if self.solve == "c":
            # the C backend forms its own right-hand sides, for the listed modes only: taken before the all-mode
            # arrays below are built (they would be unused; at N_r = 512 with 5e5 modes they cost ~40 GB and minutes)
            out = [np.empty((N_r, len(IM)), self.cplx) for _ in range(5)]
            self._substep_c(state, E, dt, IM, IK, out)
            if not p.heated:
                out[3] = None
            if full:
                shp = (N_r, p.M + 1, 2 * p.K + 1)
                out = [None if o is None else o.reshape(shp) for o in out]
            return out
        r = self.r[:, None, None]
        n = self.n[None, :, None]
        # L1 right-hand sides, formed for all modes (cheap) then gathered per mode
        up, um = ur + 1j * ut, ur - 1j * ut
        Ep, Em = E[0] + 1j * E[1], E[0] - 1j * E[1]
        dp = self.d_r(pr)
        rp = up + dt * ((1 - c) * self.lap(up, +1) + Ep - (dp - n / r * pr))
        rm = um + dt * ((1 - c) * self.lap(um, -1) + Em - (dp + n / r * pr))
        rz = uz + dt * ((1 - c) * self.lap(uz, 0) + E[2] - 1j * self.kappa[None, None, :] * pr)
        rhs = [rp, rm, rz]
        if p.heated:
            rhs.append(T + dt * ((1 - c) / p.Pr * self.lap(T, 0) + E[3]))
        # Dirichlet data (R1): u_theta = Re_i, Re_o; u_r = u_z = 0; T = +1/2, -1/2
        for a in rhs:
            a[0] = 0.0
            a[-1] = 0.0
        rp[0, 0, p.K], rp[-1, 0, p.K] = 1j * p.Re_i, 1j * p.Re_o
        rm[0, 0, p.K], rm[-1, 0, p.K] = -1j * p.Re_i, -1j * p.Re_o
        if p.heated:
            rhs[3][0, 0, p.K], rhs[3][-1, 0, p.K] = 0.5, -0.5
        nB = len(IM)
        out = [np.empty((N_r, nB), self.cplx) for _ in range(5)]

        def solve_chunk(s):
            im, ik = IM[s:s + chunk], IK[s:s + chunk]
            g_ = lambda a: a[:, im, ik].T                    # [B, N_r]
            # L2 Helmholtz solves
            ups = self._helmholtz(+1, c * dt, g_(rp), im, ik)
            ums = self._helmholtz(-1, c * dt, g_(rm), im, ik)
            uzs = self._helmholtz(0, c * dt, g_(rz), im, ik)
            Tn = self._helmholtz(0, c * dt / p.Pr, g_(rhs[3]), im, ik) if p.heated else None
            # L3 recombine + divergence
            urs = (ups + ums) / 2
            uts = (ups - ums) / 2j
            nn, kk, rr = self.n[im][:, None], self.kappa[ik][:, None], self.r[None, :]
            g = self._dr_T(urs) + urs / rr + 1j * nn / rr * uts + 1j * kk * uzs
            g[:, 0] = 0.0
            g[:, -1] = 0.0
            # L4 pressure Poisson (all modes except (0,0), O8)
            phi = self._poisson(g, im, ik)
            zero = (im == 0) & (ik == p.K)
            # L5 correct + update
            gphi = self._dr_T(phi)                            # G~ phi: D1 phi with the wall rows zeroed
            gphi[:, 0] = 0.0
            gphi[:, -1] = 0.0
            urn = urs - (gphi if self.solve == "banded" else phi @ self.Gt.T)
            utn = uts - 1j * nn / rr * phi
            uzn = uzs - 1j * kk * phi
            urn[zero] = 0.0                                   # O8: u_r(0,0) := 0
            pn = g_(pr) + phi / dt
            for o, v in zip(out, (urn, utn, uzn, Tn, pn)):
                if v is not None:
                    o[:, s:s + chunk] = v.T

        starts = list(range(0, nB, chunk))
        if self.solve == "banded" and len(starts) > 1:
            with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(starts), os.cpu_count() or 1)) as ex:
                list(ex.map(solve_chunk, starts))
        else:
            for s in starts:
                solve_chunk(s)
        if not p.heated:
            out[3] = None
        if full:
            shp = (N_r, p.M + 1, 2 * p.K + 1)
            out = [None if o is None else o.reshape(shp) for o in out]
        return out

    def _substep_c(self, state, E, dt, IM, IK, out):
        """The same sub-step for the listed modes by oracle/nsc_oracle_sub.c (plain C, OpenMP over modes)."""
        import ctypes as C
        p = self.p
        if not hasattr(self, "_clib"):
            from oracle import build_c
            self._clib = C.CDLL(build_c.build())
            self._clib.orc_substep.restype = C.c_int
            P0 = self.Q.copy()
            P0[0, :] = self.D1[0]
            P0[-1, :] = self.D1[-1]
            self._P_band_c = np.ascontiguousarray(self._band_pack(P0, 12, 12))
        ptr = lambda a: C.c_void_p(0) if a is None else a.ctypes.data_as(C.c_void_p)
        keep = []

        def arr(a, dt_):
            if a is None:
                return None
            b = np.ascontiguousarray(a, dtype=dt_)
            keep.append(b)
            return b

        fields = [arr(a, np.complex128) for a in state]
        Es = [arr(a, np.complex128) for a in E] + [None] * (4 - len(E))
        tabs = [arr(a, np.float64) for a in (self.r, self.n, self.kappa, self.D1_rows, self.L0_rows)]
        s0 = arr(self.s0, np.int32)
        im, ik = arr(IM, np.int32), arr(IK, np.int32)
        rc = self._clib.orc_substep(
            C.c_int(p.N_r), C.c_int(p.M + 1), C.c_int(2 * p.K + 1), C.c_int(p.K), C.c_int(4 if p.heated else 3),
            ptr(tabs[0]), ptr(tabs[1]), ptr(tabs[2]), ptr(tabs[3]), ptr(tabs[4]), ptr(s0), ptr(self._P_band_c),
            *[ptr(a) for a in fields], *[ptr(a) for a in Es],
            C.c_double(dt), C.c_double(p.c), C.c_double(p.Pr), C.c_double(p.Re_i), C.c_double(p.Re_o),
            ptr(im), ptr(ik), C.c_int(len(im)), *[ptr(o) for o in out])
        if rc != 0:
            raise MemoryError("orc_substep failed")

    def _dr_T(self, x):
        """D1 applied along the LAST axis of x [B, N_r] (mode-major arrays of the sub-step)."""
        if self.solve == "banded":
            xt = np.ascontiguousarray(x.T)                    # [N_r, B]
            out = np.zeros(xt.shape, np.result_type(x.dtype, self.real))
            for l in range(9):
                out += self.D1_rows[:, l][:, None] * xt[self.s0 + l]
            return np.ascontiguousarray(out.T)
        return x @ self.D1.T

    # ---------------------------------------------------------------- O7 step
    def step(self, state, dt, workers=1):
        """Predictor-corrector step (R10: c = 1/2, one corrector pass).
        N0 = N(u^n); u^1 = substep(N0) (its pressure discarded); N1 = N(u^1);
        u^{n+1} = substep(c N1 + (1-c) N0), both sub-steps starting from (u^n, T^n, p^n)."""
        c = self.p.c
        nf = 4 if self.p.heated else 3
        N0 = self.nonlinear(*state[:nf], workers=workers)
        s1 = self.substep(state, N0, dt)
        N1 = self.nonlinear(*s1[:nf], workers=workers)
        return self.substep(state, [c * a + (1 - c) * b for a, b in zip(N1, N0)], dt)

    # ---------------------------------------------------------------- NEXT-1: iterated corrector
    def step_iterated(self, state, dt, tol, max_corr):
        """Predictor-corrector step with the corrector ITERATED to convergence (the reason
        the paper gives for a predictor-corrector scheme is that it allows "a variable time step size with
        dynamic control"; its ref. [6] is not available, so the stopping rule is DESIGN.md reading R16):
            u^(1) = substep(N0),   u^(k+1) = substep(c N(u^(k)) + (1-c) N0),  k = 1, 2, ...
        every sub-step starting from (u^n, T^n, p^n); stop after pass k when
            err_k = ||u^(k+1) - u^(k)||_2 / ||u^(k+1)||_2 <= tol   (all nf fields concatenated)
        or k = max_corr.  Returns (state, k, err_k).  max_corr = 1 is ``step`` (err is still reported)."""
        c = self.p.c
        nf = 4 if self.p.heated else 3
        N0 = self.nonlinear(*state[:nf])
        cur = self.substep(state, N0, dt)
        k, err = 0, float("inf")
        while k < max_corr:
            Nk = self.nonlinear(*cur[:nf])
            new = self.substep(state, [c * a + (1 - c) * b for a, b in zip(Nk, N0)], dt)
            k += 1
            err = rel_l2(cur[:nf], new[:nf])
            cur = new
            if err <= tol:
                break
        return cur, k, err

    # ---------------------------------------------------------------- NEXT-1: dynamic step-size control
    def radial_spacing(self):
        """Delta r_j = the smaller of the two spacings next to node j (one-sided at the walls)."""
        d = np.diff(self.r.astype(np.float64))
        return np.minimum(np.concatenate([[d[0]], d]), np.concatenate([d, [d[-1]]]))

    def cfl_rate(self, state):
        """Advective CFL rate lambda (1 / time) of a state, the largest over the physical grid of
            |u_r| / Delta r_j,   |u_theta| / (r_j Delta theta),   |u_z| / Delta z,
        Delta theta = 2 pi / (k_theta0 N_theta), Delta z = 2 pi / (alpha N_z) (SURVEY.md S12's rule; R17): a step
        of size dt has CFL number lambda dt.  Returns (lambda, per-component maxima [3][N_r])."""
        p = self.p
        dth = 2 * np.pi / (p.k_theta0 * p.n_theta)
        dz = 2 * np.pi / (p.alpha * p.n_z)
        mx = np.stack([np.abs(self.to_physical(f)).reshape(p.N_r, -1).max(axis=1) for f in state[:3]]).astype(np.float64)
        r = self.r.astype(np.float64)
        lam = max(float((mx[0] / self.radial_spacing()).max()), float((mx[1] / (r * dth)).max()), float((mx[2] / dz).max()))
        return lam, mx

    @staticmethod
    def dt_grid_floor(x):
        """Largest value (8 + i) / 8 * 2^e, i = 0..7, that is <= x: step sizes are kept on this geometric grid
        (ratio ~1.09) so that a controller re-uses the factored per-mode matrices (R17)."""
        m, e = np.frexp(x)                          # x = m 2^e, 0.5 <= m < 1
        return float(np.ldexp(np.floor(m * 16) / 16, e))

    @staticmethod
    def dt_grid_next(x):
        """The grid value above the grid value x."""
        m, e = np.frexp(x)
        return float(np.ldexp((np.floor(m * 16) + 1) / 16, e))

    def advance(self, state, t_end, max_steps, dt0, tol, cfl, max_corr):
        """Time integration with dynamic step-size control ("a variable time-step size with dynamic
        control"; the paper's rule is in its ref. [6], not available: DESIGN.md reading R17).  From t = 0:
            dt_cur <- grid_floor(dt0);  repeat until t = t_end or max_steps attempts:
              lambda = cfl_rate(u^n);  dt = min(dt_cur, grid_floor(cfl / lambda), t_end - t)
              (u, k, err) = step_iterated(u^n, dt, tol, max_corr)
              err <= tol : accept, t += dt, dt_cur <- grid_next(dt) if k <= 2, err <= tol / 2 and dt == dt_cur, else kept
              err >  tol : reject (state unchanged), dt_cur <- grid_floor(dt / 2)
        Returns (state, t, log) with log = list of (dt, k, err, accepted)."""
        t, log = 0.0, []
        dt_cur = self.dt_grid_floor(dt0)
        while t < t_end and len(log) < max_steps:
            lam, _ = self.cfl_rate(state)
            dt = dt_cur
            if lam > 0.0:
                dt = min(dt, self.dt_grid_floor(cfl / lam))
            last = t_end - t <= dt
            if last:
                dt = t_end - t
            new, k, err = self.step_iterated(state, dt, tol, max_corr)
            ok = err <= tol
            log.append((dt, k, err, ok))
            if ok:
                state = new
                t = t_end if last else t + dt
                if k <= 2 and err <= 0.5 * tol and dt == dt_cur:
                    dt_cur = self.dt_grid_next(dt_cur)
            else:
                dt_cur = self.dt_grid_floor(dt / 2)
        return state, t, log

    # ---------------------------------------------------------------- NEXT-4: restart on another resolution
    def regrid_matrix(self, src):
        """[N_r, N_r_src] matrix of the degree-8 Lagrange interpolation from the radial nodes of oracle ``src`` to
        the nodes of this one (R18): row j holds the nine basis values l_q(r_j) = prod_{p != q} (r_j - x_p) / (x_q - x_p)
        on the source nodes x = r_src[s..s+8], s = clamp(c - 4, 0, N_src - 9), c = the source node nearest to r_j
        (the lower one on a tie).  Extended precision, rounded once."""
        xs = src.r.astype(LD)
        W = np.zeros((self.p.N_r, src.p.N_r), LD)
        for j, rj in enumerate(self.r.astype(LD)):
            c = int(np.argmin(np.abs(src.r.astype(np.float64) - np.float64(rj))))
            s = min(max(c - 4, 0), src.p.N_r - 9)
            x = xs[s:s + 9]
            for q in range(9):
                num = den = LD(1)
                for pp in range(9):
                    if pp != q:
                        num = num * (rj - x[pp])
                        den = den * (x[q] - x[pp])
                W[j, s + q] = num / den
        return W.astype(self.real)

    def regrid(self, state, src):
        """State of oracle ``src`` carried onto this oracle's radial grid and mode set ("At every
        restart, the spatial resolution can be changed using an automated interpolation and mode padding
        functionality"; R18): radial interpolation by ``regrid_matrix``; modes the source does not hold are zero,
        modes this oracle does not hold are dropped.  T is dropped if this oracle has no temperature."""
        p, q = self.p, src.p
        assert (p.eta, p.alpha, p.k_theta0) == (q.eta, q.alpha, q.k_theta0) and (q.heated or not p.heated)
        W = self.regrid_matrix(src)
        Mc, Kc = min(p.M, q.M), min(p.K, q.K)
        out = []
        for i, f in enumerate(state):
            if f is None or (i == 3 and not p.heated):
                out.append(None)
                continue
            g = self.zeros()
            part = f[:, :Mc + 1, q.K - Kc:q.K + Kc + 1]
            g[:, :Mc + 1, p.K - Kc:p.K + Kc + 1] = np.einsum("jl,lmk->jmk", W, part)
            out.append(g)
        return out

    # ---------------------------------------------------------------- NEXT-3: wave speed
    def wave_speed(self, state, field, j, m, k, dt, n_steps):
        """Angular phase speed of one Fourier coefficient f^(r_j; m, k) ~ e^{i (n theta - omega t)} over n_steps
        plain steps of size dt (the CI validation compares "the wave speed of a simulated wavy
        vortex flow" with an experiment): omega / n, n = m k_theta0 >= 1, with
        omega = - sum_i arg(f_{i+1} conj f_i) / (n_steps dt)  (phase increments per step, each in (-pi, pi]).
        Returns (speed, state after the steps)."""
        n = m * self.p.k_theta0
        kk = k + self.p.K
        f0 = complex(state[field][j, m, kk])
        dphi = 0.0
        for _ in range(n_steps):
            state = self.step(state, dt)
            f1 = complex(state[field][j, m, kk])
            dphi += float(np.angle(f1 * np.conj(f0)))
            f0 = f1
        return -dphi / (n_steps * dt) / n, state

    # ---------------------------------------------------------------- NEXT-3: diagnostics
    def nusselt(self, state):
        """Wall diagnostics of PAPER.md:100-108 (Fig. 3a plots Nu_i): transfer at a wall normalised by that of
        the basic state at the same parameters, from the mean mode (0,0) only (theta, z averages).
          heat  : Nu = d_r T^(0,0) / d_r T_b,        T_b = ln(r / r_o) / ln(eta) - 1/2  =>  d_r T_b = 1 / (r ln eta)
          torque: Nu_w = [r^3 d_r(u_theta / r)] / [r^3 d_r(V / r)],  V = A r + B / r   =>  r^3 d_r(V / r) = -2 B
        (u_r = 0 at the walls, so the convective part of both fluxes vanishes there).  d_r = the 9-point D1 row
        of the wall node.  Returns (Nu_i, Nu_o, Nu_w_i, Nu_w_o); the heat entries are nan without temperature."""
        p = self.p
        ur, ut, uz, T, pr = state
        r = self.r
        K = p.K
        eta = p.eta
        B = eta * (p.Re_i - eta * p.Re_o) / ((1 - eta) * (1 - eta ** 2))
        out = []
        for j in (0, p.N_r - 1):
            if p.heated:
                dT = float((self.D1[j] @ T[:, 0, K]).real)
                out.append(dT * r[j] * np.log(eta))
            else:
                out.append(float("nan"))
        for j in (0, p.N_r - 1):
            v = ut[:, 0, K].real
            dw = (self.D1[j] @ v) / r[j] - v[j] / r[j] ** 2
            out.append(float(r[j] ** 3 * dw / (-2.0 * B)) if B != 0.0 else float("nan"))
        return tuple(out)

    def probe(self, f, j, theta, z):
        """Value of the physical field of spectral coefficients ``f`` at radial node j and the point (theta, z)
        (Fig. 3b: u_theta at a fixed probe location): the series of O3 at an arbitrary point,
        Re sum_k f(0,k) e^{i kappa z} + 2 Re sum_{m>=1} sum_k f(m,k) e^{i (n theta + kappa z)}."""
        ph = np.exp(1j * (self.n[:, None] * theta + self.kappa[None, :] * z))
        t = f[j] * ph
        return float(t[0].sum().real + 2.0 * t[1:].sum().real)

    # ---------------------------------------------------------------- basic states
    def zeros(self):
        p = self.p
        return np.zeros((p.N_r, p.M + 1, 2 * p.K + 1), self.cplx)

    def base_state_discrete(self):
        """Discrete basic state: u_theta(r), T(r) (and the buoyancy-driven
        axial flow w(r), R11) solving the *discrete* steady equations in mode (0,0)."""
        p = self.p
        r = self.r

        def solve(L, bi, bo, rhs=None):
            A = L.copy()
            A[0] = 0
            A[0, 0] = 1
            A[-1] = 0
            A[-1, -1] = 1
            b = np.zeros(p.N_r) if rhs is None else rhs.copy()
            b[0], b[-1] = bi, bo
            return np.linalg.solve(A.astype(np.float64), b.astype(np.float64)).astype(self.real)

        ur, ut, uz = self.zeros(), self.zeros(), self.zeros()
        ut[:, 0, p.K] = solve(self.L0 - np.diag(1 / r ** 2), p.Re_i, p.Re_o)
        T = None
        if p.heated:
            T = self.zeros()
            T[:, 0, p.K] = solve(self.L0, 0.5, -0.5)
            uz[:, 0, p.K] = solve(self.L0, 0.0, 0.0, -(p.Ra / p.Pr) * T[:, 0, p.K].real)
        return [ur, ut, uz, T, self.zeros()]


def rel_l2(a_list, b_list):
    """R14 parity norm: ||a - b||_2 / ||b||_2 over the concatenation of all fields."""
    num = sum(np.linalg.norm((a - b).ravel()) ** 2 for a, b in zip(a_list, b_list) if b is not None)
    den = sum(np.linalg.norm(b.ravel()) ** 2 for b in b_list if b is not None)
    return float(np.sqrt(num / den))


def rel_l2_pert(a_list, b_list, K, mean_index=None):
    """The same norm with the mean mode (0,0) left out of numerator and denominator (SURVEY.md S14:
    "also report the same norm with mode (0,0) excluded"): the base flow sits in that mode and is
    10^2..10^4 times larger than the perturbation, so an error confined to the perturbation modes
    would be discounted by that factor in R14.  Arrays are [N_r, M+1, 2K+1], or [N_r, B] sampled-mode
    arrays with ``mean_index`` = the positions (along B) of mode (0,0), if any."""
    num = den = 0.0
    for a, b in zip(a_list, b_list):
        if b is None:
            continue
        d = np.abs(a - b) ** 2
        e = np.abs(b) ** 2
        if b.ndim == 3:
            d[:, 0, K] = 0.0
            e[:, 0, K] = 0.0
        elif mean_index is not None:
            d[:, mean_index] = 0.0
            e[:, mean_index] = 0.0
        num += float(d.sum())
        den += float(e.sum())
    return float(np.sqrt(num / den))
