"""Pin T5: the oracle's implicit sub-step (O5, O6; BASELINE.json north_star (b)).

* Helmholtz: a manufactured polynomial (degree <= 8, so the FD operators are exact) is
  recovered from a right-hand side built with *analytic* derivatives, for u_+, u_-, u_z, T;
* Poisson / projection: the result is discretely divergence-free to round-off, the
  projection is idempotent, and a field that is already divergence-free is left alone;
* the u_+- coupling: a sub-step with c*dt -> 0 reduces to explicit Euler written in
  (u_r, u_theta) components with the textbook vector Laplacian in cylindrical coordinates.
"""
import numpy as np
import pytest
from oracle.nsc_oracle import Params, Oracle
from paper_1908_00587_b200 import synth
from helpers import oracle_of


def scaled_div(o, ur, ut, uz):
    d = np.abs(o.divergence(ur, ut, uz))
    r = o.r[:, None, None]
    sc = (np.einsum("jl,lmk->jmk", np.abs(o.D1), np.abs(ur)) + np.abs(ur) / r
          + np.abs(o.n)[None, :, None] / r * np.abs(ut) + np.abs(o.kappa)[None, None, :] * np.abs(uz))
    sc = np.maximum(sc, 1e-12 * sc.max())
    return (d / sc)[1:-1].max()


@pytest.mark.parametrize("grid", [0, 1])
def test_helmholtz_manufactured_polynomial(grid):
    o = Oracle(Params(N_r=20, M=2, K=2, eta=0.5, alpha=2.5, k_theta0=3, Re_i=0.0, Re_o=0.0,
                      Ra=1.0, Pr=0.7, grid=grid))
    p, r = o.p, o.r
    x = r - r[0]
    v = (x * (1 - x)) * (1 + 0.5 * x - 0.3 * x ** 2)       # vanishes at both walls, degree 4
    v1 = (1 - 2 * x) * (1 + 0.5 * x - 0.3 * x ** 2) + (x - x * x) * (0.5 - 0.6 * x)
    v2 = -2 * (1 + 0.5 * x - 0.3 * x ** 2) + 2 * (1 - 2 * x) * (0.5 - 0.6 * x) + (x - x * x) * (-0.6)
    im, ik = np.array([1, 2, 0, 2]), np.array([0, 3, 4, 2])
    for shift, coef in ((+1, 0.37), (-1, 0.37), (0, 0.37), (0, 0.37 / 0.7)):
        q = ((o.n[im] + shift)[:, None] ** 2 / r[None, :] ** 2 + o.kappa[ik][:, None] ** 2)
        rhs = v[None, :] - coef * (v2 + v1 / r)[None, :] + coef * q * v[None, :]
        rhs = rhs * (1 + 2j)
        rhs[:, 0] = 0
        rhs[:, -1] = 0
        xs = o._helmholtz(shift, coef, rhs, im, ik)
        np.testing.assert_allclose(xs, np.broadcast_to(v * (1 + 2j), xs.shape), atol=2e-13)


@pytest.mark.parametrize("cfgi,N_r", [(0, 32), (1, 24), (2, 24)])
def test_projection_divergence_free_and_idempotent(cfgi, N_r):
    cfg = synth.scaled_config(cfgi, N_r=N_r, M=4, K=4)
    o = oracle_of(cfg)
    nf = 4 if o.p.heated else 3
    st = synth.make_state(cfg, o.r)
    assert scaled_div(o, *st[:3]) < 1e-10                    # the generator is divergence-free
    rng = np.random.default_rng(1)
    E = [1e3 * (rng.standard_normal(st[0].shape) + 1j * rng.standard_normal(st[0].shape)) for _ in range(nf)]
    s1 = o.substep(st, E, cfg["dt"])
    assert scaled_div(o, *s1[:3]) < 1e-10
    assert np.abs(s1[0][[0, -1]]).max() < 1e-12 * np.abs(s1[0]).max()   # u_r = 0 at the walls
    # idempotent: projecting the projected field (zero forcing, p carried) changes nothing
    # measurable in the divergence, and phi of a divergence-free u* is round-off
    im, ik = np.array([1, 2, 0]), np.array([2, 5, 6])
    g = o.divergence(*s1[:3])[:, im, ik].T.copy()
    g[:, 0] = 0
    g[:, -1] = 0
    phi = o._poisson(g, im, ik)
    gscale = np.abs(o.divergence(s1[0], 0 * s1[1], 0 * s1[2])).max()
    assert np.abs(phi).max() < 1e-9 * gscale


def test_substep_reduces_to_explicit_euler_in_components():
    """c = 0 makes the Helmholtz operators the identity: u* = u + dt (lap u + E - grad p) with
    the cylindrical vector Laplacian (lap u)_r = L_s u_r - u_r/r^2 - (2 i n / r^2) u_theta,
    (lap u)_theta = L_s u_theta - u_theta/r^2 + (2 i n / r^2) u_r  (textbook form)."""
    cfg = synth.scaled_config(1, N_r=20, M=3, K=3)
    o = Oracle(Params(**{k: cfg[k] for k in synth.PHYS_KEYS}, c=0.0))
    st = synth.make_state(cfg, o.r)
    rng = np.random.default_rng(4)
    st[4] = rng.standard_normal(st[0].shape) + 1j * rng.standard_normal(st[0].shape)
    E = [rng.standard_normal(st[0].shape) + 0j for _ in range(3)]
    dt = 1e-4
    # reproduce u* (before projection) by hand and project with the oracle's own L3-L5
    ur, ut, uz, _, pr = st
    r = o.r[:, None, None]
    n = o.n[None, :, None]
    Ls = lambda f: o.lap(f, 0)
    lr = Ls(ur) - ur / r ** 2 - 2j * n / r ** 2 * ut
    lt = Ls(ut) - ut / r ** 2 + 2j * n / r ** 2 * ur
    urs = ur + dt * (lr + E[0] - o.d_r(pr))
    uts = ut + dt * (lt + E[1] - 1j * n / r * pr)
    # compare through u_+- of the oracle's right-hand sides
    up = ur + 1j * ut
    rp = up + dt * (o.lap(up, +1) + (E[0] + 1j * E[1]) - (o.d_r(pr) - n / r * pr))
    np.testing.assert_allclose(rp[1:-1], (urs + 1j * uts)[1:-1], rtol=0, atol=1e-9 * np.abs(rp).max())
    um = ur - 1j * ut
    rm = um + dt * (o.lap(um, -1) + (E[0] - 1j * E[1]) - (o.d_r(pr) + n / r * pr))
    np.testing.assert_allclose(rm[1:-1], (urs - 1j * uts)[1:-1], rtol=0, atol=1e-9 * np.abs(rm).max())
    out = o.substep(st, E, dt)
    assert scaled_div(o, *out[:3]) < 1e-10


def test_modes_subset_equals_full():
    cfg = synth.scaled_config(2, N_r=16, M=3, K=3)
    o = oracle_of(cfg)
    st = synth.make_state(cfg, o.r)
    E = o.nonlinear(*st[:4])
    full = o.substep(st, E, cfg["dt"])
    im, ik = np.array([0, 0, 2, 3]), np.array([3, 4, 0, 6])
    sub = o.substep(st, E, cfg["dt"], modes=(im, ik))
    for a, b in zip(full, sub):
        np.testing.assert_allclose(a[:, im, ik], b, rtol=1e-13, atol=0)


# ------------------------------------------------------------------ the thermal diffusivity is 1 / Pr
def test_temperature_substep_reduces_to_explicit_euler_with_diffusivity_one_over_Pr():
    """c = 0: T_new = T + dt [ (1/Pr)(T'' + T'/r - (n^2/r^2 + kappa^2) T) + E_T ] at interior nodes, written with
    ANALYTIC derivatives of a polynomial T (degree 6: the 9-point rows are exact), Pr = 0.7 != 1.  Pins the factor
    (1 - c)/Pr of L1 (temperature equation; d_t T = ... + (1/Pr) lap T):
    Pr in place of 1/Pr, or a dropped factor, changes the result by O(dt lap T)."""
    Pr = 0.7
    o = Oracle(Params(N_r=24, M=3, K=3, eta=0.5, alpha=2.0, k_theta0=2, Re_i=0.0, Re_o=0.0, Ra=50.0, Pr=Pr, c=0.0))
    r = o.r
    x = r - r[0]
    prof = x * (1 - x) * (1.0 + 0.4 * x - 0.7 * x ** 2 + 0.2 * x ** 3) * (1 + 0.5 * x)       # degree 6, zero at the walls
    c = np.polynomial.polynomial.polyfromroots([0.0, 1.0]) * -1.0                              # x (1 - x)
    c = np.polynomial.polynomial.polymul(c, [1.0, 0.4, -0.7, 0.2])
    c = np.polynomial.polynomial.polymul(c, [1.0, 0.5])
    np.testing.assert_allclose(np.polynomial.polynomial.polyval(x, c), prof, atol=1e-14)
    d1 = np.polynomial.polynomial.polyval(x, np.polynomial.polynomial.polyder(c))
    d2 = np.polynomial.polynomial.polyval(x, np.polynomial.polynomial.polyder(c, 2))
    st = [o.zeros() for _ in range(5)]
    amp = {(1, 4): 1.0 + 0.5j, (2, 1): -0.3 + 2.0j, (0, 5): 0.7 - 0.2j}
    for (m, kk), a in amp.items():
        st[3][:, m, kk] = a * prof
    rng = np.random.default_rng(5)
    E = [o.zeros(), o.zeros(), o.zeros(), rng.standard_normal(st[0].shape) + 1j * rng.standard_normal(st[0].shape)]
    dt = 1e-3
    out = o.substep(st, E, dt)
    for (m, kk), a in amp.items():
        q = o.n[m] ** 2 / r ** 2 + o.kappa[kk] ** 2
        want = a * prof + dt * ((1.0 / Pr) * a * (d2 + d1 / r - q * prof) + E[3][:, m, kk])
        got = out[3][:, m, kk]
        scale = np.abs(dt * a * (d2 + d1 / r - q * prof)).max()
        assert scale > 1e-3                                   # the diffusion term is what is being tested
        np.testing.assert_allclose(got[1:-1], want[1:-1], rtol=0, atol=1e-10 * scale)
        wrong = a * prof + dt * (Pr * a * (d2 + d1 / r - q * prof) + E[3][:, m, kk])
        assert np.abs(got[1:-1] - wrong[1:-1]).max() > 0.1 * scale


def _cheb_dd(N):
    x = np.cos(np.pi * np.arange(N + 1) / N)
    cc = np.ones(N + 1)
    cc[0] = cc[-1] = 2
    cc *= (-1) ** np.arange(N + 1)
    X = np.tile(x, (N + 1, 1)).T
    D = np.outer(cc, 1 / cc) / (X - X.T + np.eye(N + 1))
    D -= np.diag(D.sum(1))
    return D, x


@pytest.mark.parametrize("Pr", [0.7, 3.0])
def test_conduction_mode_decays_at_the_diffusion_eigenvalue_over_Pr(Pr):
    """A temperature perturbation in one axial mode with the fluid at rest obeys d_t T = (1/Pr)(DD* - kappa^2) T,
    T = 0 at the walls, so after the transients it decays at lambda_1 / Pr with lambda_1 the leading
    eigenvalue of DD* - kappa^2 = d^2/dr^2 + (1/r) d/dr - kappa^2, computed here by Chebyshev collocation (a
    discretisation independent of the oracle's).  The implicit sub-step with no explicit term is the
    Crank-Nicolson integrator of that equation: pins both (1 - c)/Pr in L1 and c dt/Pr in L2."""
    eta, kap = 0.5, 3.0
    D, xc = _cheb_dd(40)
    rc = eta / (1 - eta) + 0.5 * (1 - xc)
    D = D / (-0.5)
    A = D @ D + np.diag(1 / rc) @ D - kap ** 2 * np.eye(41)
    lam = np.sort(np.linalg.eigvals(A[1:-1, 1:-1]).real)[::-1]
    assert lam[0] == pytest.approx(-(np.pi ** 2 + kap ** 2), rel=2e-2)     # close to the planar value
    o = Oracle(Params(N_r=32, M=1, K=1, eta=eta, alpha=kap, k_theta0=1, Re_i=0.0, Re_o=0.0, Ra=1.0, Pr=Pr))
    st = [o.zeros() for _ in range(5)]
    x = o.r - o.r[0]
    st[3][:, 0, 2] = x * (1 - x) * (1 + x)
    st[3][:, 0, 0] = np.conj(st[3][:, 0, 2])
    E = [o.zeros() for _ in range(4)]
    dt = 2e-3 * Pr
    t0, t1 = 0.3 * Pr, 0.4 * Pr
    n0, n1 = round(t0 / dt), round(t1 / dt)
    amp = {}
    for i in range(1, n1 + 1):
        st = o.substep(st, E, dt)
        if i in (n0, n1):
            amp[i] = np.linalg.norm(st[3][:, 0, 2])
    rate = np.log(amp[n1] / amp[n0]) / ((n1 - n0) * dt)
    assert rate == pytest.approx(lam[0] / Pr, rel=1e-3)
    assert abs(rate - lam[0] * Pr) > 0.3 * abs(rate)          # Pr in place of 1 / Pr would be far off
