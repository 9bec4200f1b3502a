"""Pins T3, T6, T7, T8: the oracle's full predictor-corrector step (O6-O8).

* T3  fixed points: the discrete circular Couette profile (and, heated, the conductive
      temperature with its buoyancy-driven axial flow) is unchanged by ``step`` to round-off
      for any dt, and converges to the closed forms A r + B / r, T_b(r), w_b(r)
      ("the basic state depends on r only").
* T6  linear stability: the growth rate of a tiny axisymmetric perturbation, measured through
      the full nonlinear step, approaches the leading eigenvalue of the classical Taylor
      problem computed here by an independent Chebyshev-collocation eigen-solve
      (BASELINE.json north_star: "growth rate ... must agree with a linear-stability
      eigenvalue computed by brute force on a tiny grid").
* T7  the same growth rate equals ln(mu)/dt for the dominant eigenvalue mu of the one-step
      propagator assembled column by column from the oracle itself on a tiny grid.
* T8  temporal order 2 by Richardson extrapolation; divergence stays at round-off.
"""
import numpy as np
import pytest
import scipy.linalg as sla
from oracle.nsc_oracle import Params, Oracle, rel_l2
from paper_1908_00587_b200 import synth
from helpers import oracle_of
from test_oracle_linear import scaled_div


# ------------------------------------------------------------------ T3 fixed points
@pytest.mark.parametrize("dt", [1e-3, 0.05])
def test_couette_is_a_fixed_point(dt):
    o = Oracle(Params(N_r=32, M=4, K=4, eta=0.5, alpha=3.0, k_theta0=1, Re_i=100.0, Re_o=-30.0))
    b = o.base_state_discrete()
    b1 = o.step(b, dt)
    assert rel_l2(b1[:3], b[:3]) < 5e-14
    assert np.abs(b1[0]).max() == 0.0 or np.abs(b1[0]).max() < 1e-12
    # every mode other than (0,0) stays exactly empty
    mask = np.ones(b1[1].shape, bool)
    mask[:, 0, o.p.K] = False
    assert np.abs(b1[1][mask]).max() < 1e-12


def test_discrete_couette_converges_to_closed_form():
    errs = []
    for N_r in (16, 32, 64):
        o = Oracle(Params(N_r=N_r, M=1, K=1, eta=0.5, alpha=3.0, k_theta0=1, Re_i=100.0, Re_o=0.0))
        v = o.base_state_discrete()[1][:, 0, 1].real
        errs.append(np.abs(v - synth.couette(o.r, 0.5, 100.0, 0.0)).max() / 100.0)
    assert errs[0] > errs[1] > errs[2] or errs[2] < 1e-12
    assert errs[1] < 1e-8 and errs[2] < 1e-11


def test_heated_base_state_fixed_point_and_closed_forms():
    cfg = synth.scaled_config(2, N_r=48, M=3, K=3)           # cfg 3 physics (Ra=1e6, Pr=0.7)
    o = oracle_of(cfg)
    b = o.base_state_discrete()
    for dt in (2e-6, 1e-4):
        b1 = o.step(b, dt)
        assert rel_l2(b1[:4], b[:4]) < 1e-12
    K = o.p.K
    Tb = synth.conductive_T(o.r, cfg["eta"])
    wb = synth.axial_base_flow(o.r, cfg["eta"], cfg["Ra"], cfg["Pr"])
    assert np.abs(b[3][:, 0, K].real - Tb).max() < 1e-9
    assert np.abs(b[2][:, 0, K].real - wb).max() < 1e-8 * np.abs(wb).max()
    # Nu_i = 1 for the conductive state: -dT/dr at r_i over the
    # conductive value 1 / (r_i ln(1/eta)) ... using the oracle's own D1 on the closed form
    dT = o.D1 @ Tb
    r_i = o.r[0]
    assert abs(dT[0] * r_i * np.log(cfg["eta"]) - 1.0) < 1e-7


# ------------------------------------------------------------------ T6 Taylor eigenvalue
def _cheb(N):
    x = np.cos(np.pi * np.arange(N + 1) / N)
    c = np.ones(N + 1)
    c[0] = c[-1] = 2
    c *= (-1) ** np.arange(N + 1)
    X = np.tile(x, (N + 1, 1)).T
    dX = X - X.T
    D = np.outer(c, 1 / c) / (dX + np.eye(N + 1))
    D -= np.diag(D.sum(1))
    return D, x


def taylor_eigenvalue(eta, Re_i, Re_o, kap, N=40):
    """sigma (DD* - k^2) u = (DD* - k^2)^2 u - 2 k^2 (V/r) v,  sigma v = (DD* - k^2) v - 2 A u,
    u = Du = v = 0 at both walls (classical axisymmetric Taylor problem, pressure and u_z
    eliminated), Chebyshev collocation: a discretisation independent of the oracle's."""
    D, x = _cheb(N)
    r = eta / (1 - eta) + 0.5 * (1 - x)
    D = D / (-0.5)
    n = N + 1
    I = np.eye(n)
    A = (Re_o - eta * Re_i) / (1 + eta)
    B = eta * (Re_i - eta * Re_o) / ((1 - eta) * (1 - eta ** 2))
    V = A * r + B / r
    Mop = D @ (D + np.diag(1 / r)) - kap ** 2 * I
    LA = np.zeros((2 * n, 2 * n))
    LB = np.zeros((2 * n, 2 * n))
    LA[:n, :n] = Mop @ Mop
    LA[:n, n:] = -2 * kap ** 2 * np.diag(V / r)
    LB[:n, :n] = Mop
    LA[n:, :n] = -2 * A * I
    LA[n:, n:] = Mop
    LB[n:, n:] = I
    for row, vec in ((0, I[0]), (N, I[N]), (1, D[0]), (N - 1, D[N])):
        LA[row, :] = 0
        LB[row, :] = 0
        LA[row, :n] = vec
    for row, vec in ((n, I[0]), (n + N, I[N])):
        LA[row, :] = 0
        LB[row, :] = 0
        LA[row, n:] = vec
    w = sla.eigvals(LA, LB)
    w = w[np.isfinite(w)]
    w = w[np.abs(w) < 1e6]
    return w[np.argsort(-w.real)][0]


def test_taylor_eigenvalue_reproduces_textbook_threshold():
    # eta = 0.5, outer cylinder at rest: Re_c = 68.19 at kappa = 3.16 (textbook value)
    assert taylor_eigenvalue(0.5, 68.19, 0.0, 3.16).real == pytest.approx(0.0, abs=2e-2)
    assert taylor_eigenvalue(0.5, 60.0, 0.0, 3.16).real < 0 < taylor_eigenvalue(0.5, 75.0, 0.0, 3.16).real


def _perturbed_state(o, eps=1e-6):
    """Couette flow + eps * (divergence-free axisymmetric mode (0, +-1))."""
    p = o.p
    st = o.base_state_discrete()
    x = o.r - o.r[0]
    ur = (x * (1 - x)) ** 2 * (1 + 0.3 * x) * eps * 100.0
    ut = x * (1 - x) * (0.7 - 0.2 * x) * eps * 100.0
    kap = p.alpha
    uz = -(o.D1 @ ur + ur / o.r) / (1j * kap)
    uz[0] = uz[-1] = 0
    K = p.K
    st[0][:, 0, K + 1] = ur
    st[0][:, 0, K - 1] = np.conj(ur)
    st[1][:, 0, K + 1] += ut
    st[1][:, 0, K - 1] += np.conj(ut)
    st[2][:, 0, K + 1] = uz
    st[2][:, 0, K - 1] = np.conj(uz)
    return st


def _growth_rate(N_r, dt, t0=0.5, t1=0.6, eps=1e-6):
    o = Oracle(Params(N_r=N_r, M=1, K=1, eta=0.5, alpha=3.0, k_theta0=1, Re_i=100.0, Re_o=0.0))
    st = _perturbed_state(o, eps)
    amp = {}
    n0, n1 = int(round(t0 / dt)), int(round(t1 / dt))
    for it in range(1, n1 + 1):
        st = o.step(st, dt)
        if it in (n0, n1):
            amp[it] = np.linalg.norm(st[0][:, 0, 2])
    return np.log(amp[n1] / amp[n0]) / ((n1 - n0) * dt)


def test_growth_rate_matches_taylor_eigenvalue_second_order_in_dt():
    sigma = taylor_eigenvalue(0.5, 100.0, 0.0, 3.0).real
    assert sigma == pytest.approx(12.3078, abs=2e-3)          # SURVEY T6 probe value
    e2 = _growth_rate(32, 2e-3) - sigma
    e1 = _growth_rate(32, 1e-3) - sigma
    assert abs(e1) < 6e-3                                      # ~3.6e-3 expected
    assert 2.5 < e2 / e1 < 8.0                                 # second order in dt (ratio -> 4)


# ------------------------------------------------------------------ T7 propagator
def test_propagator_eigenvalue_equals_measured_growth():
    """Tiny grid: the one-step map of a perturbation in mode (0,1), assembled column by column
    from ``step`` by central differences (exactly linear up to O(eps^2)); its dominant
    eigenvalue gives the asymptotic growth rate ln(mu)/dt that a long run measures while the
    perturbation is still small."""
    N_r, dt = 16, 2e-3
    o = Oracle(Params(N_r=N_r, M=1, K=1, eta=0.5, alpha=3.0, k_theta0=1, Re_i=100.0, Re_o=0.0))
    base = o.base_state_discrete()
    K = 1
    eps = 1e-4

    def apply(vec):
        """vec = (ur, ut, uz, p)[N_r] complex in mode (0,+1) (mirrored to (0,-1))."""
        out = []
        for sgn in (+1, -1):
            st = [a.copy() for a in base[:3]] + [None, base[4].copy()]
            for f, i in ((0, 0), (1, 1), (2, 2), (4, 3)):
                v = vec[i * N_r:(i + 1) * N_r] * (eps * sgn)
                st[f][:, 0, K + 1] += v
                st[f][:, 0, K - 1] += np.conj(v)
            s1 = o.step(st, dt)
            out.append(np.concatenate([s1[f][:, 0, K + 1] for f in (0, 1, 2, 4)]))
        return (out[0] - out[1]) / (2 * eps)

    n = 4 * N_r
    # the perturbation keeps the symmetry (u_r, u_theta, p real; u_z imaginary) for kappa real:
    # assemble the real map on that subspace
    phase = np.concatenate([np.ones(2 * N_r), 1j * np.ones(N_r), np.ones(N_r)])
    P = np.zeros((n, n))
    for c in range(n):
        e = np.zeros(n, complex)
        e[c] = phase[c]
        P[:, c] = (apply(e) / phase).real
    mu = np.linalg.eigvals(P)
    mu = mu[np.argmax(np.abs(mu))]
    assert abs(mu.imag) < 1e-6
    sig_prop = np.log(mu.real) / dt
    sig_run = _growth_rate(N_r, dt, t0=0.8, t1=1.0, eps=1e-11)
    assert sig_run == pytest.approx(sig_prop, abs=1e-4)


# ------------------------------------------------------------------ T8 temporal order
def test_second_order_in_time_and_divergence_free():
    cfg = synth.scaled_config(0, N_r=24, M=4, K=4)
    cfg["amp"] = 5e-2                                          # make the nonlinear term matter
    o = oracle_of(cfg, dft="fft")
    st0 = synth.make_state(cfg, o.r)
    # warm the pressure up with small steps so that p is consistent (p0 = 0 is a cold start)
    for _ in range(40):
        st0 = o.step(st0, 2.5e-5)
    sols = []
    for dt in (5e-4, 2.5e-4, 1.25e-4):                       # asymptotic range (coarser dt: CN pre-asymptotic)
        st = [None if a is None else a.copy() for a in st0]
        for _ in range(int(round(8e-3 / dt))):
            st = o.step(st, dt)
        sols.append(st)
        assert scaled_div(o, *st[:3]) < 1e-10
    num = np.sqrt(sum(np.linalg.norm(a - b) ** 2 for a, b in zip(sols[0][:3], sols[1][:3])))
    den = np.sqrt(sum(np.linalg.norm(a - b) ** 2 for a, b in zip(sols[1][:3], sols[2][:3])))
    assert 3.0 < num / den < 5.5


def test_cfg1_twenty_steps_stable_and_divergence_free():
    cfg = synth.config(0)
    o = oracle_of(cfg, dft="fft")
    st = synth.make_state(cfg, o.r)
    e0 = np.linalg.norm(st[0])
    for _ in range(20):
        st = o.step(st, cfg["dt"])
    assert scaled_div(o, *st[:3]) < 1e-11
    assert 0.5 < np.linalg.norm(st[0]) / e0 < 2.0


# ---------------------------------------------------------------- NEXT-1: iterated corrector (R16)
def _small_state(seed_cfg=0, N_r=16, M=4, K=4, amp=None):
    from paper_1908_00587_b200 import synth
    from helpers import oracle_of
    cfg = synth.scaled_config(seed_cfg, N_r=N_r, M=M, K=K)
    if amp is not None:
        cfg["amp"] = amp
    o = oracle_of(cfg, dft="fft")
    return cfg, o, synth.make_state(cfg, o.r)


def test_iterated_corrector_one_pass_is_the_plain_step():
    cfg, o, st = _small_state()
    a = o.step(st, cfg["dt"])
    b, k, err = o.step_iterated(st, cfg["dt"], tol=0.0, max_corr=1)
    assert k == 1 and np.isfinite(err)
    for x, y in zip(a, b):
        if x is not None:
            np.testing.assert_array_equal(x, y)


def test_iterated_corrector_converges_to_its_fixed_point():
    """The limit of the iteration solves u = substep(c N(u) + (1-c) N0): the residual of that equation
    at the returned state is of the order of the last increment, the increments contract geometrically,
    and a tighter tolerance costs more passes."""
    import numpy as np
    from oracle.nsc_oracle import rel_l2
    cfg, o, st = _small_state(amp=5e-2)
    dt = 4 * cfg["dt"]
    errs = []
    for mc in (1, 2, 3, 4):
        _, k, e = o.step_iterated(st, dt, tol=0.0, max_corr=mc)
        assert k == mc
        errs.append(e)
    assert errs[1] < 0.5 * errs[0] and errs[2] < 0.5 * errs[1] and errs[3] < 0.5 * errs[2]
    out, k, e = o.step_iterated(st, dt, tol=1e-10, max_corr=50)
    assert e <= 1e-10 and k < 50
    _, k_loose, _ = o.step_iterated(st, dt, tol=1e-6, max_corr=50)
    assert k_loose < k
    # fixed-point residual
    c = o.p.c
    N0 = o.nonlinear(*st[:3])
    Nk = o.nonlinear(*out[:3])
    again = o.substep(st, [c * a + (1 - c) * b for a, b in zip(Nk, N0)], dt)
    assert rel_l2(again[:3], out[:3]) <= 1e-9


def test_iterated_corrector_leaves_couette_flow_alone():
    from paper_1908_00587_b200 import synth
    from helpers import oracle_of
    from oracle.nsc_oracle import rel_l2
    cfg = synth.scaled_config(0, N_r=24, M=4, K=4)
    o = oracle_of(cfg, dft="fft")
    base = o.base_state_discrete()
    out, k, err = o.step_iterated(base, 1e-2, tol=1e-12, max_corr=5)
    assert k == 1 and err <= 1e-12
    assert rel_l2(out[:3], base[:3]) <= 1e-13


# ---------------------------------------------------------------- NEXT-3: diagnostics
def test_nusselt_numbers_are_one_in_the_basic_state():
    """Nu_i is normalised by the basic state, so it is 1 there -- at both walls, for the heat
    flux and for the torque, up to the truncation error of the discrete profiles (falls with N_r)."""
    from paper_1908_00587_b200 import synth
    from helpers import oracle_of
    errs = []
    for N_r in (24, 48):
        cfg = synth.scaled_config(2, N_r=N_r, M=4, K=4)          # heated, both cylinders rotating
        o = oracle_of(cfg, dft="fft")
        nu = np.array(o.nusselt(o.base_state_discrete()))
        errs.append(np.max(np.abs(nu - 1.0)))
    assert errs[0] < 1e-5 and errs[1] < 1e-8 and errs[1] < errs[0]
    cfg = synth.scaled_config(0, N_r=24, M=4, K=4)               # no temperature: heat entries are nan
    o = oracle_of(cfg, dft="fft")
    nu = o.nusselt(o.base_state_discrete())
    assert np.isnan(nu[0]) and np.isnan(nu[1]) and abs(nu[2] - 1) < 1e-5 and abs(nu[3] - 1) < 1e-5


def test_nusselt_of_a_manufactured_profile():
    """A profile with a known wall derivative: T = T_b + a (r - r_i)^2 (r_o - r) adds nothing at the inner wall
    and a (r_o - r_i)^2 * (-1) at the outer one; u_theta = V + b (r - r_i)(r_o - r) changes the torque by the
    closed-form amount (polynomials of degree <= 8: the 9-point rows are exact)."""
    from paper_1908_00587_b200 import synth
    from helpers import oracle_of
    cfg = synth.scaled_config(2, N_r=32, M=4, K=4)
    o = oracle_of(cfg, dft="fft")
    st = o.base_state_discrete()
    base = np.array(o.nusselt(st))
    r, K, eta = o.r, cfg["K"], cfg["eta"]
    ri, ro = r[0], r[-1]
    a, b = 0.3, 7.0
    st[3][:, 0, K] += a * (r - ri) ** 2 * (ro - r)
    st[1][:, 0, K] += b * (r - ri) * (ro - r)
    nu = np.array(o.nusselt(st))
    B = eta * (cfg["Re_i"] - eta * cfg["Re_o"]) / ((1 - eta) * (1 - eta ** 2))
    want = base + np.array([0.0, -a * (ro - ri) ** 2 * ro * np.log(eta),
                            ri ** 3 * (b * (ro - ri) / ri) / (-2 * B), ro ** 3 * (-b * (ro - ri) / ro) / (-2 * B)])
    np.testing.assert_allclose(nu, want, rtol=0, atol=1e-9)


def test_probe_equals_the_transform_on_grid_points_and_a_single_mode_elsewhere():
    from paper_1908_00587_b200 import synth
    from helpers import oracle_of
    cfg = synth.scaled_config(1, N_r=12, M=4, K=4)
    o = oracle_of(cfg, dft="naive")
    st = synth.make_state(cfg, o.r)
    phys = o.to_physical(st[1])                                  # [N_r, N_theta, N_z]
    Nt, Nz = phys.shape[1], phys.shape[2]
    for (j, a, b) in [(0, 0, 0), (5, 3, 7), (11, Nt - 1, Nz - 1)]:
        theta = 2 * np.pi * a / (Nt * cfg["k_theta0"])
        z = 2 * np.pi * b / (Nz * cfg["alpha"])
        assert abs(o.probe(st[1], j, theta, z) - phys[j, a, b]) <= 1e-12 * np.max(np.abs(phys))
    f = o.zeros()
    f[:, 2, cfg["K"] + 3] = 1.5 - 0.5j                           # single mode (m, k) = (2, 3)
    theta, z = 0.37, 1.1
    n, kap = 2 * cfg["k_theta0"], 3 * cfg["alpha"]
    want = 2 * ((1.5 - 0.5j) * np.exp(1j * (n * theta + kap * z))).real
    assert abs(o.probe(f, 4, theta, z) - want) <= 1e-13
