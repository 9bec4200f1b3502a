"""Pins of the oracle's NEXT-1 step-size controller (Oracle.cfl_rate / advance, reading R17) and of the
NEXT-3 wave-speed measurement (Oracle.wave_speed).  CPU only."""
import numpy as np
import pytest

from helpers import oracle_of
from oracle.nsc_oracle import Oracle, rel_l2
from paper_1908_00587_b200 import synth


def test_dt_grid():
    for x in (1e-3, 3e-5, 1.0, 0.9, 1.125, 7.3e-9, 123.4):
        f = Oracle.dt_grid_floor(x)
        m, e = np.frexp(f)
        assert f <= x < Oracle.dt_grid_next(f)
        assert (m * 16) == int(m * 16) and 8 <= m * 16 < 16          # (8 + i) / 16 * 2^e
        assert Oracle.dt_grid_floor(f) == f
        assert 1.06 < Oracle.dt_grid_next(f) / f <= 1.125 + 1e-15


def test_cfl_rate_closed_forms():
    """lambda of circular Couette flow is Re_i / (r_i dtheta) (V / r = A + B / r^2 is largest at the inner wall);
    of a single axial cosine a cos(kappa z) it is a / dz; of a single azimuthal cosine in u_r with a radial
    profile g it is max_j 2 |c| g(r_j) / dr_j."""
    cfg = synth.scaled_config(0, N_r=24, M=8, K=8)
    o = oracle_of(cfg, dft="fft")
    p = o.p
    K = p.K
    dth = 2 * np.pi / (p.k_theta0 * p.n_theta)
    dz = 2 * np.pi / (p.alpha * p.n_z)
    st = o.base_state_discrete()
    lam, mx = o.cfl_rate(st)
    assert abs(lam - p.Re_i / (o.r[0] * dth)) <= 1e-12 * lam
    np.testing.assert_allclose(mx[1], np.abs(st[1][:, 0, K].real), rtol=1e-13)
    assert mx[0].max() == 0.0 and mx[2].max() == 0.0
    # axial cosine of amplitude a, larger than the rotation's rate
    a = 5e3
    st2 = [f.copy() if f is not None else None for f in st]
    st2[2][:, 0, K + 1] = a / 2
    st2[2][:, 0, K - 1] = a / 2
    lam2, mx2 = o.cfl_rate(st2)
    assert abs(lam2 - a / dz) <= 1e-12 * lam2
    # radial velocity 2 Re(c g(r) e^{i n theta}): peak 2 |c| g on the grid points theta_a = 2 pi a / (k0 N_theta)
    g = (o.r - o.r[0]) * (o.r[-1] - o.r)
    c = 3e3 + 0j
    st3 = [f.copy() if f is not None else None for f in st]
    st3[0][:, 1, K] = c * g
    lam3, mx3 = o.cfl_rate(st3)
    expect = (2 * abs(c) * g / o.radial_spacing()).max()
    assert expect > lam and abs(lam3 - expect) <= 1e-12 * lam3
    d = np.diff(o.r)
    assert o.radial_spacing()[0] == d[0] and o.radial_spacing()[-1] == d[-1]
    assert o.radial_spacing()[5] == min(d[4], d[5])


def test_controller_is_the_identity_at_steady_couette_flow():
    """At the discrete Couette fixed point every corrector converges in one pass with err = 0: all steps are
    accepted, the state does not move, dt climbs the grid until the CFL bound holds it."""
    cfg = synth.scaled_config(0, N_r=20, M=4, K=4)
    o = oracle_of(cfg, dft="fft")
    st = o.base_state_discrete()
    lam, _ = o.cfl_rate(st)
    cfl = 0.3
    new, t, log = o.advance(st, 1.0, 40, 1e-4, 1e-8, cfl, 4)
    assert all(ok and k == 1 and err <= 1e-13 for (_, k, err, ok) in log)
    dts = [d for (d, _, _, _) in log]
    bound = Oracle.dt_grid_floor(cfl / lam)
    assert dts[0] == Oracle.dt_grid_floor(1e-4)
    assert all(b == Oracle.dt_grid_next(a) or b == bound for a, b in zip(dts, dts[1:]))
    assert dts[-1] == bound and max(dts) == bound
    assert abs(t - sum(dts)) <= 1e-15
    assert rel_l2(new[:3], st[:3]) <= 1e-13


def test_dt_shrinks_after_an_impulsive_change_of_the_rotation_rate():
    """dynamic control "is of advantage if the flow state is suddenly modified (applying
    disturbances, changing rotation rates)".  A perturbed Couette flow of Re_i = 100 handed to a context with
    Re_i = 400: the first attempts (dt0 cut to the CFL bound, then halved) are rejected because the corrector
    does not converge to tol, dt is cut, then climbs the grid again as the wall layer diffuses; time advances
    only on accepted steps; t_end is hit exactly; rejected attempts leave the state untouched."""
    cfg = synth.scaled_config(0, N_r=20, M=4, K=4)
    o1 = oracle_of(cfg, dft="fft")
    st = synth.make_state(cfg, o1.r)
    o2 = oracle_of(dict(cfg, Re_i=400.0), dft="fft")
    dt0, t_end, tol, cfl = 4e-3, 8e-3, 1e-7, 0.5
    lam, _ = o2.cfl_rate(st)
    new, t, log = o2.advance(st, t_end, 200, dt0, tol, cfl, 2)
    dts = [d for (d, _, _, _) in log]
    acc = [d for (d, _, _, ok) in log if ok]
    assert dts[0] == Oracle.dt_grid_floor(cfl / lam) < Oracle.dt_grid_floor(dt0)      # the CFL bound acts first
    assert [ok for (_, _, _, ok) in log[:3]] == [False, False, True]                  # two rejections, halved each time
    assert dts[1] == Oracle.dt_grid_floor(dts[0] / 2) and dts[2] == Oracle.dt_grid_floor(dts[1] / 2)
    assert all((err <= tol) == ok for (_, _, err, ok) in log)
    assert min(acc) <= dts[0] / 8 and max(acc[3:-1]) >= 1.5 * min(acc[:-1])           # shrank, then recovered
    assert t == t_end and abs(sum(acc) - t_end) <= 1e-15
    # a rejected first attempt leaves the state untouched: one attempt only
    same, t1, log1 = o2.advance(st, t_end, 1, dt0, tol, cfl, 2)
    assert t1 == 0.0 and log1[0][3] is False and all(a is b for a, b in zip(same, st))
    # the same end time at a fixed small step: the same flow (the impulsive start is singular in time, so the two
    # step-size sequences differ by a first-order start-up error, not by round-off)
    ref = st
    n = 80
    for _ in range(n):
        ref = o2.step(ref, t_end / n)
    assert rel_l2(new[:3], ref[:3]) <= 2e-2


@pytest.mark.parametrize("m,k", [(2, 1), (1, -2)])
def test_wave_speed_of_a_scalar_carried_by_solid_body_rotation(m, k):
    """Pin of wave_speed: with Re_i = Omega r_i and Re_o = Omega r_o the Couette flow is the solid-body rotation
    u_theta = Omega r (degree 1 in r: exactly steady on the grid).  A temperature disturbance in one mode (m, k)
    obeys dT/dt + i n Omega T = (1/Pr) L T with L real, so its phase turns at exactly -n Omega whatever its
    radial shape: angular wave speed = Omega.  (Ra is tiny: temperature on, buoyancy negligible.)  The
    predictor-corrector step is second order: the measured speed approaches Omega like dt^2."""
    Omega = 40.0
    cfg = dict(synth.scaled_config(2, N_r=16, M=4, K=4), eta=0.5, Re_i=Omega * 1.0, Re_o=Omega * 2.0, Ra=1e-9, Pr=0.7)
    o = oracle_of(cfg, dft="fft")
    st = o.base_state_discrete()
    np.testing.assert_allclose(st[1][:, 0, o.p.K].real, Omega * o.r, rtol=1e-12)
    x = o.r - o.r[0]
    st[3][:, m, k + o.p.K] += 1e-3 * x * (1 - x) * (1 + 0.5j)
    sp = [o.wave_speed(st, 3, 7, m, k, dt, 8)[0] for dt in (2.5e-4, 1.25e-4)]
    errs = [abs(v - Omega) / Omega for v in sp]
    assert errs[1] <= 3e-4
    assert 3.8 <= errs[0] / errs[1] <= 4.2                         # second order in dt
    assert abs((4 * sp[1] - sp[0]) / 3 - Omega) <= 1e-5 * Omega    # Richardson limit dt -> 0: exactly Omega


# ------------------------------------------------------------------ NEXT-4: restart on another resolution (R18)
def _pair(N_src, M_src, K_src, grid_src, N_dst, M_dst, K_dst, grid_dst, ci=0):
    a = dict(synth.scaled_config(ci, N_r=N_src, M=M_src, K=K_src), grid=grid_src)
    b = dict(synth.scaled_config(ci, N_r=N_dst, M=M_dst, K=K_dst), grid=grid_dst)
    return a, b, oracle_of(a, dft="fft"), oracle_of(b, dft="fft")


@pytest.mark.parametrize("grids", [(1, 1), (1, 0), (0, 1)])
def test_regrid_is_exact_for_polynomials_of_degree_8_and_pads_modes(grids):
    """Radial interpolation reproduces r^p, p <= 8, to round-off on any pair of grids (and not r^9); modes the
    source does not hold come out zero, modes the target does not hold are dropped, shared modes keep their place."""
    ca, cb, oa, ob = _pair(20, 4, 8, grids[0], 33, 8, 4, grids[1])
    K_a, K_b = 8, 4
    st = [oa.zeros() for _ in range(3)] + [None, oa.zeros()]
    for p in range(10):
        for f in st:
            if f is not None:
                f[...] = 0
        st[1][:, 2, K_a + 3] = (1 + 2j) * oa.r ** p          # (m, k) = (2, 3): held by both
        st[1][:, 3, K_a - 7] = oa.r ** p                     # k = -7: not held by the target (K = 4)
        st[4][:, 0, K_a] = oa.r ** p
        out = ob.regrid(st, oa)
        err = np.abs(out[1][:, 2, K_b + 3] - (1 + 2j) * ob.r ** p).max() / (ob.r[-1] ** p)
        errp = np.abs(out[4][:, 0, K_b] - ob.r ** p).max() / (ob.r[-1] ** p)
        if p <= 8:
            assert err <= 5e-14 and errp <= 5e-14
        else:
            assert err > 1e-11
        assert out[3] is None and out[0].shape == (33, 9, 9)
        mask = np.ones(out[1].shape, bool)
        mask[:, 2, K_b + 3] = False
        assert np.all(out[1][mask] == 0)                     # k = -7 dropped, m = 5..8 padded with zeros


def test_regrid_onto_the_same_grid_is_the_identity_and_nodes_in_common_keep_their_values():
    ca, cb, oa, ob = _pair(17, 4, 4, 0, 33, 4, 4, 0)        # uniform grids: every second fine node is a coarse node
    st = synth.make_state(ca, oa.r)
    same = oa.regrid(st, oa)
    for a, b in zip(same, st):
        if b is not None:
            np.testing.assert_array_equal(a, b)
    fine = ob.regrid(st, oa)
    np.testing.assert_allclose(ob.r[::2], oa.r, rtol=0, atol=1e-15)
    for a, b in zip(fine, st):
        if b is not None:
            np.testing.assert_allclose(a[::2], b, rtol=0, atol=1e-13 * np.abs(b).max())
    W = ob.regrid_matrix(oa)
    np.testing.assert_allclose(W.sum(axis=1), 1.0, rtol=0, atol=1e-13)       # partition of unity
    assert np.count_nonzero(W[5]) <= 9


def test_regrid_interpolation_error_falls_at_ninth_order():
    errs = []
    for N in (12, 24, 48):
        ca, cb, oa, ob = _pair(N, 4, 4, 0, 101, 4, 4, 0)
        st = [oa.zeros() for _ in range(3)] + [None, None]
        st[0][:, 1, 4] = np.exp(1.3 * oa.r) * np.sin(2.0 * oa.r)
        out = ob.regrid(st, oa)
        errs.append(np.abs(out[0][:, 1, 4] - np.exp(1.3 * ob.r) * np.sin(2.0 * ob.r)).max())
    assert errs[0] / errs[1] >= 2 ** 8 and errs[1] / errs[2] >= 2 ** 8 or errs[2] <= 1e-13


def test_a_regridded_flow_keeps_running():
    """Restart of cfg 1 on a finer resolution: the interpolated state is divergence-free to interpolation accuracy,
    one step later to round-off again, and the coarse and the fine run agree on the shared modes."""
    ca, cb, oa, ob = _pair(24, 8, 8, 1, 32, 8, 8, 1)
    st = synth.make_state(ca, oa.r)
    for _ in range(2):
        st = oa.step(st, ca["dt"])
    fine = ob.regrid(st, oa)
    d0 = np.abs(ob.divergence(*fine[:3])[1:-1]).max()
    nxt = ob.step(fine, cb["dt"])
    d1 = np.abs(ob.divergence(*nxt[:3])[1:-1]).max()
    scale = np.abs(ob.D1) @ np.abs(nxt[1][:, 0, 8])
    assert d0 <= 1e-6 * scale.max() and d1 <= 1e-11 * scale.max()
    ref = oa.step(st, ca["dt"])
    back = oa.regrid(nxt, ob)
    assert rel_l2(back[:3], ref[:3]) <= 5e-6          # interpolation accuracy at these resolutions
