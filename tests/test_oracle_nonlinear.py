"""Pin T4: the oracle's nonlinear term (O4; BASELINE.json north_star (a)).

(i)   hand-derived closed form for separable polynomial-in-r fields, all four equations,
      every advection and curvature term exercised with its sign;
(ii)  brute-force truncated convolution sums on a tiny mode set: equal for |k| < K, m < M,
      and independent of the padded grid there (readings R4, R5);
(iii) circular Couette flow: only N^_r(0,0) = +u_theta^2 / r survives.
"""
import numpy as np
import pytest
from oracle.nsc_oracle import Params, Oracle


def spec_from_phys_fn(o, fn):
    """Spectral coefficients of a band-limited analytic field fn(r, theta, z)."""
    p = o.p
    th = 2 * np.pi * np.arange(p.n_theta) / p.n_theta / p.k_theta0
    z = 2 * np.pi * np.arange(p.n_z) / p.n_z / p.alpha
    u = fn(o.r[:, None, None], th[None, :, None], z[None, None, :])
    return o.from_physical(u * np.ones((p.N_r, p.n_theta, p.n_z)))


@pytest.mark.parametrize("grid", [0, 1])
@pytest.mark.parametrize("heated", [False, True])
def test_closed_form_separable_fields(grid, heated):
    Ra, Pr = (3.0e3, 0.7) if heated else (0.0, 1.0)
    o = Oracle(Params(N_r=24, M=6, K=6, eta=0.6, alpha=1.7, k_theta0=2, Re_i=1.0, Re_o=0.0,
                      Ra=Ra, Pr=Pr, grid=grid))
    p = o.p
    n, kap = 2.0 * p.k_theta0, 2.0 * p.alpha                # physical wavenumbers used below
    ri = o.r[0]
    f = lambda r: 1.0 + 0.5 * (r - ri) - 0.8 * (r - ri) ** 3
    fp = lambda r: 0.5 - 2.4 * (r - ri) ** 2
    g = lambda r: 0.3 - (r - ri) ** 2 + 0.2 * (r - ri) ** 4
    gp = lambda r: -2 * (r - ri) + 0.8 * (r - ri) ** 3
    h = lambda r: -0.6 + 0.9 * (r - ri) ** 2
    hp = lambda r: 1.8 * (r - ri)
    q = lambda r: 0.4 + 0.7 * (r - ri) - 0.5 * (r - ri) ** 4
    qp = lambda r: 0.7 - 2.0 * (r - ri) ** 3
    ur = spec_from_phys_fn(o, lambda r, t, z: f(r) * np.cos(n * t))
    ut = spec_from_phys_fn(o, lambda r, t, z: g(r) * np.sin(n * t) + 0.25 * r)
    uz = spec_from_phys_fn(o, lambda r, t, z: h(r) * np.cos(kap * z))
    T = spec_from_phys_fn(o, lambda r, t, z: q(r) * np.sin(kap * z + n * t)) if heated else None
    out = o.nonlinear(ur, ut, uz, T)
    r = o.r[:, None, None]
    th = (2 * np.pi * np.arange(p.n_theta) / p.n_theta / p.k_theta0)[None, :, None]
    z = (2 * np.pi * np.arange(p.n_z) / p.n_z / p.alpha)[None, None, :]
    Ur, Ut, Uz = f(r) * np.cos(n * th), g(r) * np.sin(n * th) + 0.25 * r, h(r) * np.cos(kap * z)
    dUr = (fp(r) * np.cos(n * th), -n * f(r) * np.sin(n * th), 0.0)
    dUt = (gp(r) * np.sin(n * th) + 0.25, n * g(r) * np.cos(n * th), 0.0)
    dUz = (hp(r) * np.cos(kap * z), 0.0, -kap * h(r) * np.sin(kap * z))
    adv = lambda d: Ur * d[0] + Ut / r * d[1] + Uz * d[2]
    Nr = -(adv(dUr) - Ut * Ut / r)
    Nt = -(adv(dUt) + Ur * Ut / r)
    Nz = -adv(dUz) + 0 * th
    ph = [o.to_physical(a) for a in out]
    if heated:
        ph_arg = kap * z + n * th
        Tt = q(r) * np.sin(ph_arg)
        dT = (qp(r) * np.sin(ph_arg), n * q(r) * np.cos(ph_arg), kap * q(r) * np.cos(ph_arg))
        Nz = Nz + (Ra / Pr) * Tt
        np.testing.assert_allclose(ph[3], -adv(dT), atol=2e-12)
    np.testing.assert_allclose(ph[0], Nr, atol=2e-12)
    np.testing.assert_allclose(ph[1], Nt, atol=2e-12)
    np.testing.assert_allclose(ph[2], Nz * np.ones_like(ph[2]), atol=2e-9 if heated else 2e-12)


def full_spectrum(f, M, K):
    """[M+1, 2K+1] half spectrum of a real field -> dict over m in [-M, M]."""
    F = {}
    for m in range(-M, M + 1):
        for k in range(-K, K + 1):
            F[m, k] = f[m, k + K] if m >= 0 else np.conj(f[-m, -k + K])
    return F


def conv(F, G, M, K):
    out = np.zeros((M + 1, 2 * K + 1), complex)
    for m in range(0, M + 1):
        for k in range(-K, K + 1):
            s = 0.0
            for (m1, k1), a in F.items():
                b = G.get((m - m1, k - k1))
                if b is not None:
                    s += a * b
            out[m, k + K] = s
    return out


def test_brute_force_convolution_and_grid_independence():
    M, K = 3, 3
    base = dict(N_r=12, M=M, K=K, eta=0.5, alpha=3.0, k_theta0=1, Re_i=1.0, Re_o=0.0, Ra=50.0, Pr=0.7)
    o = Oracle(Params(**base))
    rng = np.random.default_rng(11)
    fields = []
    for _ in range(4):
        f = rng.standard_normal((12, M + 1, 2 * K + 1)) + 1j * rng.standard_normal((12, M + 1, 2 * K + 1))
        f[:, 0, :K] = np.conj(f[:, 0, :K:-1])
        f[:, 0, K] = f[:, 0, K].real
        fields.append(f)
    out = o.nonlinear(*fields)
    j = 5
    rj = o.r[j]
    i_n = 1j * o.n[:, None]
    i_k = 1j * o.kappa[None, :]
    S = lambda a: full_spectrum(a, M, K)
    U = [S(f[j]) for f in fields]
    dR = [S(np.einsum("l,lmk->mk", o.D1[j], f)) for f in fields]
    dT = [S(i_n * f[j]) for f in fields]
    dZ = [S(i_k * f[j]) for f in fields]
    adv = lambda i: conv(U[0], dR[i], M, K) + conv(U[1], dT[i], M, K) / rj + conv(U[2], dZ[i], M, K)
    ref = [-(adv(0) - conv(U[1], U[1], M, K) / rj),
           -(adv(1) + conv(U[0], U[1], M, K) / rj),
           -adv(2) + (50.0 / 0.7) * fields[3][j],
           -adv(3)]
    inner = (slice(0, M), slice(1, 2 * K))                 # m < M, |k| < K
    scale = max(np.abs(a).max() for a in ref)
    for a, b in zip(out, ref):
        np.testing.assert_allclose(a[j][inner], b[inner], atol=1e-12 * scale)
    # aliasing touches the extreme modes only: other padded grids agree on the inner set
    for nt, nz in ((9, 18), (12, 12), (16, 10)):
        o2 = Oracle(Params(**base, n_theta=nt, n_z=nz))
        out2 = o2.nonlinear(*fields, nodes=[j])
        for a, b in zip(out2, ref):
            np.testing.assert_allclose(a[0][inner], b[inner], atol=1e-12 * scale)
    # ... and the 3/2 grid does differ from the exact sum at |k| = K (reading R5)
    assert max(np.abs(a[j] - b).max() for a, b in zip(out, ref)) > 1e-6 * scale


def test_couette_only_centrifugal_term():
    o = Oracle(Params(N_r=16, M=4, K=4, eta=0.5, alpha=3.0, k_theta0=1, Re_i=100.0, Re_o=-20.0))
    st = o.base_state_discrete()
    v = st[1][:, 0, 4].real
    Nr, Nt, Nz = o.nonlinear(*st[:3])
    ref = np.zeros_like(Nr)
    ref[:, 0, 4] = v * v / o.r
    np.testing.assert_allclose(Nr, ref, atol=1e-11)
    assert np.abs(Nt).max() == 0.0 and np.abs(Nz).max() == 0.0


def test_nodes_subset_equals_full():
    o = Oracle(Params(N_r=14, M=3, K=4, eta=0.7, alpha=2.0, k_theta0=3, Re_i=10.0, Re_o=0.0, Ra=10.0))
    rng = np.random.default_rng(2)
    fs = [rng.standard_normal((14, 4, 9)) + 1j * rng.standard_normal((14, 4, 9)) for _ in range(4)]
    full = o.nonlinear(*fs)
    sub = o.nonlinear(*fs, nodes=[0, 6, 13])
    for a, b in zip(full, sub):
        np.testing.assert_array_equal(a[[0, 6, 13]], b)


# ------------------------------------------------------------------ T9 spatial order
def test_T9_spatial_order_of_the_nonlinear_term_on_the_uniform_grid():
    """Pin T9: for a non-polynomial field the error of N falls at >= 7th order under N_r doubling on
    the uniform grid (nine-point rows: degree-8 exactness).  Field: azimuthal flow V(r) = J_1(2.3 r)
    (a Bessel function) in mode (0,0) and a radial velocity a(r) e^{i(n theta + kappa z)} + c.c. with
    a = e^{-r}: the (m1,k1) coefficient of N_theta is then exactly -a (V' + V / r) (u_r d_r u_theta + u_r u_theta / r;
    every other product lands in other modes), and d_r V is the only place the finite differences enter."""
    from scipy.special import jv, jvp
    errs = []
    sizes = (12, 24, 48)
    for N_r in sizes:
        o = Oracle(Params(N_r=N_r, M=4, K=4, eta=0.5, alpha=1.5, k_theta0=2, Re_i=0.0, Re_o=0.0, grid=0))
        r = o.r
        ur, ut, uz = o.zeros(), o.zeros(), o.zeros()
        V, dV = jv(1, 2.3 * r), 2.3 * jvp(1, 2.3 * r)
        a = np.exp(-r) * (0.8 - 0.3j)
        ut[:, 0, 4] = V
        ur[:, 1, 5] = a
        N = o.nonlinear(ur, ut, uz)
        exact = -a * (dV + V / r)
        errs.append(np.abs(N[1][:, 1, 5] - exact).max() / np.abs(exact).max())
        # and N_r of the same pair: (u_theta / r) d_theta u_r = (V / r) i n a, no radial derivative: exact at any N_r
        exact_r = -(V / r) * 1j * o.n[1] * a
        assert np.abs(N[0][:, 1, 5] - exact_r).max() <= 1e-13 * np.abs(exact_r).max()
    assert errs[0] > 1e-9                                      # resolvable truncation error on the coarse grid
    orders = [np.log(errs[i] / errs[i + 1]) / np.log((sizes[i + 1] - 1) / (sizes[i] - 1)) for i in range(2)]
    assert orders[0] >= 7.0, (errs, orders)
    assert orders[1] >= 7.0 or errs[2] <= 1e-13, (errs, orders)
