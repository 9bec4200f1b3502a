"""Pin T2: the oracle's transforms (O3).

* closed form: a single retained mode maps to the cosine it stands for;
* round trip spectral -> physical -> spectral is the identity on the retained set;
* Parseval: mean(u^2) = sum_k |u^(0,k)|^2 + 2 sum_{m>=1,k} |u^(m,k)|^2;
* the naive sums agree with numpy's FFT routines (library special case), which also pins
  the ``dft="fft"`` backend used at the large configurations;
* the m = 0 row takes the real part (reading R6).
"""
import numpy as np
import pytest
from oracle.nsc_oracle import Params, Oracle


def make(M=4, K=5, n_theta=0, n_z=0, dft="naive"):
    return Oracle(Params(N_r=9, M=M, K=K, eta=0.5, alpha=2.0, k_theta0=1, Re_i=1.0, Re_o=0.0,
                         n_theta=n_theta, n_z=n_z), dft=dft)


def rand_spec(o, rng, hermitian_m0=True):
    p = o.p
    f = rng.standard_normal((2, p.M + 1, 2 * p.K + 1)) + 1j * rng.standard_normal((2, p.M + 1, 2 * p.K + 1))
    if hermitian_m0:
        f[:, 0, :p.K] = np.conj(f[:, 0, :p.K:-1])
        f[:, 0, p.K] = f[:, 0, p.K].real
    return f


@pytest.mark.parametrize("m,k", [(0, 0), (0, 2), (3, 0), (2, -3), (4, 5), (1, 1)])
def test_single_mode_closed_form(m, k):
    o = make()
    p = o.p
    f = np.zeros((1, p.M + 1, 2 * p.K + 1), complex)
    amp = 0.7 - 0.4j
    f[0, m, k + p.K] = amp
    if m == 0 and k != 0:
        f[0, 0, -k + p.K] = np.conj(amp)
    if m == 0 and k == 0:
        f[0, 0, p.K] = amp.real
    u = o.to_physical(f)[0]
    th = 2 * np.pi * np.arange(p.n_theta) / p.n_theta
    z = 2 * np.pi * np.arange(p.n_z) / p.n_z
    ph = m * th[:, None] + k * z[None, :]
    if m == 0 and k == 0:
        ref = amp.real + 0 * ph
    else:
        ref = 2 * (amp.real * np.cos(ph) - amp.imag * np.sin(ph))
    np.testing.assert_allclose(u, ref, atol=1e-14)


@pytest.mark.parametrize("grid", [(0, 0), (12, 30), (15, 15), (16, 17)])
def test_round_trip_and_parseval(grid):
    o = make(n_theta=grid[0], n_z=grid[1])
    rng = np.random.default_rng(3)
    f = rand_spec(o, rng)
    u = o.to_physical(f)
    assert u.dtype == np.float64
    g = o.from_physical(u)
    np.testing.assert_allclose(g, f, atol=5e-14)
    w = np.where(np.arange(o.p.M + 1) == 0, 1.0, 2.0)[None, :, None]
    np.testing.assert_allclose((u ** 2).mean(axis=(1, 2)), (w * np.abs(f) ** 2).sum(axis=(1, 2)), rtol=1e-12)


@pytest.mark.parametrize("grid", [(0, 0), (12, 30), (15, 15)])
def test_naive_sums_equal_library_fft(grid):
    o = make(n_theta=grid[0], n_z=grid[1])
    of = make(n_theta=grid[0], n_z=grid[1], dft="fft")
    rng = np.random.default_rng(5)
    f = rand_spec(o, rng, hermitian_m0=False)          # generic m=0 row on purpose
    u, uf = o.to_physical(f), of.to_physical(f)
    np.testing.assert_allclose(u, uf, atol=2e-13)
    x = rng.standard_normal(u.shape)
    np.testing.assert_allclose(o.from_physical(x), of.from_physical(x), atol=2e-14)


def test_m0_row_takes_real_part():
    o = make()
    rng = np.random.default_rng(7)
    f = rand_spec(o, rng, hermitian_m0=False)
    f[:, 1:, :] = 0
    # symmetrised copy of the m = 0 row gives the same physical field
    g = f.copy()
    g[:, 0, :] = 0.5 * (f[:, 0, :] + np.conj(f[:, 0, ::-1]))
    np.testing.assert_allclose(o.to_physical(f), o.to_physical(g), atol=1e-14)


@pytest.mark.parametrize("M,K", [(256, 8), (8, 256), (512, 4), (4, 512), (128, 128)])
def test_library_fft_pinned_to_naive_sums_at_the_long_lengths(M, K):
    """The ``dft="fft"`` backend (numpy FFT as a library primitive) against the naive sums at the line lengths of
    BASELINE.json configs[2..4] (384, 768, 1536), where the 20-step parity runs use it as the checker."""
    p = Params(N_r=9, M=M, K=K, eta=0.5, alpha=3.0, k_theta0=1, Re_i=1.0, Re_o=0.0)
    o, of = Oracle(p), Oracle(p, dft="fft")
    rng = np.random.default_rng(11)
    f = (rng.standard_normal((2, M + 1, 2 * K + 1)) + 1j * rng.standard_normal((2, M + 1, 2 * K + 1)))
    u, uf = o.to_physical(f), of.to_physical(f)
    assert np.abs(u - uf).max() <= 1e-13 * np.abs(u).max()
    x = rng.standard_normal(u.shape)
    a, b = o.from_physical(x), of.from_physical(x)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()
