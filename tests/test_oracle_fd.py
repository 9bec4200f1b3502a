"""Pin T1: the oracle's finite-difference tables (O2, "nine points").

* exact for polynomials of degree <= 8 on both grids, not for degree 9;
* on a uniform grid the centred rows are the textbook 8th-order coefficients
  (tests/golden/fd8_central.txt).
"""
import os
import numpy as np
import pytest
from oracle.nsc_oracle import radial_grid, fd_tables, stencil_start, LD

GOLD = os.path.join(os.path.dirname(__file__), "golden", "fd8_central.txt")


@pytest.mark.parametrize("kind", [0, 1])
@pytest.mark.parametrize("N_r", [9, 16, 33])
def test_polynomial_exactness(kind, N_r):
    r = radial_grid(N_r, 0.5, kind, dtype=LD)
    D1, D2 = (a.astype(float) for a in fd_tables(r))
    rf = r.astype(float)
    x = rf - rf[0] - 0.5                      # centred variable keeps the scale O(1)
    for p in range(0, 9):
        f = x ** p
        d1 = p * x ** (p - 1) if p > 0 else 0 * x
        d2 = p * (p - 1) * x ** (p - 2) if p > 1 else 0 * x
        s1 = np.abs(D1) @ np.abs(f) + 1e-300
        s2 = np.abs(D2) @ np.abs(f) + 1e-300
        assert np.max(np.abs(D1 @ f - d1) / s1) < 5e-15, (kind, N_r, p)
        assert np.max(np.abs(D2 @ f - d2) / s2) < 5e-15, (kind, N_r, p)
    f = x ** 9
    err = np.max(np.abs(D1 @ f - 9 * x ** 8))
    if N_r < 33:
        assert err > 1e-9                     # degree 9 is NOT reproduced (so the order is exactly 8)


def test_textbook_central_coefficients():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    c1 = np.array([float(LD(a) / LD(b)) for a, b in (t.split("/") for t in rows[0])])
    c2 = np.array([float(LD(a) / LD(b)) for a, b in (t.split("/") for t in rows[1])])
    N_r = 17
    r = radial_grid(N_r, 0.5, 0, dtype=LD)
    D1, D2 = (a.astype(float) for a in fd_tables(r))
    h = 1.0 / (N_r - 1)
    j = 8
    assert stencil_start(j, N_r) == 4
    np.testing.assert_allclose(D1[j, 4:13] * h, c1, rtol=0, atol=2e-15)
    np.testing.assert_allclose(D2[j, 4:13] * h * h, c2, rtol=0, atol=2e-14)
    assert np.count_nonzero(D2[j]) == 9 and np.all(D1[j, :4] == 0) and np.all(D1[j, 13:] == 0)


def test_wall_stencils_are_shifted_windows():
    N_r = 20
    r = radial_grid(N_r, 0.71, 1, dtype=LD)
    D1, _ = fd_tables(r)
    for j in range(N_r):
        nz = np.nonzero(D1[j].astype(float))[0]
        s = stencil_start(j, N_r)
        assert nz.min() >= s and nz.max() <= s + 8
    assert stencil_start(0, N_r) == 0 and stencil_start(3, N_r) == 0 and stencil_start(5, N_r) == 1
    assert stencil_start(N_r - 1, N_r) == N_r - 9
