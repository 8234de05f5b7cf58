"""Pins for the oracle's tricubic B-spline (pins T3/T4).

Every check is a closed form or an invariant of uniform cubic B-splines, not a re-typing of
the oracle's sum:  partition of unity; the quasi-interpolation identities
    sum_m a_m(t) (m-1-t)^0 = 1,   sum_m a_m(t) (i-1+m) = i + t,   sum_m a_m(t) (i-1+m)^2 = (i+t)^2 + 1/3
(the cubic B-spline has mean 0 and variance 1/3); the DFT eigenvalue (4 + 2 cos w)/6 at grid
points; periodicity; central finite differences.
"""
import numpy as np
import pytest

import oracle


def make_sys(coefs, box, n_orb=None):
    g = coefs.shape[:3]
    m = coefs.shape[3]
    return oracle.OracleSystem(2 * m, g, box, coefs)


GRID = (6, 7, 8)          # deliberately non-cubic: catches axis mix-ups
BOX = (3.0, 4.2, 5.6)     # h = 0.5, 0.6, 0.7


def idx_table(axis, power, m=2):
    g = GRID
    t = np.zeros(g + (m,))
    ii = np.arange(g[axis], dtype=np.float64) ** power
    shape = [1, 1, 1, 1]
    shape[axis] = g[axis]
    t += ii.reshape(shape)
    return t


def interior_points(rng, n):
    # keep the 4-point stencil away from the periodic wrap: i-1 >= 0 and i+2 <= Ng-1
    pts = []
    for _ in range(n):
        p = []
        for c in range(3):
            h = BOX[c] / GRID[c]
            p.append(rng.uniform(1.0 * h, (GRID[c] - 2.0) * h))
        pts.append(p)
    return np.array(pts)


def test_weights_identities():
    for t in np.linspace(0.0, 1.0, 21):
        a, da, d2a = oracle.bspline_weights(float(t))
        m = np.arange(4.0)
        assert abs(a.sum() - 1) < 1e-15 and abs(da.sum()) < 1e-15 and abs(d2a.sum()) < 1e-15
        assert np.all(a >= 0)
        assert abs((a * m).sum() - (t + 1)) < 1e-15                 # first moment
        assert abs((a * (m - 1 - t) ** 2).sum() - 1.0 / 3.0) < 1e-15  # variance 1/3
        assert abs((da * m).sum() - 1) < 1e-15                      # d/dt of first moment
        assert abs((d2a * m ** 2).sum() - 2) < 1e-14                # d2/dt2 of second moment


def test_weights_continuity_across_cells():
    # C2 continuity: weights at t=1 of cell i equal weights at t=0 of cell i+1 shifted by one
    a1, da1, d2a1 = oracle.bspline_weights(1.0)
    a0, da0, d2a0 = oracle.bspline_weights(0.0)
    np.testing.assert_allclose(a1[1:], a0[:3], atol=1e-16)
    np.testing.assert_allclose(da1[1:], da0[:3], atol=1e-16)
    np.testing.assert_allclose(d2a1[1:], d2a0[:3], atol=1e-16)
    assert a1[0] == 0 and a0[3] == 0


def test_partition_of_unity():
    coefs = np.full(GRID + (3,), 2.5)
    coefs[..., 1] = -1.0
    s = make_sys(np.concatenate([coefs, coefs[..., :1]], axis=3), BOX)
    rng = np.random.default_rng(0)
    for r in rng.uniform(-10, 10, size=(20, 3)):
        phi, dphi, d2phi = s.spo_vgl(r)
        np.testing.assert_allclose(phi, [2.5, -1.0, 2.5, 2.5], rtol=0, atol=1e-14)
        assert np.max(np.abs(dphi)) < 1e-13 and np.max(np.abs(d2phi)) < 1e-12


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_linear_table_closed_form(axis):
    s = make_sys(idx_table(axis, 1), BOX)
    h = BOX[axis] / GRID[axis]
    for r in interior_points(np.random.default_rng(axis), 25):
        phi, dphi, d2phi = s.spo_vgl(r)
        np.testing.assert_allclose(phi, r[axis] / h, rtol=1e-13)
        expect = np.zeros(3)
        expect[axis] = 1 / h
        np.testing.assert_allclose(dphi[:, 0], expect, atol=1e-12)
        assert np.max(np.abs(d2phi)) < 1e-11


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_quadratic_table_closed_form(axis):
    # phi = u^2 + 1/3, d/dx = 2u/h, Laplacian = 2/h^2  (u = x/h)
    s = make_sys(idx_table(axis, 2), BOX)
    h = BOX[axis] / GRID[axis]
    for r in interior_points(np.random.default_rng(10 + axis), 25):
        u = r[axis] / h
        phi, dphi, d2phi = s.spo_vgl(r)
        np.testing.assert_allclose(phi, u * u + 1 / 3, rtol=1e-13)
        expect = np.zeros(3)
        expect[axis] = 2 * u / h
        np.testing.assert_allclose(dphi[:, 1], expect, atol=1e-11)
        np.testing.assert_allclose(d2phi, 2 / h ** 2, rtol=1e-12)


def test_sum_of_squares_laplacian_and_product_table():
    # P = ix^2 + iy^2 + iz^2 -> Laplacian = 2/hx^2 + 2/hy^2 + 2/hz^2 ; P = ix*iy*iz -> phi = ux uy uz
    t2 = idx_table(0, 2, 1) + idx_table(1, 2, 1) + idx_table(2, 2, 1)
    tp = idx_table(0, 1, 1) * idx_table(1, 1, 1) * idx_table(2, 1, 1)
    s = make_sys(np.concatenate([t2, tp], axis=3), BOX)
    h = np.array(BOX) / np.array(GRID)
    for r in interior_points(np.random.default_rng(5), 25):
        u = r / h
        phi, dphi, d2phi = s.spo_vgl(r)
        np.testing.assert_allclose(phi[0], (u ** 2).sum() + 1.0, rtol=1e-13)
        np.testing.assert_allclose(d2phi[0], (2 / h ** 2).sum(), rtol=1e-12)
        np.testing.assert_allclose(dphi[:, 0], 2 * u / h, rtol=1e-12)
        np.testing.assert_allclose(phi[1], u.prod(), rtol=1e-13)
        np.testing.assert_allclose(dphi[:, 1], u.prod() / u / h, rtol=1e-12)
        assert abs(d2phi[1]) < 1e-10


def test_orbital_index_is_innermost():
    m = 5
    coefs = np.zeros(GRID + (m,))
    coefs += np.arange(m, dtype=np.float64)
    coefs = np.concatenate([coefs, coefs[..., :1]], axis=3)   # even count not needed; M = 6
    s = make_sys(coefs, BOX)
    phi, _, _ = s.spo_vgl([0.3, 0.1, 0.2])
    np.testing.assert_allclose(phi, [0, 1, 2, 3, 4, 0], atol=1e-14)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_cosine_table_at_grid_points(axis):
    # DFT eigenvalue of the cubic B-spline mask (1,4,1)/6: includes the periodic wrap (i = 0, Ng-1)
    ng = GRID[axis]
    for q in (1, 2):
        t = np.zeros(GRID + (2,))
        shape = [1, 1, 1, 1]
        shape[axis] = ng
        t += np.cos(2 * np.pi * q * np.arange(ng) / ng).reshape(shape)
        s = make_sys(t, BOX)
        h = BOX[axis] / ng
        for i in range(-2, ng + 3):
            r = np.array([0.123, 0.456, 0.789])
            r[axis] = i * h + 1e-13      # just inside cell i (t ~ 0)
            phi, _, _ = s.spo_vgl(r)
            expect = np.cos(2 * np.pi * q * i / ng) * (4 + 2 * np.cos(2 * np.pi * q / ng)) / 6
            np.testing.assert_allclose(phi, expect, atol=1e-11)


def test_periodicity_and_negative_coordinates():
    rng = np.random.default_rng(3)
    coefs = rng.uniform(-1, 1, size=GRID + (4,))
    s = make_sys(coefs, BOX)
    for r in rng.uniform(-3, 8, size=(10, 3)):
        ref = s.spo_vgl(r)
        for c in range(3):
            for sh in (-2, -1, 1):
                r2 = r.copy()
                r2[c] += sh * BOX[c]
                got = s.spo_vgl(r2)
                for a, b in zip(ref, got):
                    np.testing.assert_allclose(a, b, atol=1e-9)   # t differs by rounding of the shift


def test_finite_differences_random_table():
    rng = np.random.default_rng(4)
    coefs = rng.uniform(-1, 1, size=GRID + (4,))
    s = make_sys(coefs, BOX)
    eps = 1e-5
    for r in rng.uniform(-1, 6, size=(10, 3)):
        phi, dphi, d2phi = s.spo_vgl(r)
        lap = np.zeros_like(phi)
        for c in range(3):
            rp, rm = r.copy(), r.copy()
            rp[c] += eps
            rm[c] -= eps
            pp, dp, _ = s.spo_vgl(rp)
            pm, dm, _ = s.spo_vgl(rm)
            np.testing.assert_allclose(dphi[c], (pp - pm) / (2 * eps), atol=1e-8)
            lap += (dp[c] - dm[c]) / (2 * eps)
        np.testing.assert_allclose(d2phi, lap, atol=1e-7)


def test_float32_table_gives_same_values_as_its_float64_copy():
    rng = np.random.default_rng(6)
    c32 = rng.standard_normal(size=GRID + (4,), dtype=np.float32)
    s32, s64 = make_sys(c32, BOX), make_sys(c32.astype(np.float64), BOX)
    for r in rng.uniform(-1, 6, size=(5, 3)):
        for a, b in zip(s32.spo_vgl(r), s64.spo_vgl(r)):
            assert np.array_equal(a, b)
