"""Pins of the oracle's kinetic energy (Alg. 1 line 11).

Nothing here re-types the oracle's formula: the reference values are (1) central second differences of the
brute-force wave function Psi(R) = det A_up(R) det A_dn(R) exp(J(R)) evaluated with numpy determinants -- exact for
the piecewise-cubic orbitals as long as the stencil stays inside one grid cell, O(h^2) for the Jastrow; (2) the
two-electron Jastrow-only closed form; (3) a plane-wave-like separable orbital where lap phi / phi is known.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi


def _system(n_elec, grid, box, seed, j2_a=0.5, j2_b=1.0, coefs=None):
    wl = qi.small_workload(n_elec=n_elec, grid=grid, box=box, coef_dtype="f64", coef_dist="uniform", n_walkers=1, cfg=seed)
    coefs = qi.make_coefs(wl) if coefs is None else coefs
    return oracle.OracleSystem(n_elec, (grid,) * 3, (box,) * 3, coefs, j2_a=j2_a, j2_b=j2_b, tau=0.02), wl


def _psi(osys, R):
    """Brute force: numpy determinants of the Slater matrices times exp(J)."""
    n = osys.n_elec // 2
    A = np.array([osys.spo_vgl(R[i])[0] for i in range(osys.n_elec)])
    return np.linalg.det(A[:n]) * np.linalg.det(A[n:]) * np.exp(osys.j2_logpsi(R))


def _inverses(osys, R):
    n = osys.n_elec // 2
    A = np.array([osys.spo_vgl(R[i])[0] for i in range(osys.n_elec)])
    return np.linalg.inv(A[:n]).T.copy(), np.linalg.inv(A[n:]).T.copy()


def _positions_inside_cells(rng, n_elec, grid, box, margin):
    """Positions whose +-margin stencil stays inside one grid cell on every axis (cubic pieces => exact FD)."""
    h = box / grid
    cell = rng.integers(0, grid, size=(n_elec, 3))
    frac = rng.uniform(margin / h + 0.05, 1.0 - margin / h - 0.05, size=(n_elec, 3))
    return (cell + frac) * h


@pytest.mark.parametrize("n_elec,grid,j2_a", [(4, 6, 0.5), (8, 8, 0.5), (6, 5, 0.0)])
def test_kinetic_matches_finite_difference_laplacian_of_brute_force_psi(n_elec, grid, j2_a):
    box, hfd = 4.0, 2e-4
    osys, _ = _system(n_elec, grid, box, seed=41 + n_elec, j2_a=j2_a)
    rng = np.random.default_rng(7 + n_elec)
    R = _positions_inside_cells(rng, n_elec, grid, box, hfd)
    Bu, Bd = _inverses(osys, R)
    t, e = osys.kinetic_energy(R, Bu, Bd)
    psi0 = _psi(osys, R)
    e_fd = np.zeros(n_elec)
    for k in range(n_elec):
        lap = 0.0
        for c in range(3):
            Rp, Rm = R.copy(), R.copy()
            Rp[k, c] += hfd
            Rm[k, c] -= hfd
            lap += (_psi(osys, Rp) + _psi(osys, Rm) - 2.0 * psi0) / hfd ** 2
        e_fd[k] = -0.5 * lap / psi0
    assert np.allclose(e, e_fd, rtol=0, atol=2e-5 * max(1.0, np.abs(e_fd).max()))
    assert abs(t - e.sum()) <= 1e-12 * max(1.0, abs(t))


def test_two_electron_jastrow_only_closed_form():
    """Constant orbital (one electron per spin, phi = 1): Psi = exp(u(r12)); lap_k Psi / Psi = u'' + 2u'/r + u'^2."""
    grid, box, a, b = 4, 6.0, 0.7, 1.3
    coefs = np.ones((grid, grid, grid, 1))
    osys, _ = _system(2, grid, box, seed=50, j2_a=a, j2_b=b, coefs=coefs)
    R = np.array([[1.0, 1.2, 0.9], [2.1, 0.7, 1.6]])
    r = np.linalg.norm(R[0] - R[1])
    du, d2u = a / (1 + b * r) ** 2, -2 * a * b / (1 + b * r) ** 3
    per = -0.5 * (d2u + 2 * du / r + du ** 2)
    one = np.ones((1, 1))
    t, e = osys.kinetic_energy(R, one, one)
    assert np.allclose(e, [per, per], rtol=1e-12) and abs(t - 2 * per) < 1e-12


def test_single_orbital_no_jastrow_is_minus_half_lap_phi_over_phi():
    """n = 1 per spin, a = 0: Psi = phi(r_0) phi(r_1), so the electron term is -1/2 lap phi / phi from the spline."""
    grid, box = 8, 4.0
    osys, _ = _system(2, grid, box, seed=51, j2_a=0.0)
    R = np.array([[0.31, 1.7, 2.9], [3.3, 0.4, 1.1]])
    vals = [osys.spo_vgl(R[i]) for i in range(2)]
    Bu, Bd = np.array([[1.0 / vals[0][0][0]]]), np.array([[1.0 / vals[1][0][0]]])
    t, e = osys.kinetic_energy(R, Bu, Bd)
    ref = [-0.5 * vals[i][2][0] / vals[i][0][0] for i in range(2)]
    assert np.allclose(e, ref, rtol=1e-12)
