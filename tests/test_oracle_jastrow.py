"""Pins for the oracle's two-body Jastrow factor (pin T5)."""
import numpy as np

import oracle


def make_sys(n_elec, box, a=0.5, b=1.0):
    m = n_elec // 2
    coefs = np.zeros((4, 4, 4, m))
    return oracle.OracleSystem(n_elec, (4, 4, 4), box, coefs, j2_a=a, j2_b=b)


def test_two_electron_closed_form_and_minimum_image():
    s = make_sys(2, (5.0, 5.0, 5.0))
    # r = 1: u = 0.5*1/(1+1) = 0.25
    assert abs(s.j2_logpsi([[0, 0, 0], [1, 0, 0]]) - 0.25) < 1e-16
    # separation 4 along x in a box of 5 -> minimum image distance 1, direction reversed
    assert abs(s.j2_logpsi([[0, 0, 0], [4, 0, 0]]) - 0.25) < 1e-15
    # r = 3 along the diagonal (1,2,2): u = 1.5/4
    assert abs(s.j2_logpsi([[0.5, 0.5, 0.5], [1.5, 2.5, 2.5]]) - 0.375) < 1e-15
    us, g = s.j2_usum_grad([[0, 0, 0], [1, 0, 0]], 0, [0, 0, 0])
    # electron 0 at origin, other at +x: d = r0 - r1 = (-1,0,0); u' = 0.5/4 -> grad = u' d/r
    assert abs(us - 0.25) < 1e-16
    np.testing.assert_allclose(g, [-0.125, 0, 0], atol=1e-16)
    us, g = s.j2_usum_grad([[0, 0, 0], [4, 0, 0]], 0, [0, 0, 0])
    np.testing.assert_allclose(g, [+0.125, 0, 0], atol=1e-15)   # image at -1 => d = (+1,0,0)


def test_sign_gives_positive_cusp():
    # d ln Psi_J / d r -> +a = +1/2 as r -> 0 (reading A14)
    s = make_sys(2, (5.0, 5.0, 5.0))
    e = 1e-7
    slope = (s.j2_logpsi([[0, 0, 0], [2 * e, 0, 0]]) - s.j2_logpsi([[0, 0, 0], [e, 0, 0]])) / e
    assert abs(slope - 0.5) < 1e-6


def test_non_cubic_box_and_parameters():
    s = make_sys(2, (3.0, 4.0, 6.0), a=0.7, b=2.0)
    # separations 2.9, 3.9, 5.9 -> images -0.1, -0.1, -0.1 -> r = 0.1*sqrt(3)
    r = 0.1 * np.sqrt(3)
    val = s.j2_logpsi([[0, 0, 0], [2.9, 3.9, 5.9]])
    assert abs(val - 0.7 * r / (1 + 2 * r)) < 1e-14


def test_ratio_equals_full_pair_sum_difference():
    rng = np.random.default_rng(0)
    n_elec, L = 10, 4.0
    s = make_sys(n_elec, (L, L, L))
    R = rng.uniform(0, L, size=(n_elec, 3))
    for k in range(n_elec):
        rnew = R[k] + rng.normal(0, 0.5, 3)
        u_old, _ = s.j2_usum_grad(R, k, R[k])
        u_new, _ = s.j2_usum_grad(R, k, rnew)
        R2 = R.copy()
        R2[k] = rnew
        assert abs((u_new - u_old) - (s.j2_logpsi(R2) - s.j2_logpsi(R))) < 1e-13


def test_gradient_by_finite_differences():
    rng = np.random.default_rng(1)
    n_elec, L = 8, 6.0
    s = make_sys(n_elec, (L, L, L))
    R = rng.uniform(0, L, size=(n_elec, 3))
    eps = 1e-6
    for k in range(n_elec):
        # stay away from the planes where a component of d crosses +-L/2 (gradient jumps there)
        d = R[k] - np.delete(R, k, axis=0)
        d -= L * np.rint(d / L)
        if np.min(np.abs(np.abs(d) - L / 2)) < 1e-3:
            continue
        _, g = s.j2_usum_grad(R, k, R[k])
        for c in range(3):
            Rp, Rm = R.copy(), R.copy()
            Rp[k, c] += eps
            Rm[k, c] -= eps
            fd = (s.j2_logpsi(Rp) - s.j2_logpsi(Rm)) / (2 * eps)
            assert abs(g[c] - fd) < 1e-8
