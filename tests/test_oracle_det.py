"""Pins for the oracle's determinant algebra (pins T1/T2).

Reference = brute force with numpy's LAPACK: det(A')/det(A) and inv(A').T recomputed from
scratch.  The oracle never calls LAPACK (its LU is hand written), so this is independent.
"""
import numpy as np
import pytest

import oracle


def rand_matrix(rng, n):
    return rng.standard_normal((n, n)) + 0.5 * np.eye(n)


@pytest.mark.parametrize("n", [1, 2, 4, 8, 33])
def test_lu_inverse_transpose_vs_lapack(n):
    rng = np.random.default_rng(n)
    A = rand_matrix(rng, n)
    st, B, logabs, sign = oracle.lu_inverse_transpose(A)
    assert st == 0
    np.testing.assert_allclose(B, np.linalg.inv(A).T, rtol=1e-11, atol=1e-12)
    sg, la = np.linalg.slogdet(A)
    assert sign == int(sg) and abs(logabs - la) < 1e-12


def test_lu_needs_pivoting_and_flags_singular():
    A = np.array([[0.0, 2.0], [3.0, 1.0]])           # zero leading pivot
    st, B, _, sign = oracle.lu_inverse_transpose(A)
    assert st == 0 and sign == -1
    np.testing.assert_allclose(B, np.linalg.inv(A).T, atol=1e-15)
    st, *_ = oracle.lu_inverse_transpose(np.array([[1.0, 2.0], [2.0, 4.0]]))
    assert st == 4
    st, *_ = oracle.lu_inverse_transpose(np.array([[np.nan, 1.0], [2.0, 4.0]]))
    assert st == 4


@pytest.mark.parametrize("n", [2, 4, 8])
def test_ratio_is_brute_force_determinant_ratio(n):
    # T1: rho_D = B[k,:].phi' must equal det(A')/det(A) with row k of A replaced by phi'
    rng = np.random.default_rng(100 + n)
    A = rand_matrix(rng, n)
    _, B, _, _ = oracle.lu_inverse_transpose(A)
    for k in range(n):
        phi = rng.standard_normal(n)
        A2 = A.copy()
        A2[k] = phi
        rho = B[k] @ phi
        assert abs(rho - np.linalg.det(A2) / np.linalg.det(A)) < 1e-11 * max(1, abs(rho))


@pytest.mark.parametrize("n", [2, 4, 8, 32])
def test_sherman_morrison_vs_reinversion(n):
    rng = np.random.default_rng(200 + n)
    A = rand_matrix(rng, n)
    _, B, _, _ = oracle.lu_inverse_transpose(A)
    for k in rng.permutation(n)[: min(n, 8)]:
        phi = rng.standard_normal(n)
        rho = B[k] @ phi
        B = oracle.sm_update(B, int(k), phi, rho)
        A[k] = phi
        np.testing.assert_allclose(B, np.linalg.inv(A).T, rtol=1e-9, atol=1e-10)


def _window(rng, A, B0, rows):
    n = A.shape[0]
    V = rng.standard_normal((len(rows), n))
    Cm = B0[rows].copy()
    A2 = A.copy()
    for l, r in enumerate(rows):
        A2[r] = V[l]
    return V, Cm, A2


@pytest.mark.parametrize("n,m", [(4, 1), (4, 3), (8, 4), (16, 5), (32, 32)])
def test_delayed_row_and_flush_vs_reinversion(n, m):
    rng = np.random.default_rng(300 + 10 * n + m)
    A = rand_matrix(rng, n)
    _, B0, _, _ = oracle.lu_inverse_transpose(A)
    rows = rng.permutation(n)[:m].astype(np.int32)
    V, Cm, A2 = _window(rng, A, B0, rows)
    Bref = np.linalg.inv(A2).T
    for k in range(n):                                  # rows in and out of the window
        b = oracle.delayed_row(B0, rows, V, Cm, k)
        np.testing.assert_allclose(b, Bref[k], rtol=1e-8, atol=1e-9)
    Bf = oracle.delayed_flush(B0, rows, V, Cm)
    np.testing.assert_allclose(Bf, Bref, rtol=1e-8, atol=1e-9)


def test_delayed_rank1_equals_sherman_morrison_and_empty_window_is_identity():
    rng = np.random.default_rng(7)
    n = 6
    A = rand_matrix(rng, n)
    _, B0, _, _ = oracle.lu_inverse_transpose(A)
    phi = rng.standard_normal(n)
    k = 2
    Bsm = oracle.sm_update(B0, k, phi, B0[k] @ phi)
    Bd = oracle.delayed_flush(B0, [k], phi[None, :], B0[[k]])
    np.testing.assert_allclose(Bd, Bsm, rtol=1e-12, atol=1e-13)
    empty = np.zeros((0, n))
    assert np.array_equal(oracle.delayed_flush(B0, [], empty, empty), B0)
    assert np.array_equal(oracle.delayed_row(B0, [], empty, empty, 3), B0[3])


def test_delayed_ratios_are_sequential_determinant_ratios():
    # growing window: each new ratio b.phi' equals det(A_{m+1})/det(A_m) (Schur complement identity)
    rng = np.random.default_rng(8)
    n = 8
    A = rand_matrix(rng, n)
    _, B0, _, _ = oracle.lu_inverse_transpose(A)
    rows, V, Cm = [], np.zeros((0, n)), np.zeros((0, n))
    Acur = A.copy()
    for k in [5, 0, 3, 7, 1]:
        phi = rng.standard_normal(n)
        b = oracle.delayed_row(B0, rows, V, Cm, k)
        Anew = Acur.copy()
        Anew[k] = phi
        assert abs(b @ phi - np.linalg.det(Anew) / np.linalg.det(Acur)) < 1e-10
        rows.append(k)
        V = np.vstack([V, phi])
        Cm = np.vstack([Cm, B0[k]])
        Acur = Anew
