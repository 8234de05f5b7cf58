"""Pins of the oracle's mixed-precision mode (reading R6): the carried inverse is
STORED in fp32 -- rounded after every operation that writes it -- and every dot product / update is evaluated in fp64
on the stored values.  Written and pinned before any kernel stores an fp32 inverse.

  * storage: every element of the carried inverse is its own fp32 rounding, after create, after every rank-1 update,
    after every flush, after a recompute; the fp64 mode is untouched by the flag being off;
  * placement of the rounding: the stored inverse after a sweep equals a numpy replay of the logged moves that applies
    the textbook update in fp64 and rounds once per write (Sherman-Morrison per accepted move; the delayed window's
    product form per flush) -- bit for bit except where the two fp64 results straddle an fp32 rounding boundary
    (at most one fp32 ulp, a handful of elements);
  * accuracy: the stored inverse stays within 4 kappa_inf(A) 2^-24 of the exact inverse of the Slater matrix at the
    carried positions, sweep after sweep (every accepted move replaces one row of the matrix the stored inverse
    inverts exactly, so rounding errors do not accumulate beyond one sweep's worth); a recompute brings it back to
    one rounding of the exact inverse.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi

EPS32 = 2.0 ** -24


def _crowd(n_elec, kd, W=4, fp32=True, grid=8, tau=0.01, cfg=41):
    wl = qi.small_workload(n_elec=n_elec, grid=grid, box=1.44 * n_elec ** (1 / 3), coef_dtype="f32",
                           coef_dist="normal", n_walkers=W, tau=tau, delay_rank=kd, cfg=cfg)
    coefs, pos = qi.make_coefs(wl), qi.make_positions(wl)
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, tau=wl.tau, delay_rank=kd,
                               inverse_fp32=fp32)
    return wl, osys, oracle.OracleCrowd(osys, pos), pos


def _slater(osys, R, spin):
    n = osys.n
    return np.array([osys.spo_vgl(R[spin * n + i])[0] for i in range(n)])


@pytest.mark.parametrize("kd", [1, 4, 8])
def test_stored_inverse_is_fp32_valued_at_every_write(kd):
    wl, osys, oc, _ = _crowd(24, kd)
    _, _, ref, _ = _crowd(24, kd, fp32=False)
    for step in range(3):
        for spin in (0, 1):
            B = oc.inverse(spin)
            assert np.array_equal(B, B.astype(np.float32).astype(np.float64))
            assert not np.array_equal(ref.inverse(spin), ref.inverse(spin).astype(np.float32).astype(np.float64))
        oc.sweep(1)
        ref.sweep(1)
    oc.recompute()
    for spin in (0, 1):
        B = oc.inverse(spin)
        assert np.array_equal(B, B.astype(np.float32).astype(np.float64))
    assert np.array_equal(oracle.round_to_fp32(np.array([[1.0 + 2.0 ** -30, 1.0 + 2.0 ** -23], [1 / 3, -0.1]])),
                          np.array([[1.0, 1.0 + 2.0 ** -23], [np.float32(1 / 3), np.float32(-0.1)]], dtype=np.float64))


def _ulp32(x):
    return np.spacing(np.abs(x).astype(np.float32)).astype(np.float64)


@pytest.mark.parametrize("kd", [1, 6])
def test_rounding_is_applied_once_per_write_numpy_replay(kd):
    """The logged moves replayed in numpy: fp64 update on the fp32-valued state, one rounding per write."""
    n_elec = 24
    wl, osys, oc, pos = _crowd(n_elec, kd, W=3)
    n = n_elec // 2
    B0 = [oc.inverse(0).copy(), oc.inverse(1).copy()]
    _, log = oc.sweep(1, log=True)
    for w in range(3):
        for spin in (0, 1):
            B = B0[spin][w].copy()
            pending = []                                     # accepted moves of the open window: (row, phi)
            for kk in range(n):
                rec = log[0, w, spin * n + kk]
                if rec["accepted"]:
                    phi = osys.spo_vgl(rec["rnew"])[0]
                    if kd == 1:
                        f = (B @ phi - np.eye(n)[kk]) / rec["rho_d"]
                        B = (B - np.outer(f, B[kk].copy())).astype(np.float32).astype(np.float64)
                    else:
                        pending.append((kk, phi))
                if kd > 1 and ((kk + 1) % kd == 0 or kk == n - 1):
                    if pending:                              # the window's moves one after the other in fp64, ONE rounding
                        X = B.copy()
                        for row, phi in pending:
                            f = (X @ phi - np.eye(n)[row]) / (X[row] @ phi)
                            X = X - np.outer(f, X[row].copy())
                        B = X.astype(np.float32).astype(np.float64)
                    pending = []
            got = oc.inverse(spin)[w]
            diff = got != B
            assert diff.mean() <= 2e-3, diff.sum()           # two fp64 evaluation orders: a rounding straddle is rare
            assert (np.abs(got - B) <= 1.001 * _ulp32(B)).all()


@pytest.mark.parametrize("n_elec,kd", [(32, 1), (64, 8), (128, 32)])
def test_stored_inverse_stays_within_the_first_order_bound(n_elec, kd):
    wl, osys, oc, _ = _crowd(n_elec, kd, W=4)
    _, _, ref, _ = _crowd(n_elec, kd, W=4, fp32=False)
    n = n_elec // 2
    worst = 0.0
    for sweep in range(4):
        oc.sweep(1)
        ref.sweep(1)
        for (crowd, mixed) in ((oc, True), (ref, False)):
            R = crowd.positions()
            for w in range(4):
                for spin in (0, 1):
                    A = _slater(osys, R[w], spin)
                    Bex = np.linalg.inv(A).T
                    err = np.abs(crowd.inverse(spin)[w] - Bex).max() / np.abs(Bex).max()
                    kap = np.linalg.cond(A, np.inf)
                    if mixed:
                        assert err <= 4.0 * kap * EPS32, (sweep, w, spin, err, kap)
                        worst = max(worst, err)
                    else:
                        assert err <= 1e-4 * kap * EPS32       # the fp64 mode is orders of magnitude closer
    assert worst > 1e-9                                        # the mode does store in fp32
    oc.recompute()
    R = oc.positions()
    for w in range(4):
        for spin in (0, 1):
            Bex = np.linalg.inv(_slater(osys, R[w], spin)).T
            B = oc.inverse(spin)[w]
            assert (np.abs(B - Bex) <= 0.5001 * _ulp32(Bex) + 1e-11 * np.abs(Bex).max()).all()


def test_recompute_keeps_the_trajectory_definition():
    """oracle_crowd_recompute replaces the carried inverse by the inverse at the carried positions and leaves
    positions and caches as they are: in fp64 mode the next sweep is the same to rounding."""
    wl, osys, a, _ = _crowd(16, 4, W=3, fp32=False)
    _, _, b, _ = _crowd(16, 4, W=3, fp32=False)
    a.sweep(2)
    b.sweep(2)
    b.recompute()
    assert np.array_equal(a.positions(), b.positions())
    for spin in (0, 1):
        assert np.abs(a.inverse(spin) - b.inverse(spin)).max() <= 1e-9 * np.abs(a.inverse(spin)).max()
