"""Periodic recompute of the inverses (first half; include/qmc_crowd.h qmc_recompute_inverse).

Definition checked here: after a recompute the carried inverse IS the inverse of the Slater matrix at the carried positions
(PAPER.md:76 names the carried data; oracle: oracle_lu_inverse_transpose of the oracle's own spline values), the
trajectory continues from it exactly as a fresh crowd created at those positions would, and the round-off drift the
updates accumulate is removed.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy

pytestmark = pytest.mark.gpu


def _wl(kd, coef_dtype="f64", W=6, n_elec=32, cfg=21):
    return qi.small_workload(n_elec=n_elec, grid=10, box=6.0, coef_dtype=coef_dtype, coef_dist="normal", n_walkers=W,
                             tau=0.02, delay_rank=kd, cfg=cfg)


@pytest.mark.parametrize("kd", [1, 4, 8])
def test_recompute_is_the_inverse_at_the_carried_positions(kd):
    wl = _wl(kd)
    crowd, osys, _, _ = make_pair(wl)
    crowd.qmc_sweep(3)
    stats0 = crowd.stats()
    crowd.qmc_recompute_inverse()
    assert crowd.stats() == stats0  # counters kept
    R = npy(crowd.positions())
    n = wl.n_elec // 2
    for spin in (0, 1):
        B = npy(crowd.inverse(spin))
        for w in range(wl.n_walkers):
            A = np.array([osys.spo_vgl(R[w, spin * n + i])[0] for i in range(n)])
            Bo = oracle.lu_inverse_transpose(A)[1]
            assert np.abs(B[w] - Bo).max() <= 1e-10 * np.abs(Bo).max()


@pytest.mark.parametrize("kd", [1, 8])
def test_trajectory_after_recompute_equals_fresh_crowd_and_oracle(kd):
    """sweeps, recompute, sweeps == a crowd created at the intermediate positions with the sweep index set; and the
    oracle restarted the same way (new OracleCrowd at those positions) makes the same decisions (fp64 tables)."""
    import torch
    wl = _wl(kd, cfg=22)
    a, osys, coefs, pos = make_pair(wl)
    a.qmc_sweep(2)
    a.qmc_recompute_inverse()
    R2 = npy(a.positions()).copy()
    b, _, _, _ = make_pair(wl, coefs=coefs, pos=R2)
    b.set_sweep_index(2)
    for spin in (0, 1):
        assert np.array_equal(npy(a.inverse(spin)), npy(b.inverse(spin)))
    a.qmc_sweep(2)
    b.qmc_sweep(2)
    assert np.array_equal(npy(a.positions()), npy(b.positions()))
    for spin in (0, 1):
        assert np.array_equal(npy(a.inverse(spin)), npy(b.inverse(spin)))
    oc = oracle.OracleCrowd(osys, R2)
    oc.set_sweep_index(2)
    oc.sweep(2)
    assert np.array_equal(npy(a.positions()), oc.positions())
    for spin in (0, 1):
        Bo = oc.inverse(spin)
        assert np.abs(npy(a.inverse(spin)) - Bo).max() <= 1e-10 * np.abs(Bo).max()
    del torch


def test_recompute_every_option_matches_manual_schedule():
    import paper_2209_14487_b200 as q
    wl = _wl(4, coef_dtype="f32", cfg=23)
    a, _, coefs, pos = make_pair(wl)
    b, _, _, _ = make_pair(wl, coefs=coefs, pos=pos)
    a.set_option(q.QMC_OPT_RECOMPUTE_EVERY, 2)
    a.qmc_sweep(3)
    a.qmc_sweep(2)  # schedule counted on the sweep index: recomputes after sweeps 2 and 4
    b.qmc_sweep(2)
    b.qmc_recompute_inverse()
    b.qmc_sweep(2)
    b.qmc_recompute_inverse()
    b.qmc_sweep(1)
    assert np.array_equal(npy(a.positions()), npy(b.positions()))
    for spin in (0, 1):
        assert np.array_equal(npy(a.inverse(spin)), npy(b.inverse(spin)))
    assert a.stats() == b.stats()
    with pytest.raises(q.QmcError):
        a.set_option(q.QMC_OPT_RECOMPUTE_EVERY, -1)


def test_recompute_removes_update_drift():
    """After many sweeps the carried inverse differs from the recomputed one by accumulated round-off; the recompute
    brings the residual |A B^T - I| back to the level of a fresh inversion (H8)."""
    wl = _wl(8, coef_dtype="f64", W=4, n_elec=48, cfg=24)
    crowd, osys, _, _ = make_pair(wl)
    crowd.qmc_sweep(30)
    R = npy(crowd.positions())
    n = wl.n_elec // 2
    A = [np.array([[osys.spo_vgl(R[w, s * n + i])[0] for i in range(n)] for w in range(wl.n_walkers)]) for s in (0, 1)]

    def residual():
        return max(np.abs(A[s][w] @ npy(crowd.inverse(s))[w].T - np.eye(n)).max()
                   for s in (0, 1) for w in range(wl.n_walkers))

    r_carried = residual()
    crowd.qmc_recompute_inverse()
    r_fresh = residual()
    assert r_fresh <= r_carried * 1.0 + 1e-15
    assert r_fresh < 1e-9


def test_recompute_refused_mid_move():
    import paper_2209_14487_b200 as q
    wl = _wl(4, cfg=25)
    crowd, _, _, _ = make_pair(wl)
    crowd.qmc_spo_vgl(0)
    with pytest.raises(q.QmcError):
        crowd.qmc_recompute_inverse()
