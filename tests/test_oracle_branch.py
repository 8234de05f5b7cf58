"""Pins for the oracle's branching data movement (oracle_crowd_branch; Alg. 1 L13).

The operation is a gather of whole walker states, so the pins are about completeness and consistency of what is
moved: the copied inverse must be the inverse of the Slater matrix at the copied positions, and the copied caches must
be those of the copied positions (a crowd re-created there makes the same moves)."""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi


def _setup(kd=4, W=6, cfg=31):
    wl = qi.small_workload(n_elec=16, grid=8, box=5.0, coef_dtype="f64", coef_dist="normal", n_walkers=W, tau=0.02,
                           delay_rank=kd, cfg=cfg)
    coefs = qi.make_coefs(wl)
    pos = qi.make_positions(wl, W)
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, j2_a=wl.j2_a, j2_b=wl.j2_b, tau=wl.tau,
                               seed=wl.seed, delay_rank=kd)
    return wl, osys, pos


def test_identity_map_changes_nothing():
    wl, osys, pos = _setup()
    a, b = oracle.OracleCrowd(osys, pos), oracle.OracleCrowd(osys, pos)
    a.sweep(2)
    b.sweep(2)
    a.branch(np.arange(wl.n_walkers))
    a.sweep(1)
    b.sweep(1)
    assert np.array_equal(a.positions(), b.positions())
    for spin in (0, 1):
        assert np.array_equal(a.inverse(spin), b.inverse(spin))


@pytest.mark.parametrize("kd", [1, 4])
def test_branched_state_is_a_consistent_walker(kd):
    wl, osys, pos = _setup(kd=kd)
    W, n = wl.n_walkers, wl.n_elec // 2
    c = oracle.OracleCrowd(osys, pos)
    c.sweep(2)
    R0 = c.positions()
    B0 = [c.inverse(s) for s in (0, 1)]
    src = np.array([0, 0, 2, 5, 2, 5], dtype=np.int32)
    c.branch(src)
    R1 = c.positions()
    for w in range(W):
        assert np.array_equal(R1[w], R0[src[w]])
    for spin in (0, 1):
        B1 = c.inverse(spin)
        for w in range(W):
            assert np.array_equal(B1[w], B0[spin][src[w]])
            # the inverse that arrived belongs to the positions that arrived
            A = np.array([osys.spo_vgl(R1[w, spin * n + i])[0] for i in range(n)])
            assert np.abs(A @ B1[w].T - np.eye(n)).max() < 1e-9
    # the caches that arrived belong to those positions too: a crowd created at R1 (fresh caches) moves identically
    f = oracle.OracleCrowd(osys, R1)
    f.set_sweep_index(2)
    c.sweep(1)
    f.sweep(1)
    assert np.array_equal(c.positions(), f.positions())
    # random streams stay with the slot: a copy and its source part ways
    assert not np.array_equal(c.positions()[0], c.positions()[1])


def test_general_gather_and_bad_entries():
    wl, osys, pos = _setup()
    c = oracle.OracleCrowd(osys, pos)
    R0 = c.positions()
    c.branch(np.array([1, 2, 3, 4, 5, 0]))  # the oracle is the plain definition: any map in range is a gather
    assert np.array_equal(c.positions(), R0[[1, 2, 3, 4, 5, 0]])
    with pytest.raises(ValueError):
        c.branch(np.array([0, 1, 2, 3, 4, 6]))
    with pytest.raises(ValueError):
        c.branch(np.array([0, 1, 2, 3, 4, -1]))
