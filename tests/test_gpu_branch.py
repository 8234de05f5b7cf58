"""qmc_crowd_branch (Alg. 1 L13) against the oracle's oracle_crowd_branch."""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy

pytestmark = pytest.mark.gpu


def _i32(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).cuda()


@pytest.mark.parametrize("kd,coef_dtype", [(1, "f64"), (8, "f64"), (4, "f32")])
def test_branch_matches_oracle_and_trajectory_continues(kd, coef_dtype):
    wl = qi.small_workload(n_elec=32, grid=10, box=6.0, coef_dtype=coef_dtype, coef_dist="normal", n_walkers=7,
                           tau=0.02, delay_rank=kd, cfg=32)
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    src = np.array([0, 0, 2, 6, 2, 5, 6], dtype=np.int32)
    exact = coef_dtype == "f64"
    crowd.qmc_sweep(2)
    if exact:
        oc.sweep(2)
    R0 = npy(crowd.positions()).copy()
    B0 = [npy(crowd.inverse(s)).copy() for s in (0, 1)]
    C0 = [npy(x).copy() for x in crowd.caches()]
    assert crowd.qmc_crowd_branch(_i32(src)) == 3
    # the CUDA path: an exact gather of its own state
    assert np.array_equal(npy(crowd.positions()), R0[src])
    for s in (0, 1):
        assert np.array_equal(npy(crowd.inverse(s)), B0[s][src])
    for x0, x1 in zip(C0, crowd.caches()):
        assert np.array_equal(npy(x1), x0[src])
    if exact:   # against the oracle (fp64 tables: free-running trajectories agree bit for bit, D:A7)
        oc.branch(src)
        assert np.array_equal(npy(crowd.positions()), oc.positions())
        for s in (0, 1):
            Bo = oc.inverse(s)
            assert np.abs(npy(crowd.inverse(s)) - Bo).max() <= 1e-10 * np.abs(Bo).max()
        crowd.qmc_sweep(1)
        oc.sweep(1)
        assert np.array_equal(npy(crowd.positions()), oc.positions())
        for s in (0, 1):
            Bo = oc.inverse(s)
            assert np.abs(npy(crowd.inverse(s)) - Bo).max() <= 1e-10 * np.abs(Bo).max()
        # a copy leaves its source at the next move (the Philox stream belongs to the slot)
        assert not np.array_equal(npy(crowd.positions())[0], npy(crowd.positions())[1])


def test_invalid_maps_are_refused_and_change_nothing():
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=16, grid=8, box=5.0, coef_dtype="f32", coef_dist="normal", n_walkers=5, tau=0.02,
                           delay_rank=4, cfg=33)
    crowd, _, _, _ = make_pair(wl)
    crowd.qmc_sweep(1)
    R0 = npy(crowd.positions()).copy()
    B0 = npy(crowd.inverse(0)).copy()
    for bad in ([0, 1, 2, 3, 5], [0, 1, 2, 3, -1], [1, 2, 2, 3, 4]):   # out of range; a source that is itself replaced
        with pytest.raises(q.QmcError):
            crowd.qmc_crowd_branch(_i32(bad))
        assert np.array_equal(npy(crowd.positions()), R0)
        assert np.array_equal(npy(crowd.inverse(0)), B0)
    assert crowd.qmc_crowd_branch(_i32([0, 1, 2, 3, 4])) == 0
    crowd.qmc_sweep(1)   # the crowd is still usable (flags cleared)
    crowd.qmc_spo_vgl(0)
    with pytest.raises(q.QmcError):
        crowd.qmc_crowd_branch(_i32([0, 1, 2, 3, 4]))   # in the middle of a move


def test_branch_flushes_an_open_window_first():
    wl = qi.small_workload(n_elec=16, grid=8, box=5.0, coef_dtype="f64", coef_dist="normal", n_walkers=4, tau=0.02,
                           delay_rank=8, cfg=34)
    a, _, coefs, pos = make_pair(wl)
    b, _, _, _ = make_pair(wl, coefs=coefs, pos=pos)
    for c in (a, b):
        for k in range(3):
            c.qmc_spo_vgl(k)
            c.qmc_ratio_grad(k)
            c.qmc_accept_reject(k)
    b.qmc_flush_delayed()
    src = _i32([0, 0, 3, 3])
    a.qmc_crowd_branch(src)
    b.qmc_crowd_branch(src)
    for s in (0, 1):
        assert np.array_equal(npy(a.inverse(s)), npy(b.inverse(s)))
    assert np.array_equal(npy(a.positions()), npy(b.positions()))


def test_export_import_moves_walkers_between_crowds():
    """qmc_crowd_export_walkers / import_walkers (the load-balance message): walkers exported from crowd A
    and imported into crowd B carry their whole state; B then equals, slot by slot, the oracle crowd whose slots were
    filled by oracle_crowd_branch from the same sources (the two crowds here are two halves of one global crowd)."""
    import torch
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=32, grid=10, box=6.0, coef_dtype="f64", coef_dist="normal", n_walkers=8, tau=0.02,
                           delay_rank=8, cfg=35)
    full, osys, coefs, pos = make_pair(wl)                       # only for coefs / positions / oracle system
    full.close()
    A, _, _, _ = make_pair(wl, coefs=coefs, pos=pos[:4])                    # global walkers 0..3
    B, _, _, _ = make_pair(wl, coefs=coefs, pos=pos[4:], walker_id0=4)      # global walkers 4..7
    oc = oracle.OracleCrowd(osys, pos)                                      # all eight
    A.qmc_sweep(2)
    B.qmc_sweep(2)
    oc.sweep(2)
    nbytes = A.walker_state_bytes()
    n = wl.n_elec // 2
    assert nbytes == B.walker_state_bytes() == 2 * n * n * 8 + wl.n_elec * 4 * n * 8 + wl.n_elec * 24
    buf = A.qmc_crowd_export_walkers(_i32([3, 1]))
    assert tuple(buf.shape) == (2, nbytes)
    RA = npy(A.positions())
    # the tail of a packed state is the walker's positions, its head the spin-up inverse
    assert np.array_equal(buf[0, -wl.n_elec * 24:].cpu().numpy().view(np.float64).reshape(-1, 3), RA[3])
    assert np.array_equal(buf[1, :n * n * 8].cpu().numpy().view(np.float64).reshape(n, n), npy(A.inverse(0))[1])
    B.qmc_crowd_import_walkers(_i32([0, 2]), buf)                # global slots 4 and 6 <- global walkers 3 and 1
    oc.branch(np.array([0, 1, 2, 3, 3, 5, 1, 7], dtype=np.int32))
    assert np.array_equal(npy(B.positions()), oc.positions()[4:])
    for s in (0, 1):
        Bo = oc.inverse(s)[4:]
        assert np.abs(npy(B.inverse(s)) - Bo).max() <= 1e-10 * np.abs(Bo).max()
    A.qmc_sweep(1)
    B.qmc_sweep(1)
    oc.sweep(1)
    assert np.array_equal(npy(A.positions()), oc.positions()[:4])
    assert np.array_equal(npy(B.positions()), oc.positions()[4:])
    # refused: duplicate or out-of-range slots, nothing copied
    R0 = npy(B.positions()).copy()
    for bad in ([1, 1], [0, 4], [-1, 2]):
        with pytest.raises(q.QmcError):
            B.qmc_crowd_import_walkers(_i32(bad), buf)
        with pytest.raises(q.QmcError):
            B.qmc_crowd_export_walkers(_i32(bad))
    assert np.array_equal(npy(B.positions()), R0)
    B.qmc_sweep(1)   # still usable: marks and flags were cleared
    assert B.qmc_crowd_export_walkers(_i32([])).shape[0] == 0
    del torch
