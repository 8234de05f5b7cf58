"""Degenerate and boundary cases of the C ABI on the GPU: the smallest system (one electron per spin), zero sweeps,
a delay rank the block does not fill, negative / far-away coordinates (periodic wrap of the stencil), argument
and state errors.  Every free-running case is compared with the oracle (fp64 tables: bit-identical positions)."""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kd", [1, 2, 8])
def test_one_electron_per_spin(kd):
    wl = qi.small_workload(n_elec=2, grid=6, box=3.0, coef_dtype="f64", coef_dist="uniform", n_walkers=6, tau=0.05,
                           delay_rank=kd, cfg=71)
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    acc = oc.sweep(5)
    crowd.qmc_sweep(5)
    assert np.array_equal(npy(crowd.positions()), oc.positions())
    assert crowd.stats()["accepted"] == acc
    for spin in (0, 1):
        assert relerr(npy(crowd.inverse(spin)), oc.inverse(spin)) < 1e-10
    ek = npy(crowd.qmc_kinetic_energy())
    R, Bu, Bd = oc.positions(), oc.inverse(0), oc.inverse(1)
    for w in range(6):
        t_ref, e_ref = osys.kinetic_energy(R[w], Bu[w], Bd[w])
        assert abs(ek[w] - t_ref) <= 1e-9 * max(1.0, np.abs(e_ref).max())


def test_zero_sweeps_and_idempotent_flush():
    wl = qi.small_workload(n_elec=12, grid=6, box=4.0, coef_dtype="f32", coef_dist="normal", n_walkers=2, delay_rank=4, cfg=72)
    crowd, _, _, pos = make_pair(wl)
    crowd.qmc_sweep(0)
    crowd.qmc_flush_delayed()
    crowd.qmc_flush_delayed()
    assert np.array_equal(npy(crowd.positions()), pos)
    assert crowd.stats() == {"proposed": 0, "accepted": 0, "flushes": 0}


def test_positions_far_outside_the_box_wrap_periodically():
    """Positions are never wrapped (reading C1 / A11): a crowd started at R and one started at R + (7, -5, 3) L see
    the same orbitals and minimum-image distances; with an fp64 table the trajectories are translates of each other
    up to the rounding of the shifted coordinates, so decisions agree and displacements are bit-identical."""
    wl = qi.small_workload(n_elec=8, grid=8, box=4.0, coef_dtype="f64", coef_dist="uniform", n_walkers=4, tau=0.02,
                           delay_rank=4, cfg=73)
    a, osys, _, pos = make_pair(wl)
    shift = np.array([7.0, -5.0, 3.0]) * wl.box
    b, _, _, _ = make_pair(wl, pos=pos + shift)
    oc = oracle.OracleCrowd(osys, pos + shift)
    for _ in range(2):
        a.qmc_sweep(1)
        b.qmc_sweep(1)
        oc.sweep(1)
        assert np.array_equal(npy(b.positions()), oc.positions())
    assert a.stats()["accepted"] == b.stats()["accepted"]
    assert np.abs((npy(b.positions()) - shift) - npy(a.positions())).max() < 1e-9


def test_argument_and_state_errors():
    import torch
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=8, grid=6, box=4.0, coef_dtype="f64", coef_dist="uniform", n_walkers=2, delay_rank=2, cfg=74)
    crowd, _, coefs, pos = make_pair(wl)
    with pytest.raises(q.QmcError) as e:
        crowd.qmc_ratio_grad(0)                       # no qmc_spo_vgl before it
    assert e.value.status == q.QMC_ERR_STATE
    with pytest.raises(q.QmcError) as e:
        crowd.qmc_spo_vgl(99)
    assert e.value.status == q.QMC_ERR_INVALID_ARG
    crowd.qmc_spo_vgl(0); crowd.qmc_ratio_grad(0); crowd.qmc_accept_reject(0)
    crowd.qmc_spo_vgl(1); crowd.qmc_ratio_grad(1); crowd.qmc_accept_reject(1)
    with pytest.raises(q.QmcError) as e:
        crowd.qmc_spo_vgl(2)                          # window of rank 2 is full: flush is due
    assert e.value.status == q.QMC_ERR_STATE
    crowd.qmc_flush_delayed()
    crowd.qmc_spo_vgl(2)
    with pytest.raises(q.QmcError) as e:
        crowd.qmc_sweep(1)                            # in the middle of a move
    assert e.value.status == q.QMC_ERR_STATE
    with pytest.raises(q.QmcError) as e:              # odd electron count
        q.Crowd(torch.from_numpy(coefs).cuda(), wl.box, torch.from_numpy(pos[:, :7].copy()).cuda(), tau=0.01)
    assert e.value.status == q.QMC_ERR_INVALID_ARG


@pytest.mark.parametrize("tau,kd,n_elec,rows", [(1e-6, 8, 80, 0), (1e-6, 1, 80, 0), (0.6, 8, 80, 0), (0.6, 1, 80, 0),
                                                 (0.6, 32, 80, 0), (1e-6, 32, 128, 32), (0.6, 32, 128, 32),
                                                 (0.6, 16, 128, 32), (0.6, 64, 256, 32)])
def test_acceptance_extremes(tau, kd, n_elec, rows):
    """Nearly every move accepted (full windows, m = k) and nearly every move rejected (windows with m = 0 or 1, flushes
    that have nothing to do): the free-running trajectory still equals the oracle's on an fp64 table.  rows = 32: the
    32-row strip kernel forced (QMC_OPT_STRIP_ROWS), whose GEMM 2 skips k-steps by the number of accepted moves -- windows
    with m = 0, 1..4, 5..8 and full ones all occur."""
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=n_elec, grid=12, box=7.0 * (n_elec / 80) ** (1 / 3), coef_dtype="f64", coef_dist="uniform",
                           n_walkers=5, tau=tau, delay_rank=kd, cfg=76)
    crowd, osys, _, pos = make_pair(wl)
    if rows:
        crowd.set_option(q.QMC_OPT_STRIP_ROWS, rows)
    oc = oracle.OracleCrowd(osys, pos)
    acc = oc.sweep(2)
    crowd.qmc_sweep(2)
    frac = acc / (2 * 5 * n_elec)
    assert frac > 0.98 if tau < 1e-3 else frac < 0.5, frac
    assert crowd.stats()["accepted"] == acc
    assert np.array_equal(npy(crowd.positions()), oc.positions())
    for spin in (0, 1):
        assert relerr(npy(crowd.inverse(spin)), oc.inverse(spin)) < 1e-10


@pytest.mark.parametrize("kd", [1, 8])
def test_anisotropic_grid_and_box(kd):
    """Different grid sizes and box lengths per axis (the C ABI takes grid[3], box[3]): a transposed axis anywhere in the
    stencil offsets, the weights or the minimum image would move the trajectory off the oracle's."""
    import torch
    import paper_2209_14487_b200 as q
    n_elec, W, grid, box = 24, 4, (6, 9, 11), (3.0, 4.5, 5.5)
    rng = np.random.default_rng(77)
    coefs = rng.uniform(-1.0, 1.0, size=grid + (n_elec // 2,))
    pos = rng.uniform(0.0, 1.0, size=(W, n_elec, 3)) * np.array(box)
    osys = oracle.OracleSystem(n_elec, grid, box, coefs, j2_a=0.5, j2_b=1.0, tau=0.02, seed=5, delay_rank=kd)
    oc = oracle.OracleCrowd(osys, pos)
    crowd = q.Crowd(torch.from_numpy(coefs).cuda(), box, torch.from_numpy(pos).cuda(), tau=0.02, delay_rank=kd,
                    j2_a=0.5, j2_b=1.0, seed=5)
    acc = oc.sweep(3)
    crowd.qmc_sweep(3)
    assert crowd.stats()["accepted"] == acc
    assert np.array_equal(npy(crowd.positions()), oc.positions())
    for spin in (0, 1):
        assert relerr(npy(crowd.inverse(spin)), oc.inverse(spin)) < 1e-10
    phi, dphi, d2phi = (npy(x) for x in crowd.qmc_spo_vgl(0, want_outputs=True))
    mv = npy(crowd.move()["rnew"])
    for w in range(W):
        p, dp, d2p = osys.spo_vgl(mv[w])
        assert relerr(phi[w], p) < 1e-12 and relerr(dphi[w], dp) < 1e-12 and relerr(d2phi[w], d2p) < 1e-12


def test_crowd_size_limit_is_checked_at_create():
    """Several kernels put W (or 2 W) in gridDim.y (<= 65535): a crowd larger than 32767 walkers is refused with a clear
    message instead of failing at a launch; a population that large is split into crowds."""
    import torch
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=8, grid=4, box=3.0, coef_dtype="f32", coef_dist="normal", n_walkers=4, cfg=75)
    coefs = torch.from_numpy(qi.make_coefs(wl)).cuda()
    pos = torch.rand((32768, 8, 3), dtype=torch.float64, device="cuda") * 3.0
    with pytest.raises(q.QmcError) as e:
        q.Crowd(coefs, wl.box, pos, tau=0.01)
    assert e.value.status == q.QMC_ERR_INVALID_ARG and "32767" in str(e.value)
    c = q.Crowd(coefs, wl.box, pos[:32767].contiguous(), tau=0.01)
    c.qmc_sweep(1)
    assert c.stats()["proposed"] == 32767 * 8
