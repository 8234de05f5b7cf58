"""qmc_sweep with a delayed update (window kernel + triangular finalize + DMMA strip, R5) against the
oracle's C6 delayed update, free-running.

With an fp64 coefficient table both sides compute the same real numbers to ~1e-13; the displacement is quantised to
fp32 (reading A7), so positions and accept/reject decisions must come out bit-identical and the inverses within 1e-10
(P-free protocol extended to delay_rank > 1).  Shapes cover: the window equal to the whole spin block, a partial last
window, a delay rank larger than the block, padded ranks (3 -> 8), rank 64, a single walker, and ragged n (ns padding).
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_elec,kd,W,sweeps", [
    pytest.param(8, 4, 4, 6, id="cfg1_shape_window_is_block"),
    pytest.param(24, 8, 5, 3, id="n12_k8_partial_last_window"),
    pytest.param(12, 8, 3, 4, id="n6_rank_larger_than_block"),
    pytest.param(40, 3, 4, 2, id="n20_k3_padded_rank"),
    pytest.param(140, 64, 2, 1, id="n70_k64_two_windows"),
    pytest.param(36, 16, 1, 3, id="single_walker"),
])
def test_window_sweep_matches_oracle_fp64_table(n_elec, kd, W, sweeps):
    wl = qi.small_workload(n_elec=n_elec, grid=12, box=6.0, coef_dtype="f64", coef_dist="uniform", n_walkers=W,
                           tau=0.02, delay_rank=kd, cfg=21)
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    total = 0
    for s in range(sweeps):
        acc, log = oc.sweep(1, log=True)
        total += acc
        crowd.qmc_sweep(1)
        assert np.array_equal(npy(crowd.positions()), oc.positions()), f"positions differ after sweep {s}"
        for spin in (0, 1):
            assert relerr(npy(crowd.inverse(spin)), oc.inverse(spin)) < 1e-10
        assert log["disp_margin"].min() > 1e-7, "an fp32 rounding straddle is plausible: inspect (reading A7)"
    st = crowd.stats()
    assert st["accepted"] == total and st["proposed"] == W * n_elec * sweeps
    n = n_elec // 2
    windows_per_block = -(-n // kd)
    assert st["flushes"] == 2 * windows_per_block * sweeps


def test_window_sweep_then_step_calls_share_state():
    """A sweep leaves an empty window and a fully updated inverse: step calls continue from it, and a sweep
    after step calls (which leave an open window) flushes first."""
    wl = qi.small_workload(n_elec=32, grid=10, box=6.0, coef_dtype="f64", coef_dist="uniform", n_walkers=3, tau=0.02,
                           delay_rank=8, cfg=22)
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    oc.sweep(1)
    crowd.qmc_sweep(1)
    crowd.set_sweep_index(1)
    # three step moves of sweep 1, window left open
    _, log = oc.sweep(1, log=True)
    for k in range(3):
        crowd.qmc_spo_vgl(k)
        crowd.qmc_ratio_grad(k)
        acc = npy(crowd.qmc_accept_reject(k))
        assert np.array_equal(acc.astype(np.int32), log[0, :, k]["accepted"])
    crowd.qmc_flush_delayed()
    assert crowd.stats()["proposed"] == 3 * 32 + 3 * 3
