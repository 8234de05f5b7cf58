"""qmc_kinetic_energy against the oracle, teacher-forced: the oracle gets the CUDA path's
own positions and inverses, so only the energy kernel is compared.  fp64 tables: 1e-10 (everything is fp64 on both
sides); fp32 tables: the cached grad / lap phi are fp32, so 1e-5 of the largest per-electron term (north_star's
orbital tolerance)."""
import numpy as np
import pytest

import qmc_inputs as qi
from gpu_util import make_pair, npy

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_elec,kd,dtype,tol", [
    (8, 1, "f64", 1e-10), (24, 8, "f64", 1e-10), (40, 16, "f32", 1e-5), (140, 32, "f32", 1e-5),
])
def test_kinetic_energy_matches_oracle_after_sweeps(n_elec, kd, dtype, tol):
    wl = qi.small_workload(n_elec=n_elec, grid=10, box=6.0, coef_dtype=dtype,
                           coef_dist="uniform" if dtype == "f64" else "normal", n_walkers=5, tau=0.02, delay_rank=kd, cfg=61)
    crowd, osys, _, _ = make_pair(wl)
    for sweeps in (0, 2):
        if sweeps:
            crowd.qmc_sweep(sweeps)
        ekin, e = crowd.qmc_kinetic_energy(per_electron=True)
        ekin, e = npy(ekin), npy(e)
        R, Bu, Bd = npy(crowd.positions()), npy(crowd.inverse(0)), npy(crowd.inverse(1))
        for w in range(wl.n_walkers):
            t_ref, e_ref = osys.kinetic_energy(R[w], Bu[w], Bd[w])
            scale = np.abs(e_ref).max()
            assert np.abs(e[w] - e_ref).max() <= tol * scale, (w, np.abs(e[w] - e_ref).max() / scale)
            assert abs(ekin[w] - t_ref) <= tol * scale * np.sqrt(n_elec) + 1e-12 * abs(t_ref)
            assert abs(ekin[w] - e[w].sum()) <= 1e-12 * max(1.0, np.abs(e[w]).sum())


def test_kinetic_energy_needs_a_flushed_window_and_changes_no_state():
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=16, grid=8, box=5.0, coef_dtype="f64", coef_dist="uniform", n_walkers=3, tau=0.02,
                           delay_rank=4, cfg=62)
    crowd, _, _, _ = make_pair(wl)
    before = (npy(crowd.positions()).copy(), npy(crowd.inverse(0)).copy())
    a = npy(crowd.qmc_kinetic_energy())
    b = npy(crowd.qmc_kinetic_energy())
    assert np.array_equal(a, b)
    assert np.array_equal(npy(crowd.positions()), before[0]) and np.array_equal(npy(crowd.inverse(0)), before[1])
    crowd.qmc_spo_vgl(0); crowd.qmc_ratio_grad(0); crowd.qmc_accept_reject(0)
    with pytest.raises(q.QmcError) as ei:
        crowd.qmc_kinetic_energy()
    assert ei.value.status == q.QMC_ERR_STATE
    crowd.qmc_flush_delayed()
    crowd.qmc_kinetic_energy()
