"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (config 5:
768 electrons, 80^3 fp32 table, delayed rank 32, crowd of 4096 walkers), on SAMPLED walkers the oracle can
compute one by one, plus properties that hold at any size.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu

W = 4096
SAMPLE = (0, 777, 4095)


@pytest.fixture(scope="module")
def full():
    import torch
    if torch.cuda.get_device_properties(0).total_memory < 80e9:
        pytest.skip("needs ~45 GB of device memory")
    wl = qi.WORKLOADS[5]
    crowd, osys, coefs, pos = make_pair(wl, n_walkers=W)
    yield wl, crowd, osys, pos
    crowd.close()


def test_full_size_sweep_then_sampled_step_parity(full):
    import torch
    wl, crowd, osys, pos = full
    N, n, kd, tau = wl.n_elec, wl.n, wl.delay_rank, wl.tau
    crowd.qmc_sweep(1)
    st = crowd.stats()
    assert st["proposed"] == W * N and st["flushes"] == 2 * (n // kd)
    alpha = st["accepted"] / st["proposed"]
    assert 0.5 < alpha < 0.99
    R1 = npy(crowd.positions())
    moved = np.any(R1 != pos, axis=2)
    assert moved.sum() == st["accepted"]            # every accepted move changed exactly one electron once
    assert np.isfinite(R1).all()

    # ---- P-inv on sampled walkers: the carried inverse inverts the Slater matrix of its own orbitals
    idx = torch.tensor(SAMPLE, device="cuda")
    for spin in (0, 1):
        Bg = npy(crowd.inverse(spin)[idx])
        A = np.zeros((len(SAMPLE), n, n))
        for i in range(n):
            e = spin * n + i
            phi, _, _ = crowd.qmc_spo_vgl(e, rnew=torch.from_numpy(np.ascontiguousarray(R1[:, e])).cuda(), want_outputs=True)
            A[:, i] = npy(phi[idx]).astype(np.float64)
            if i % 97 == 0:                          # the spline itself against the oracle, a few electrons
                for s, w in enumerate(SAMPLE):
                    assert relerr(A[s, i], osys.spo_vgl(R1[w, e])[0]) < 1e-5
        for s in range(len(SAMPLE)):
            res = np.abs(A[s] @ Bg[s].T - np.eye(n)).max()
            assert res < 1e-8, res

    # ---- teacher-free step calls into the second sweep, checked on the sampled walkers mid-window
    crowd.set_sweep_index(1)
    for k in range(0, 11):
        crowd.qmc_spo_vgl(k)
        crowd.qmc_ratio_grad(k)
        crowd.qmc_accept_reject(k)
    k, spin, kk = 11, 0, 11
    B0 = npy(crowd.inverse(0)[idx])
    m, rows, V, Cm, _ = crowd.window()
    m, rows, V, Cm = npy(m[idx]), npy(rows[idx]), npy(V[idx]), npy(Cm[idx])
    dc = npy(crowd.caches()[0][idx, k]).astype(np.float64)
    Rk = npy(crowd.positions()[idx])
    phi, dphi, d2phi = (npy(x[idx]).astype(np.float64) for x in crowd.qmc_spo_vgl(k, want_outputs=True))
    mv = {a: npy(b[idx]) for a, b in crowd.move().items()}
    crowd.qmc_ratio_grad(k)
    mv2 = {a: npy(b[idx]) for a, b in crowd.move().items()}
    acc = npy(crowd.qmc_accept_reject(k)[idx])
    mv3 = {a: npy(b[idx]) for a, b in crowd.move().items()}
    assert 0 < m.min() and m.max() <= 11
    for s, w in enumerate(SAMPLE):
        mw = int(m[s])
        b_ref = oracle.delayed_row(B0[s], rows[s, :mw], V[s, :mw], Cm[s, :mw], kk)
        assert relerr(mv["brow"][s], b_ref) < 1e-10
        us_old, gj_old = osys.j2_usum_grad(Rk[s], k, Rk[s, k])
        assert relerr(mv["g_old"][s], dc[s] @ mv["brow"][s] + gj_old) < 1e-10
        delta, rnew, _ = oracle.move_propose(tau, Rk[s, k], mv["g_old"][s], oracle.rng_gauss3(wl.seed, w, k, 1))
        assert np.array_equal(mv["delta"][s], delta) and np.array_equal(mv["rnew"][s], rnew)
        p_ref, dp_ref, d2p_ref = osys.spo_vgl(rnew)
        assert relerr(phi[s], p_ref) < 1e-5 and relerr(dphi[s], dp_ref) < 1e-5 and relerr(d2phi[s], d2p_ref) < 1e-5
        b = mv["brow"][s]
        rho_d = b @ phi[s]
        assert abs(mv2["rho_d"][s] - rho_d) <= 1e-10 * max(abs(rho_d), np.abs(b * phi[s]).max())
        us_new, gj_new = osys.j2_usum_grad(Rk[s], k, rnew)
        assert abs(mv2["rho_j"][s] - np.exp(us_new - us_old)) <= 1e-10 * mv2["rho_j"][s]
        assert relerr(mv2["g_new"][s], (dphi[s] @ b) / mv2["rho_d"][s] + gj_new) < 1e-10
        u = oracle.rng_uniform(wl.seed, w, k, 1)
        a_ref, p_acc = oracle.move_accept(tau, mv3["delta"][s], mv3["g_old"][s], mv3["g_new"][s], mv3["rho_d"][s],
                                          mv3["rho_j"][s], u)
        assert mv3["u"][s] == u and bool(acc[s]) == a_ref

    # ---- finish the window and flush: sampled walkers against the oracle's row-by-row flush
    for k in range(12, 32):
        crowd.qmc_spo_vgl(k)
        crowd.qmc_ratio_grad(k)
        crowd.qmc_accept_reject(k)
    m, rows, V, Cm, _ = crowd.window()
    m, rows, V, Cm = npy(m[idx]), npy(rows[idx]), npy(V[idx]), npy(Cm[idx])
    all_m = npy(crowd.window()[0])
    assert all_m.max() <= kd and abs(all_m.mean() / kd - alpha) < 0.05      # ragged fill ~ acceptance
    crowd.qmc_flush_delayed()
    B1 = npy(crowd.inverse(0)[idx])
    for s in range(len(SAMPLE)):
        mw = int(m[s])
        assert relerr(B1[s], oracle.delayed_flush(B0[s], rows[s, :mw], V[s, :mw], Cm[s, :mw])) < 1e-10
