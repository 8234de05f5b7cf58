"""P-step parity: every exported call of the CUDA path against the
oracle on identical inputs, move by move through one full sweep, through the C ABI.

  qmc_spo_vgl       inverse row (window applied), G_k(R), proposal (bit-exact), orbitals
  qmc_ratio_grad    rho_D, rho_J, gradient, fed the GPU's own phi / inverse row
  qmc_accept_reject uniform and decision (bit-exact), positions, caches, Sherman-Morrison / append
  qmc_flush_delayed against the oracle's row-by-row flush of the same window

Tolerances (BASELINE.json north_star): 1e-10 relative on ratios / inverses (fp64), 1e-5 relative on
fp32 orbitals, 1e-12 on fp64 orbitals; integer / decision / position work bit-exact.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu

CASES = [
    # n_elec, grid, box, dtype, dist, W, tau, kd, orb_pad
    pytest.param(8, 16, 5.0, "f64", "uniform", 4, 0.02, 1, 0, id="cfg1_shape_sm"),
    pytest.param(24, 12, 6.0, "f32", "normal", 5, 0.02, 1, 1, id="n12_ragged_sm_padded_table"),
    pytest.param(64, 32, 10.0, "f32", "normal", 6, 0.01, 1, 0, id="cfg2_shape_sm"),
    pytest.param(40, 10, 7.0, "f32", "normal", 5, 0.02, 8, 0, id="n20_delay8_partial_last_window"),
    pytest.param(64, 16, 10.0, "f32", "normal", 4, 0.02, 16, 0, id="n32_delay16"),
    pytest.param(96, 12, 11.0, "f64", "uniform", 3, 0.02, 32, 0, id="n48_delay32_f64"),
    pytest.param(140, 9, 12.0, "f32", "normal", 3, 0.02, 64, 2, id="n70_delay64_two_strips"),
    pytest.param(12, 7, 4.0, "f64", "uniform", 2, 0.05, 3, 0, id="n6_delay3_tiny"),
]


@pytest.mark.parametrize("n_elec,grid,box,dtype,dist,W,tau,kd,orb_pad", CASES)
def test_one_sweep_step_by_step(n_elec, grid, box, dtype, dist, W, tau, kd, orb_pad):
    wl = qi.small_workload(n_elec=n_elec, grid=grid, box=box, coef_dtype=dtype, coef_dist=dist, n_walkers=W, tau=tau,
                           delay_rank=kd, cfg=7)
    crowd, osys, coefs, pos = make_pair(wl, orb_pad=orb_pad)
    N, n, M = n_elec, n_elec // 2, n_elec // 2
    tol_phi = 1e-5 if dtype == "f32" else 1e-12
    sweep = 3
    crowd.set_sweep_index(sweep)
    n_acc = n_rej = 0

    # create: caches and inverse against the oracle's definitions
    R = npy(crowd.positions())
    assert np.array_equal(R, pos)
    dc, d2c = (npy(x).astype(np.float64) for x in crowd.caches())
    for w in range(W):
        for s in range(2):
            A = np.array([osys.spo_vgl(R[w, s * n + i])[0] for i in range(n)])
            st, Bref, _, _ = oracle.lu_inverse_transpose(A)
            assert st == 0
            assert relerr(npy(crowd.inverse(s))[w], Bref) < (1e-4 if dtype == "f32" else 1e-9)
        for e in (0, N - 1):
            _, dref, d2ref = osys.spo_vgl(R[w, e])
            assert relerr(dc[w, e], dref) < tol_phi and relerr(d2c[w, e], d2ref) < tol_phi

    for k in range(N):
        spin, kk = divmod(k, n)
        R = npy(crowd.positions())
        B0 = npy(crowd.inverse(spin))
        dc, _ = (npy(x).astype(np.float64) for x in crowd.caches())
        if kd > 1:
            m, rows, V, Cm, Sinv = (npy(x) for x in crowd.window())
        # ---- qmc_spo_vgl
        phi, dphi, d2phi = (npy(x).astype(np.float64) for x in crowd.qmc_spo_vgl(k, want_outputs=True))
        mv = {a: npy(b) for a, b in crowd.move().items()}
        for w in range(W):
            if kd > 1:
                mw = int(m[w])
                b_ref = oracle.delayed_row(B0[w], rows[w, :mw], V[w, :mw], Cm[w, :mw], kk)
            else:
                b_ref = B0[w, kk]
            assert relerr(mv["brow"][w], b_ref) < 1e-10
            us_old, gj_old = osys.j2_usum_grad(R[w], k, R[w, k])
            g_ref = dc[w, k] @ mv["brow"][w] + gj_old
            assert relerr(mv["g_old"][w], g_ref) < 1e-10
            chi = oracle.rng_gauss3(wl.seed, w, k, sweep)
            delta, rnew, _ = oracle.move_propose(tau, R[w, k], mv["g_old"][w], chi)
            assert np.array_equal(mv["delta"][w], delta) and np.array_equal(mv["rnew"][w], rnew)
            p_ref, dp_ref, d2p_ref = osys.spo_vgl(mv["rnew"][w])
            assert relerr(phi[w], p_ref) < tol_phi
            assert relerr(dphi[w], dp_ref) < tol_phi
            assert relerr(d2phi[w], d2p_ref) < tol_phi
        # ---- qmc_ratio_grad
        ratio, grad = (npy(x) for x in crowd.qmc_ratio_grad(k))
        mv = {a: npy(b) for a, b in crowd.move().items()}
        for w in range(W):
            b = mv["brow"][w]
            rho_d = b @ phi[w]
            us_old, _ = osys.j2_usum_grad(R[w], k, R[w, k])
            us_new, gj_new = osys.j2_usum_grad(R[w], k, mv["rnew"][w])
            rho_j = np.exp(us_new - us_old)
            assert abs(mv["rho_d"][w] - rho_d) <= 1e-10 * max(abs(rho_d), np.abs(b * phi[w]).max())
            assert abs(mv["rho_j"][w] - rho_j) <= 1e-10 * rho_j
            assert abs(ratio[w] - mv["rho_d"][w] * mv["rho_j"][w]) <= 1e-14 * abs(ratio[w])
            g_ref = (dphi[w] @ b) / mv["rho_d"][w] + gj_new
            assert relerr(mv["g_new"][w], g_ref) < 1e-10
            assert np.array_equal(grad[w], mv["g_new"][w])
        # ---- qmc_accept_reject
        acc = npy(crowd.qmc_accept_reject(k))
        mv = {a: npy(b) for a, b in crowd.move().items()}
        R2 = npy(crowd.positions())
        B1 = npy(crowd.inverse(spin))
        dc2, d2c2 = (npy(x).astype(np.float64) for x in crowd.caches())
        if kd > 1:
            m2, rows2, V2, C2, Sinv2 = (npy(x) for x in crowd.window())
        for w in range(W):
            u = oracle.rng_uniform(wl.seed, w, k, sweep)
            assert mv["u"][w] == u
            a_ref, p_ref = oracle.move_accept(tau, mv["delta"][w], mv["g_old"][w], mv["g_new"][w], mv["rho_d"][w],
                                              mv["rho_j"][w], u)
            assert abs(mv["p"][w] - p_ref) <= 1e-12 * abs(p_ref)
            if abs(u - p_ref) > 1e-12 * p_ref:
                assert bool(acc[w]) == a_ref
            Rexp = R[w].copy()
            if acc[w]:
                n_acc += 1
                Rexp[k] = mv["rnew"][w]
                assert np.array_equal(dc2[w, k], dphi[w]) and np.array_equal(d2c2[w, k], d2phi[w])
            else:
                n_rej += 1
                assert np.array_equal(dc2[w, k], dc[w, k])
            assert np.array_equal(R2[w], Rexp)
            if kd == 1:
                if acc[w]:
                    assert relerr(B1[w], oracle.sm_update(B0[w], kk, phi[w], mv["rho_d"][w])) < 1e-10
                else:
                    assert np.array_equal(B1[w], B0[w])
            else:
                assert np.array_equal(B1[w], B0[w])          # B0 untouched until the flush
                mw = int(m[w])
                assert int(m2[w]) == mw + int(acc[w])
                if acc[w]:
                    assert rows2[w, mw] == kk
                    assert np.array_equal(V2[w, mw], phi[w]) and np.array_equal(C2[w, mw], B0[w, kk])
                    S = V2[w, :mw + 1] @ C2[w, :mw + 1].T
                    assert relerr(Sinv2[w, :mw + 1, :mw + 1], np.linalg.inv(S)) < 1e-9
        # ---- qmc_flush_delayed on the schedule of D:C6
        if kd > 1 and ((kk + 1) % kd == 0 or kk == n - 1):
            crowd.qmc_flush_delayed()
            B2 = npy(crowd.inverse(spin))
            for w in range(W):
                mw = int(m2[w])
                ref = oracle.delayed_flush(B0[w], rows2[w, :mw], V2[w, :mw], C2[w, :mw]) if mw else B0[w]
                assert relerr(B2[w], ref) < 1e-10
            assert int(npy(crowd.window()[0]).max()) == 0
            crowd.qmc_flush_delayed()                          # idempotent when empty
            assert np.array_equal(npy(crowd.inverse(spin)), B2)
    assert n_acc > 0 and n_rej > 0, (n_acc, n_rej)
    st = crowd.stats()
    assert st["proposed"] == W * N and st["accepted"] == n_acc


def test_teacher_forced_position_and_state_errors():
    import paper_2209_14487_b200 as q
    import torch
    wl = qi.small_workload(n_elec=16, grid=8, box=5.0, coef_dtype="f32", coef_dist="normal", n_walkers=3, tau=0.02,
                           delay_rank=4, cfg=8)
    crowd, osys, _, pos = make_pair(wl)
    rn = pos[:, 5] + np.array([0.3, -0.2, 0.1])
    phi, dphi, d2phi = (npy(x) for x in crowd.qmc_spo_vgl(5, rnew=torch.from_numpy(rn).cuda(), want_outputs=True))
    mv = crowd.move()
    assert np.array_equal(npy(mv["rnew"]), rn) and np.array_equal(npy(mv["delta"]), rn - pos[:, 5])
    for w in range(3):
        assert relerr(phi[w], osys.spo_vgl(rn[w])[0]) < 1e-5
    with pytest.raises(q.QmcError) as e:
        crowd.qmc_accept_reject(5)            # ratio_grad skipped
    assert e.value.status == q.QMC_ERR_STATE
    with pytest.raises(q.QmcError):
        crowd.qmc_ratio_grad(4)               # wrong electron
    crowd.qmc_ratio_grad(5)
    crowd.qmc_accept_reject(5)
    with pytest.raises(q.QmcError) as e:
        crowd.qmc_spo_vgl(5)                  # same electron twice in one window
    assert e.value.status == q.QMC_ERR_STATE
    with pytest.raises(q.QmcError):
        crowd.qmc_spo_vgl(9)                  # other spin block before the flush
    for k in (0, 1, 2):
        crowd.qmc_spo_vgl(k); crowd.qmc_ratio_grad(k); crowd.qmc_accept_reject(k)
    with pytest.raises(q.QmcError):
        crowd.qmc_spo_vgl(3)                  # window of 4 proposals is full
    crowd.qmc_flush_delayed()
    crowd.qmc_spo_vgl(3)


def test_create_rejects_bad_arguments():
    import paper_2209_14487_b200 as q
    import torch
    wl = qi.small_workload(n_elec=8, grid=6, coef_dtype="f32", coef_dist="normal", n_walkers=2, cfg=9)
    coefs = torch.from_numpy(qi.make_coefs(wl)).cuda()
    pos = torch.from_numpy(qi.make_positions(wl)).cuda()
    with pytest.raises(q.QmcError):
        q.Crowd(coefs, wl.box, pos, tau=-1.0)
    with pytest.raises(q.QmcError):
        q.Crowd(coefs, wl.box, pos, tau=0.01, delay_rank=65)
    # singular start: two electrons of one spin at the same point (D:A16)
    bad = pos.clone()
    bad[1, 1] = bad[1, 0]
    with pytest.raises(q.QmcError) as e:
        q.Crowd(coefs, wl.box, bad, tau=0.01)
    assert e.value.status == q.QMC_ERR_SINGULAR
