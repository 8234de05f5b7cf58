"""Free-running parity of qmc_sweep (DESIGN.md "Parity protocols" P-free and P-inv).

P-free: BASELINE.json config 1 (all fp64): accept/reject decisions and positions bit-exact against
the oracle over the 10 configured sweeps, ratios and inverses within 1e-10 relative.
P-inv: fp32-table shapes, where trajectories legitimately diverge (reading A8): the inverse the
CUDA path carries after free-running sweeps must still invert the Slater matrix rebuilt from its
own orbitals at the final positions, as well as the oracle's does; acceptance fractions agree.
Also: graph replay == plain launches, crowd splitting leaves trajectories unchanged,
qmc_sweep_host == set_positions + qmc_sweep.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu


def test_cfg1_trajectory_bit_exact():
    wl = qi.WORKLOADS[1]
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    total_acc = 0
    for s in range(wl.sweeps):
        acc, log = oc.sweep(1, log=True)
        total_acc += acc
        crowd.qmc_sweep(1)
        assert np.array_equal(npy(crowd.positions()), oc.positions()), f"positions differ after sweep {s}"
        for spin in (0, 1):
            assert relerr(npy(crowd.inverse(spin)), oc.inverse(spin)) < 1e-10
        assert log["disp_margin"].min() > 1e-7, "an fp32 rounding straddle is plausible: inspect (reading A7)"
    st = crowd.stats()
    assert st["accepted"] == total_acc and st["proposed"] == wl.n_walkers * wl.n_elec * wl.sweeps
    assert 0.2 < total_acc / st["proposed"] < 0.999


def test_cfg1_step_api_matches_oracle_log():
    """Same trajectory through the three step calls; every logged quantity of every move."""
    wl = qi.WORKLOADS[1]
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    for s in range(3):
        _, log = oc.sweep(1, log=True)
        crowd.set_sweep_index(s)
        for k in range(wl.n_elec):
            crowd.qmc_spo_vgl(k)
            crowd.qmc_ratio_grad(k)
            acc = npy(crowd.qmc_accept_reject(k))
            mv = {a: npy(b) for a, b in crowd.move().items()}
            rec = log[0, :, k]
            assert np.array_equal(acc.astype(np.int32), rec["accepted"])
            assert np.array_equal(mv["rnew"], rec["rnew"]) and np.array_equal(mv["delta"], rec["delta"])
            assert np.array_equal(mv["u"], rec["u"])
            for name in ("rho_d", "rho_j", "p"):
                assert np.all(np.abs(mv[name] - rec[name]) <= 1e-10 * np.abs(rec[name])), name
            assert relerr(mv["g_old"], rec["g_old"]) < 1e-10 and relerr(mv["g_new"], rec["g_new"]) < 1e-10
    assert np.array_equal(npy(crowd.positions()), oc.positions())


@pytest.mark.parametrize("kd", [1, 8])
def test_graph_replay_equals_plain_launches_and_crowd_split(kd):
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=32, grid=12, box=6.0, coef_dtype="f32", coef_dist="normal", n_walkers=6, tau=0.02,
                           delay_rank=kd, cfg=11)
    a, _, coefs, pos = make_pair(wl)
    b, _, _, _ = make_pair(wl)
    b.set_option(q.QMC_OPT_GRAPH, 0)
    a.qmc_sweep(3)
    b.qmc_sweep(3)
    Ra, Rb = npy(a.positions()), npy(b.positions())
    assert np.array_equal(Ra, Rb)
    for spin in (0, 1):
        assert np.array_equal(npy(a.inverse(spin)), npy(b.inverse(spin)))
    assert a.stats() == b.stats()
    assert a.launch_count() == b.launch_count()
    # two crowds of 2 and 4 walkers with global walker ids == one crowd of 6 (reading A6)
    c1, _, _, _ = make_pair(wl, pos=pos[:2].copy(), walker_id0=0)
    c2, _, _, _ = make_pair(wl, pos=pos[2:].copy(), walker_id0=2)
    c1.qmc_sweep(3)
    c2.qmc_sweep(3)
    assert np.array_equal(np.concatenate([npy(c1.positions()), npy(c2.positions())]), Ra)
    assert not np.array_equal(Ra, pos)


@pytest.mark.parametrize("n_elec,kd", [(48, 8), (40, 16), (24, 1)])
def test_sweep_equals_the_three_step_calls(n_elec, kd):
    """qmc_sweep against the three step calls on the same crowd.  delay_rank = 1: same device functions,
    bit-identical.  delay_rank > 1: qmc_sweep runs the window kernel in the eager-block form of the delayed
    update (R5), the step calls the bordered-S^-1 form of C6: the two agree to rounding (1e-13),
    which the fp32 quantisation of the displacement (A7) turns into identical positions and decisions;
    the inverses agree to 1e-10."""
    wl = qi.small_workload(n_elec=n_elec, grid=10, box=6.0, coef_dtype="f32", coef_dist="normal", n_walkers=7,
                           tau=0.02, delay_rank=kd, cfg=14)
    a, _, _, _ = make_pair(wl)
    b, _, _, _ = make_pair(wl)
    n = n_elec // 2
    for s in range(2):
        a.qmc_sweep(1)
        b.set_sweep_index(s)
        for k in range(n_elec):
            b.qmc_spo_vgl(k)
            b.qmc_ratio_grad(k)
            b.qmc_accept_reject(k)
            kk = k % n
            if kd > 1 and ((kk + 1) % kd == 0 or kk == n - 1):
                b.qmc_flush_delayed()
        assert np.array_equal(npy(a.positions()), npy(b.positions()))
        for spin in (0, 1):
            if kd == 1:
                assert np.array_equal(npy(a.inverse(spin)), npy(b.inverse(spin)))
            else:
                assert relerr(npy(a.inverse(spin)), npy(b.inverse(spin))) < 1e-10
    assert a.stats() == b.stats()


def _gpu_slater(crowd, R, spin):
    """A[w][i][j] = phi_j(r_{spin n + i}) from the CUDA spline at given positions (teacher-forced)."""
    import torch
    n = crowd.n
    rows = []
    for i in range(n):
        phi, _, _ = crowd.qmc_spo_vgl(spin * n + i, rnew=torch.from_numpy(np.ascontiguousarray(R[:, spin * n + i])).cuda(),
                                      want_outputs=True)
        rows.append(npy(phi).astype(np.float64))
    return np.stack(rows, axis=1)


@pytest.mark.parametrize("n_elec,grid,box,kd,W,sweeps", [
    pytest.param(64, 32, 10.0, 1, 24, 4, id="cfg2_shape_rank1"),
    pytest.param(192, 16, 14.0, 32, 8, 2, id="cfg3_shape_delay32"),
    pytest.param(96, 16, 11.0, 16, 12, 3, id="n48_delay16"),
])
def test_free_running_inverse_residual_and_acceptance(n_elec, grid, box, kd, W, sweeps):
    wl = qi.small_workload(n_elec=n_elec, grid=grid, box=box, coef_dtype="f32", coef_dist="normal", n_walkers=W,
                           tau=0.01, delay_rank=kd, cfg=12)
    crowd, osys, _, pos = make_pair(wl)
    oc = oracle.OracleCrowd(osys, pos)
    acc_o = oc.sweep(sweeps)
    crowd.qmc_sweep(sweeps)
    st = crowd.stats()
    n_prop = W * n_elec * sweeps
    fo, fg = acc_o / n_prop, st["accepted"] / n_prop
    se = np.sqrt(max(fo * (1 - fo), 1e-4) / n_prop)
    assert abs(fo - fg) < 3 * np.sqrt(2) * se + 1e-3, (fo, fg)
    Rg, Ro = npy(crowd.positions()), oc.positions()
    n = n_elec // 2
    for spin in (0, 1):
        Bg = npy(crowd.inverse(spin))
        Ag = _gpu_slater(crowd, Rg, spin)
        Bo = oc.inverse(spin)
        res_g = max(np.abs(Ag[w] @ Bg[w].T - np.eye(n)).max() for w in range(W))
        res_o = 0.0
        for w in range(W):
            Ao = np.array([osys.spo_vgl(Ro[w, spin * n + i])[0] for i in range(n)])
            res_o = max(res_o, np.abs(Ao @ Bo[w].T - np.eye(n)).max())
        assert res_g <= 10 * res_o + 1e-9, (res_g, res_o)


def test_sweep_host_equals_set_positions_plus_sweep():
    import torch
    wl = qi.small_workload(n_elec=32, grid=12, box=6.0, coef_dtype="f32", coef_dist="normal", n_walkers=5, tau=0.02,
                           delay_rank=4, cfg=13)
    a, _, _, pos = make_pair(wl)
    b, _, _, _ = make_pair(wl)
    pos2 = pos + 0.05
    host = torch.from_numpy(pos2.copy()).pin_memory()
    stats = a.qmc_sweep_host(host, 2)
    b.set_positions(torch.from_numpy(pos2).cuda())
    b.qmc_sweep(2)
    assert np.array_equal(host.numpy(), npy(b.positions()))
    assert np.array_equal(npy(a.positions()), host.numpy())
    assert stats == b.stats()


def test_sub_crowds_on_separate_streams_do_not_change_results():
    """QMC_OPT_SUBCROWDS: qmc_sweep advances the crowd as independent sub-crowds on separate streams;
    walkers are independent and counters are global, so every split gives bit-identical state."""
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=48, grid=10, box=6.0, coef_dtype="f32", coef_dist="normal", n_walkers=11, tau=0.02,
                           delay_rank=8, cfg=15)
    ref, _, _, _ = make_pair(wl)
    ref.qmc_sweep(2)
    for nsub, graph in ((2, 1), (3, 0), (4, 1)):
        c, _, _, _ = make_pair(wl)
        c.set_option(q.QMC_OPT_GRAPH, graph)
        c.set_option(q.QMC_OPT_SUBCROWDS, nsub)
        c.qmc_sweep(1)
        c.qmc_sweep(1)
        assert np.array_equal(npy(c.positions()), npy(ref.positions()))
        for spin in (0, 1):
            assert np.array_equal(npy(c.inverse(spin)), npy(ref.inverse(spin)))
        assert c.stats() == ref.stats()


def test_crowds_on_host_threads_and_streams_equal_one_crowd():
    """PAPER.md Alg. 4: several crowds, each advanced by its own host thread on its own stream.
    With global walker ids the union of the crowds is the one big crowd, walker by walker (same threads-per-walker
    class here, so bit-identical)."""
    import threading
    import torch
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=48, grid=10, box=6.0, coef_dtype="f32", coef_dist="normal", n_walkers=12, tau=0.02,
                           delay_rank=8, cfg=16)
    ref, _, coefs, pos = make_pair(wl)
    ref.qmc_sweep(3)
    dev = torch.device("cuda:0")
    tab = torch.from_numpy(coefs).to(dev)
    parts = [(0, 5), (5, 9), (9, 12)]
    crowds = []
    for lo, hi in parts:
        st = torch.cuda.Stream(device=dev)
        crowds.append(q.Crowd(tab, wl.box, torch.from_numpy(pos[lo:hi].copy()).to(dev), tau=wl.tau, delay_rank=8,
                              j2_a=wl.j2_a, j2_b=wl.j2_b, seed=wl.seed, walker_id0=lo, stream=st))

    def drive(c):
        torch.cuda.set_device(dev)
        for _ in range(3):
            c.qmc_sweep(1)

    th = [threading.Thread(target=drive, args=(c,)) for c in crowds]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    Rref = npy(ref.positions())
    tot = {"proposed": 0, "accepted": 0}
    for (lo, hi), c in zip(parts, crowds):
        assert np.array_equal(npy(c.positions()), Rref[lo:hi])
        for spin in (0, 1):
            assert np.array_equal(npy(c.inverse(spin)), npy(ref.inverse(spin))[lo:hi])
        s = c.stats()
        tot["proposed"] += s["proposed"]
        tot["accepted"] += s["accepted"]
    assert tot["proposed"] == ref.stats()["proposed"] and tot["accepted"] == ref.stats()["accepted"]
