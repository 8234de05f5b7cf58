"""Pins for the oracle's move and whole sweep (pins T8/T9).

The paper prints no worked trajectory (T9: "parity unpinned by the paper"), so the sweep is
pinned through what every logged move must satisfy when re-derived by brute force from the
positions alone: rho = Psi(R')/Psi(R) with Psi from LAPACK determinants of freshly built
Slater matrices times the full Jastrow pair sum; G = finite-difference gradient of ln|Psi|;
the inverse after the sweep = inverse recomputed from the final positions; and the chain
samples |Psi|^2 (histogram test), which a wrong sign or a dropped term in the acceptance
rule breaks.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi


def build(wl, delay_rank=None, coefs=None, **kw):
    coefs = qi.make_coefs(wl) if coefs is None else coefs
    s = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, j2_a=kw.get("j2_a", wl.j2_a),
                            j2_b=wl.j2_b, tau=kw.get("tau", wl.tau), seed=wl.seed,
                            delay_rank=wl.delay_rank if delay_rank is None else delay_rank)
    return s


def slater(s, R, spin):
    n = s.n
    return np.array([s.spo_vgl(R[spin * n + i])[0] for i in range(n)])


def log_abs_psi(s, R):
    sg, la = 1.0, s.j2_logpsi(R)
    for spin in (0, 1):
        sgn, l = np.linalg.slogdet(slater(s, R, spin))
        sg *= sgn
        la += l
    return sg, la


def fd_grad(s, R, k, eps=1e-6):
    g = np.zeros(3)
    for c in range(3):
        Rp, Rm = R.copy(), R.copy()
        Rp[k, c] += eps
        Rm[k, c] -= eps
        g[c] = (log_abs_psi(s, Rp)[1] - log_abs_psi(s, Rm)[1]) / (2 * eps)
    return g


# ---------------------------------------------------------------- the two halves of a move
def test_propose_hand_values():
    tau = 0.02
    d, rn, margin = oracle.move_propose(tau, [1.0, 2.0, 3.0], [1.0, 0.0, -2.0], [0.0, 1.0, 0.5])
    expect = np.array([np.float32(0.02), np.float32(np.sqrt(0.02)), np.float32(-0.04 + 0.5 * np.sqrt(0.02))],
                      dtype=np.float64)
    assert np.array_equal(d, expect)
    assert np.array_equal(rn, np.array([1.0, 2.0, 3.0]) + expect)
    assert np.array_equal(d.astype(np.float32).astype(np.float64), d)   # fp32-valued (A7)
    assert 0 <= margin <= 0.5


def test_accept_rule_symmetry_and_limits():
    tau = 0.05
    rng = np.random.default_rng(0)
    for _ in range(20):
        delta, g0, g1 = rng.normal(0, 0.2, 3), rng.normal(0, 1, 3), rng.normal(0, 1, 3)
        rho_d, rho_j = rng.normal(0, 1.5), np.exp(rng.normal(0, 0.3))
        _, p_f = oracle.move_accept(tau, delta, g0, g1, rho_d, rho_j, 0.5)
        _, p_b = oracle.move_accept(tau, -delta, g1, g0, 1 / rho_d, 1 / rho_j, 0.5)
        assert abs(p_f * p_b - 1) < 1e-12          # detailed balance: T(R->R')p_f = T(R'->R) with p_b = 1/p_f
    # no drift, symmetric proposal: p = rho^2 exactly
    acc, p = oracle.move_accept(tau, [0.1, 0, 0], [0, 0, 0], [0, 0, 0], -0.5, 1.0, 0.2)
    assert p == 0.25 and acc
    acc, _ = oracle.move_accept(tau, [0.1, 0, 0], [0, 0, 0], [0, 0, 0], -0.5, 1.0, 0.25)
    assert not acc                                  # strict u < p
    # pure drift step Delta = tau*G with G' = -G... forward exponent 0, backward -|(-tau G) - tau G'|^2/2tau
    acc, p = oracle.move_accept(tau, [tau * 2.0, 0, 0], [2.0, 0, 0], [1.0, 0, 0], 1.0, 1.0, 0.0)
    assert abs(p - np.exp(-((3 * tau) ** 2) / (2 * tau))) < 1e-15
    # degenerate inputs reject
    assert not oracle.move_accept(tau, [0, 0, 0], [0, 0, 0], [0, 0, 0], 0.0, 1.0, 0.0)[0]
    assert not oracle.move_accept(tau, [0, 0, 0], [0, 0, 0], [np.nan, 0, 0], 1.0, 1.0, 0.0)[0]
    assert not oracle.move_accept(tau, [0, 0, 0], [0, 0, 0], [0, 0, 0], np.inf, 1.0, 0.0)[0]


# ---------------------------------------------------------------- whole sweeps, re-derived
@pytest.mark.parametrize("delay_rank", [1, 2, 3, 4])
def test_every_logged_move_rederived_by_brute_force(delay_rank):
    wl = qi.small_workload(n_elec=8, grid=6, box=3.0, n_walkers=2, tau=0.05)
    s = build(wl, delay_rank=delay_rank)
    R0 = qi.make_positions(wl)
    crowd = oracle.OracleCrowd(s, R0)
    n_sw = 2
    acc, log = crowd.sweep(n_sw, log=True)
    assert acc == int(log["accepted"].sum())
    n_checked_acc = 0
    for w in range(wl.n_walkers):
        R = R0[w].copy()
        for it in range(n_sw):
            for k in range(wl.n_elec):
                rec = log[it, w, k]
                # proposal re-derived: same counter-based normals, drift from FD of ln|Psi|
                chi = oracle.rng_gauss3(wl.seed, w, k, it)
                np.testing.assert_allclose(rec["g_old"], fd_grad(s, R, k), rtol=2e-5, atol=2e-6)
                d, rn, _ = oracle.move_propose(wl.tau, R[k], rec["g_old"], chi)
                assert np.array_equal(d, rec["delta"]) and np.array_equal(rn, rec["rnew"])
                R2 = R.copy()
                R2[k] = rec["rnew"]
                sg0, l0 = log_abs_psi(s, R)
                sg1, l1 = log_abs_psi(s, R2)
                rho = rec["rho_d"] * rec["rho_j"]
                assert np.sign(rho) == sg0 * sg1
                assert abs(np.log(abs(rho)) - (l1 - l0)) < 1e-9
                assert abs(np.log(rec["rho_j"]) - (s.j2_logpsi(R2) - s.j2_logpsi(R))) < 1e-12
                np.testing.assert_allclose(rec["g_new"], fd_grad(s, R2, k), rtol=2e-5, atol=2e-6)
                assert rec["u"] == oracle.rng_uniform(wl.seed, w, k, it)
                acc_k, p = oracle.move_accept(wl.tau, rec["delta"], rec["g_old"], rec["g_new"], rec["rho_d"],
                                              rec["rho_j"], rec["u"])
                assert p == rec["p"] and int(acc_k) == rec["accepted"] == int(rec["u"] < rec["p"])
                if rec["accepted"]:
                    R = R2
                    n_checked_acc += 1
        np.testing.assert_array_equal(crowd.positions()[w], R)
        for spin in (0, 1):
            np.testing.assert_allclose(crowd.inverse(spin)[w], np.linalg.inv(slater(s, R, spin)).T,
                                       rtol=1e-7, atol=1e-8)
    assert 0 < n_checked_acc < n_sw * wl.n_walkers * wl.n_elec     # both branches exercised


def test_delay_rank_does_not_change_the_trajectory():
    # exact algebra: rank-1 and delayed chains make the same decisions (tiny system, fp64)
    wl = qi.small_workload(n_elec=8, grid=6, box=3.0, n_walkers=3, tau=0.05)
    R0 = qi.make_positions(wl)
    outs = []
    for kd in (1, 2, 4):
        c = oracle.OracleCrowd(build(wl, delay_rank=kd), R0)
        c.sweep(3)
        outs.append(c.positions())
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_crowd_partition_invariance_and_crowd_of_one():
    # a crowd is just a batch; walkers are independent (counter-based RNG, A6)
    wl = qi.WORKLOADS[1]
    s = build(wl)
    R0 = qi.make_positions(wl)
    whole = oracle.OracleCrowd(s, R0)
    whole.sweep(2)
    a = oracle.OracleCrowd(s, R0[:1], walker_id0=0)
    b = oracle.OracleCrowd(s, R0[1:], walker_id0=1)
    a.sweep(2)
    b.sweep(2)
    assert np.array_equal(whole.positions(), np.concatenate([a.positions(), b.positions()]))


def test_reject_changes_nothing_and_sweep_index_selects_the_stream():
    wl = qi.WORKLOADS[1]
    s = build(wl)
    R0 = qi.make_positions(wl)
    c = oracle.OracleCrowd(s, R0)
    _, log = c.sweep(1, log=True)
    pos = c.positions()
    for w in range(wl.n_walkers):
        for k in range(wl.n_elec):
            if not log[0, w, k]["accepted"]:
                assert np.array_equal(pos[w, k], R0[w, k])      # PAPER.md:76 "rejecting ... zero cost"
            else:
                assert np.array_equal(pos[w, k], log[0, w, k]["rnew"])
    c2 = oracle.OracleCrowd(s, R0)
    c2.set_sweep_index(5)
    _, log2 = c2.sweep(1, log=True)
    assert not np.array_equal(log2["u"], log["u"])
    assert log2[0, 0, 0]["u"] == oracle.rng_uniform(wl.seed, 0, 0, 5)


def test_constant_orbital_no_jastrow_accepts_everything():
    # T8: n = 1 per spin, constant orbital, a = 0 -> rho = 1, G = 0, p = 1
    wl = qi.small_workload(n_elec=2, grid=4, box=2.0, n_walkers=4, tau=0.1)
    coefs = np.full((4, 4, 4, 1), 1.7)
    s = build(wl, coefs=coefs, j2_a=0.0)
    c = oracle.OracleCrowd(s, qi.make_positions(wl))
    acc, log = c.sweep(5, log=True)
    assert acc == 5 * 4 * 2
    np.testing.assert_allclose(log["p"], 1.0, atol=1e-12)
    assert np.max(np.abs(log["g_old"])) < 1e-12 and np.max(np.abs(log["rho_d"] - 1)) < 1e-13


def test_acceptance_tends_to_one_as_tau_vanishes():
    wl = qi.small_workload(n_elec=8, grid=6, box=3.0, n_walkers=8)
    R0 = qi.make_positions(wl)
    rates = []
    for tau in (0.2, 1e-2, 1e-4):
        c = oracle.OracleCrowd(build(wl, tau=tau), R0)
        rates.append(c.sweep(4) / (4 * 8 * 8))
    assert rates[0] < rates[1] <= rates[2] and rates[2] > 0.97


def test_chain_samples_phi_squared():
    # One electron per spin in a positive orbital phi(x) = spline of 2 + cos(2 pi i/Ng), no Jastrow:
    # each electron samples phi^2.  A wrong sign / missing factor in the Green's function ratio or a
    # missing square on rho shifts the histogram by far more than the tolerance.
    ng, L, W, tau = 8, 4.0, 256, 0.3
    wl = qi.small_workload(n_elec=2, grid=ng, box=L, n_walkers=W, tau=tau)
    coefs = np.zeros((ng, ng, ng, 1))
    coefs += (2.0 + np.cos(2 * np.pi * np.arange(ng) / ng)).reshape(ng, 1, 1, 1)
    s = build(wl, coefs=coefs, j2_a=0.0)
    c = oracle.OracleCrowd(s, qi.make_positions(wl))
    c.sweep(60)
    nb = 8
    hist = np.zeros(nb)
    n_samp = 0
    acc = 0
    for _ in range(150):
        acc += c.sweep(2)
        x = np.mod(c.positions()[:, :, 0].ravel(), L)
        hist += np.histogram(x, bins=nb, range=(0, L))[0]
        n_samp += x.size
    rate = acc / (150 * 2 * W * 2)
    assert 0.3 < rate < 0.99
    xs = (np.arange(nb * 200) + 0.5) * (L / (nb * 200))
    dens = np.array([s.spo_vgl([x, 0.1, 0.2])[0][0] ** 2 for x in xs]).reshape(nb, 200).sum(axis=1)
    expect = dens / dens.sum()
    got = hist / n_samp
    # ~76800 samples, autocorrelation of a few sweeps: 3-sigma is ~0.01 absolute; bins span 0.03..0.27
    assert np.max(np.abs(got - expect)) < 0.012, (got, expect)
