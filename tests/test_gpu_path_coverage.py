"""Every kernel instantiation qmc_sweep can select at a BASELINE.json config, against the oracle.

Round-1 parity tests met the oracle only through `rank1_kernel<T,1>`, `sweep1_kernel` and `window_kernel<double,512>`.
This file closes the rest (fp64 tables: the free-running trajectory must equal `oracle.OracleCrowd` bit for bit --
positions and accepted counts -- and the inverses within 1e-10, P-free protocol of DESIGN.md section 3):

  * delay_rank = 1 with ns > 128: the per-move launch sequence of qmc_sweep (spline_vgl, ratio_accept, rank1<T,NV>,
    row_propose inside one captured graph) at NV = 3 (n = 132) and NV = 6 (n = 384, the benched instance), and once at
    n = 520 (ns = 528 > 512: rank1_generic_kernel, the unblocked inversion, the long-row branch of the window kernel);
  * the three threads-per-walker classes of the window kernel (512 / 256 / 128 threads for W <= 148 / <= 296 / more);
  * the benched class window_kernel<float,128> through the chain step calls <-> oracle (test_gpu_step_parity) and
    qmc_sweep <-> step calls at W = 300 on an fp32 table;
  * several crowds on several streams / host threads and sub-crowds on internal streams (Alg. 4, P:145-168;
    P:131 "a crowd is a sub-organization of the walker population"): the union equals ONE oracle crowd.
"""
import threading

import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import FreeRunningCheck, make_pair, npy, relerr, straddled_walkers

pytestmark = pytest.mark.gpu

def _free_running_vs_oracle(wl, sweeps, options=()):
    """qmc_sweep against the oracle's crowd, sweep by sweep, by the P-free protocol with classification
    (gpu_util.FreeRunningCheck): bit-exact up to a rounding straddle the oracle itself reports as undecided."""
    crowd, osys, _, pos = make_pair(wl)
    for opt, val in options:
        crowd.set_option(opt, val)
    oc = oracle.OracleCrowd(osys, pos)
    chk = FreeRunningCheck(wl.n_walkers, wl.tau)
    Rg_prev, Ro_prev = pos, pos
    for s in range(sweeps):
        _, log = oc.sweep(1, log=True)
        crowd.qmc_sweep(1)
        Rg, Ro = npy(crowd.positions()), oc.positions()
        chk.sweep(Rg_prev, Rg, Ro_prev, Ro, log[0])
        for spin in (0, 1):
            Bg, Bo = npy(crowd.inverse(spin)), oc.inverse(spin)
            for w in range(wl.n_walkers):
                assert relerr(Bg[w], Bo[w]) < chk.inverse_tol(w), (s, spin, w)
        Rg_prev, Ro_prev = Rg, Ro
    assert crowd.stats()["proposed"] == wl.n_walkers * wl.n_elec * sweeps
    return crowd, chk


# name: (n_elec, grid, W, delay_rank, sweeps, box or None, smallest fraction of the moves that must match bit for bit)
LARGE_CASES = {
    "n132_rank1_NV3_graph_path": (264, 10, 4, 1, 2, None, 0.5),
    "n384_rank1_NV6_benched_instance": (768, 8, 4, 1, 1, None, 0.25),
    "n520_rank1_generic_and_unblocked_inversion": (1040, 10, 2, 1, 1, None, 0.2),
    "n520_k16_long_rows": (1040, 10, 2, 16, 1, None, 0.2),
    "n96_k32_W300_window128": (192, 8, 300, 32, 1, None, 0.8),
    "n12_k8_W7_threads512": (24, 10, 7, 8, 3, 5.0, 0.99),
    "n12_k8_W200_threads256": (24, 10, 200, 8, 3, 5.0, 0.99),
    "n12_k8_W300_threads128": (24, 10, 300, 8, 3, 5.0, 0.99),
}
# several crowds / sub-crowds
CROWD_CASES = {
    "n24_k8_W11_subcrowds": (48, 10, 11, 8, 2, 6.0, 0.99),
    "n24_k8_W400_subcrowds": (48, 10, 400, 8, 2, 6.0, 0.99),
    "n24_k8_W12_crowds": (48, 10, 12, 8, 3, 6.0, 0.99),
    "n24_k8_W400_crowds": (48, 10, 400, 8, 3, 6.0, 0.99),
}


def case_workload(name):
    n_elec, grid, W, kd, sweeps, box, min_exact = {**LARGE_CASES, **CROWD_CASES}[name]
    wl = qi.small_workload(n_elec=n_elec, grid=grid, box=box or 0.9 * n_elec ** (1 / 3), coef_dtype="f64",
                           coef_dist="uniform", n_walkers=W, tau=0.02, delay_rank=kd, cfg=31)
    return wl, sweeps, min_exact


@pytest.mark.parametrize("name", list(LARGE_CASES))
def test_large_n_sweep_matches_oracle(name):
    """delay_rank = 1 and ns > SWEEP1_MAX_NS: four launches per move inside one captured graph (D:C5; P:73
    particle-by-particle, P:76 update on accept) at the rank1_kernel instances NV = 3, NV = 6 (the benched one) and the
    generic one (ns = 528 > 512, which also takes the unblocked inversion at create); delay_rank = 16 at ns = 528: the
    two-pass branch of block_rows_update; delay_rank = 32 with 300 walkers: the benched window class, 128 threads;
    n = 12 with 7 / 200 / 300 walkers: the three threads-per-walker classes of the window kernel (512 / 256 / 128; block
    sums depend on the class at the rounding level only, move.cuh)."""
    wl, sweeps, min_exact = case_workload(name)
    crowd, chk = _free_running_vs_oracle(wl, sweeps)
    assert chk.exact_moves >= min_exact * wl.n_walkers * wl.n_elec * sweeps, (chk.exact_moves, chk.departed.sum())
    if wl.delay_rank == 1:   # per move: spline, ratio + accept, rank-1, row / proposal of the next move
        assert crowd.launch_count() >= sweeps * 4 * wl.n_elec


@pytest.mark.parametrize("n_elec,kd", [(264, 1), (768, 1)])
def test_rank1_large_n_step_parity(n_elec, kd):
    """Moves at both ends of both spin blocks through the step calls at the large-n instances of rank1_kernel:
    the updated inverse against oracle.sm_update on the same B, phi, rho_D (1e-10)."""
    wl = qi.small_workload(n_elec=n_elec, grid=8, box=0.9 * n_elec ** (1 / 3), coef_dtype="f64",
                           coef_dist="uniform", n_walkers=3, tau=0.02, delay_rank=kd, cfg=32)
    crowd, osys, _, pos = make_pair(wl)
    n = n_elec // 2
    n_acc = 0
    for k in (0, 1, n - 1, n, n_elec - 1):
        spin, kk = divmod(k, n)
        B0 = npy(crowd.inverse(spin))
        phi, _, _ = (npy(x) for x in crowd.qmc_spo_vgl(k, want_outputs=True))
        crowd.qmc_ratio_grad(k)
        acc = npy(crowd.qmc_accept_reject(k))
        mv = {a: npy(b) for a, b in crowd.move().items()}
        B1 = npy(crowd.inverse(spin))
        for w in range(3):
            assert np.array_equal(mv["brow"][w], B0[w, kk])
            if acc[w]:
                n_acc += 1
                assert relerr(B1[w], oracle.sm_update(B0[w], kk, phi[w], mv["rho_d"][w])) < 1e-10
            else:
                assert np.array_equal(B1[w], B0[w])
    assert n_acc > 0


@pytest.mark.parametrize("n_elec,kd,sweeps,W,box", [(48, 8, 2, 300, 6.0), (192, 32, 1, 300, 6.0), (768, 32, 1, 5, 8.2),
                                                    (768, 32, 1, 160, 8.2)])
def test_sweep_equals_step_calls_in_the_benched_window_class(n_elec, kd, sweeps, W, box):
    """qmc_sweep through window_kernel<float,128> (W = 300, fp32 table) against the three step calls, which
    test_gpu_step_parity compares with the oracle call by call: identical positions and decisions, inverses 1e-10.
    n = 24: the generic instance; n = 96: a shape-specialised instance (window_kernel<float,128,96>, as cfgs 3-5 run);
    n = 384 with 5 / 160 walkers: the small-crowd instances of cfg 5, window_kernel<float,512,384> with the block rows in
    shared memory and window_kernel<float,256,384>."""
    wl = qi.small_workload(n_elec=n_elec, grid=10, box=box, coef_dtype="f32", coef_dist="normal", n_walkers=W,
                           tau=0.02, delay_rank=kd, cfg=36)
    a, _, _, R_prev = make_pair(wl)
    b, _, _, _ = make_pair(wl)
    n = n_elec // 2
    for s in range(sweeps):
        a.qmc_sweep(1)
        b.set_sweep_index(s)
        for k in range(n_elec):
            b.qmc_spo_vgl(k)
            b.qmc_ratio_grad(k)
            b.qmc_accept_reject(k)
            kk = k % n
            if (kk + 1) % kd == 0 or kk == n - 1:
                b.qmc_flush_delayed()
        Ra, Rb = npy(a.positions()), npy(b.positions())
        off = straddled_walkers(Ra, Rb, R_prev, cascade=n_elec >= 768)
        assert not off.any() or sweeps == 1   # a straddled walker is not followed into another sweep
        for spin in (0, 1):
            Ba, Bb = npy(a.inverse(spin)), npy(b.inverse(spin))
            assert relerr(Ba[~off], Bb[~off]) < 1e-10
            # (departed walkers: positions within 1e-5 after up to 700 more moves, amplified by the matrices' conditioning)
            assert not off.any() or relerr(Ba[off], Bb[off]) < (1e-3 if n_elec >= 768 else 1e-5)
        R_prev = Ra
    assert a.stats() == b.stats()


# name: (n_elec, grid, W, delay_rank, sweeps): shapes of the 32-row strip kernel (ns % 32 == 0, delay rank >= 16)
STRIP_CASES = {
    "n96_k32_three_strips_one_warp_ctas": (192, 8, 5, 32, 1),
    "n128_k32_four_strips_one_cta": (256, 8, 3, 32, 1),
    "n192_k16_two_window_blocks": (384, 9, 3, 16, 1),
    "n128_k64_two_sections": (256, 8, 3, 64, 1),
    "n384_k32_benched_instance": (768, 9, 3, 32, 1),
}


@pytest.mark.parametrize("rows", [32, 16])
@pytest.mark.parametrize("name", list(STRIP_CASES))
def test_both_strip_kernels_of_the_flush_match_the_oracle(name, rows):
    """QMC_OPT_STRIP_ROWS: flush32_kernel (32-row strips, window moves permuted inside the MMA tiles, padding k-steps
    skipped; what crowds of two waves and more run at cfgs 3-5) and flush_kernel (16-row strips; small crowds, fp32-stored
    inverses) forced in turn on crowds of a few walkers: qmc_sweep against the oracle's C6 flush, positions bit for bit
    up to a classified rounding straddle, inverses 1e-10; then the step-call flush (qmc_flush_delayed, the C / S^-T form
    of the finalize) of a teacher-forced window against oracle.delayed_flush."""
    import paper_2209_14487_b200 as q
    n_elec, grid, W, kd, sweeps = STRIP_CASES[name]
    wl = qi.small_workload(n_elec=n_elec, grid=grid, box=0.9 * n_elec ** (1 / 3), coef_dtype="f64", coef_dist="uniform",
                           n_walkers=W, tau=0.02, delay_rank=kd, cfg=37)
    crowd, chk = _free_running_vs_oracle(wl, sweeps, options=[(q.QMC_OPT_STRIP_ROWS, rows)])
    assert chk.exact_moves >= 0.2 * W * n_elec * sweeps
    # step calls: one window of the up spin, flushed by qmc_flush_delayed with the same kernel forced
    crowd.set_sweep_index(sweeps)
    B0 = npy(crowd.inverse(0))
    for k in range(min(kd, n_elec // 2)):
        crowd.qmc_spo_vgl(k)
        crowd.qmc_ratio_grad(k)
        crowd.qmc_accept_reject(k)
    m, rws, V, Cm, _ = (npy(x) for x in crowd.window())
    crowd.qmc_flush_delayed()
    B1 = npy(crowd.inverse(0))
    assert m.sum() > 0
    for w in range(W):
        mw = int(m[w])
        ref = oracle.delayed_flush(B0[w], rws[w, :mw], V[w, :mw], Cm[w, :mw]) if mw else B0[w]
        assert relerr(B1[w], ref) < 1e-10


def test_strip_rows_option_is_validated():
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=16, grid=8, box=4.0, coef_dtype="f64", n_walkers=2, delay_rank=4, cfg=38)
    crowd, _, _, _ = make_pair(wl)
    with pytest.raises(q.QmcError) as e:
        crowd.set_option(q.QMC_OPT_STRIP_ROWS, 8)
    assert e.value.status == q.QMC_ERR_INVALID_ARG
    crowd.set_option(q.QMC_OPT_STRIP_ROWS, 32)      # n = 8: the shape does not allow 32-row strips, 16 are used
    crowd.qmc_sweep(1)


# ---- several crowds / sub-crowds against ONE oracle crowd (fp64 tables) ----------------------------------------
def _union_vs_oracle(name, advance, positions, inverse):
    """advance(): one sweep of every crowd; positions() / inverse(spin): the union in global walker order.
    Compared with ONE oracle crowd of all walkers, sweep by sweep (gpu_util.FreeRunningCheck)."""
    wl, sweeps, min_exact = case_workload(name)
    coefs, pos = qi.make_coefs(wl), qi.make_positions(wl)
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, j2_a=wl.j2_a, j2_b=wl.j2_b,
                               tau=wl.tau, seed=wl.seed, delay_rank=wl.delay_rank)
    oc = oracle.OracleCrowd(osys, pos)
    chk = FreeRunningCheck(wl.n_walkers, wl.tau)
    Rg_prev, Ro_prev = pos, pos
    for s in range(sweeps):
        _, log = oc.sweep(1, log=True)
        advance()
        Rg, Ro = positions(), oc.positions()
        chk.sweep(Rg_prev, Rg, Ro_prev, Ro, log[0])
        for spin in (0, 1):
            Bg, Bo = inverse(spin), oc.inverse(spin)
            for w in range(wl.n_walkers):
                assert relerr(Bg[w], Bo[w]) < chk.inverse_tol(w), (s, spin, w)
        Rg_prev, Ro_prev = Rg, Ro
    assert chk.exact_moves >= min_exact * wl.n_walkers * wl.n_elec * sweeps, (chk.exact_moves, chk.departed.sum())


@pytest.mark.parametrize("name", ["n24_k8_W11_subcrowds", "n24_k8_W400_subcrowds"])
def test_sub_crowds_on_streams_equal_one_oracle_crowd(name):
    """QMC_OPT_SUBCROWDS (crowds on independent streams): every split equals the oracle's single crowd, and
    every split equals every other split bit for bit.  W = 400 would cross the threads-per-walker thresholds when split
    (sub-crowds of 200 / 134 / 100 walkers): the class is chosen from the whole crowd, so no reduction tree changes."""
    import paper_2209_14487_b200 as q
    wl, sweeps, _ = case_workload(name)
    ref = None
    for nsub, graph in ((1, 1), (2, 1), (3, 0), (4, 1)):
        c, _, _, _ = make_pair(wl)
        c.set_option(q.QMC_OPT_GRAPH, graph)
        c.set_option(q.QMC_OPT_SUBCROWDS, nsub)
        _union_vs_oracle(name, lambda: c.qmc_sweep(1), lambda: npy(c.positions()), lambda spin: npy(c.inverse(spin)))
        state = [npy(c.positions()), npy(c.inverse(0)), npy(c.inverse(1)), c.stats()]
        if ref is None:
            ref = state
        else:
            assert all(np.array_equal(a, b) for a, b in zip(state[:3], ref[:3])) and state[3] == ref[3]
        c.close()


@pytest.mark.parametrize("name,parts", [
    pytest.param("n24_k8_W12_crowds", [(0, 5), (5, 9), (9, 12)], id="W12_three_crowds"),
    pytest.param("n24_k8_W400_crowds", [(0, 100), (100, 300), (300, 400)], id="W400_crowds_in_different_thread_classes"),
])
def test_crowds_on_host_threads_equal_one_oracle_crowd(name, parts):
    """PAPER.md Alg. 4: several crowds, each advanced by its own host thread on its own stream, with
    global walker ids: their union is the oracle's one crowd, walker by walker (crowds of different sizes run
    different threads-per-walker classes of the window kernel: 512 / 256 / 128)."""
    import torch
    import paper_2209_14487_b200 as q
    wl, sweeps, _ = case_workload(name)
    coefs, pos = qi.make_coefs(wl), qi.make_positions(wl)
    dev = torch.device("cuda:0")
    tab = torch.from_numpy(coefs).to(dev)
    crowds = []
    for lo, hi in parts:
        st = torch.cuda.Stream(device=dev)
        crowds.append(q.Crowd(tab, wl.box, torch.from_numpy(pos[lo:hi].copy()).to(dev), tau=wl.tau,
                              delay_rank=wl.delay_rank, j2_a=wl.j2_a, j2_b=wl.j2_b, seed=wl.seed, walker_id0=lo, stream=st))

    def advance():
        def drive(c):
            torch.cuda.set_device(dev)
            c.qmc_sweep(1)
        th = [threading.Thread(target=drive, args=(c,)) for c in crowds]
        for t in th:
            t.start()
        for t in th:
            t.join()
        torch.cuda.synchronize()

    _union_vs_oracle(name, advance, lambda: np.concatenate([npy(c.positions()) for c in crowds]),
                     lambda spin: np.concatenate([npy(c.inverse(spin)) for c in crowds]))
    assert sum(c.stats()["proposed"] for c in crowds) == wl.n_walkers * wl.n_elec * sweeps
    for c in crowds:
        c.close()
