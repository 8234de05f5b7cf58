"""Host-side logic that the GPU tests and bench.py rely on, checked on CPU: the classification of rounding straddles
(reading A7) used by the free-running parity protocol, bench.py's byte counts and its --gpus N launch."""
import json
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import FreeRunningCheck, straddle_flags

ROOT = Path(__file__).resolve().parent.parent


def _oracle_sweep(n_elec=16, W=6, kd=4, seed=3):
    wl = qi.small_workload(n_elec=n_elec, grid=8, box=4.0, coef_dtype="f64", coef_dist="uniform", n_walkers=W,
                           tau=0.02, delay_rank=kd, cfg=91, seed=seed)
    coefs, pos = qi.make_coefs(wl), qi.make_positions(wl)
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, tau=wl.tau, seed=wl.seed, delay_rank=kd)
    oc = oracle.OracleCrowd(osys, pos)
    _, log = oc.sweep(1, log=True)
    return wl, pos, oc.positions(), log[0]


def test_straddle_flags_follow_the_margin_and_the_size_of_the_displacement():
    wl, _, _, log = _oracle_sweep()
    rec = log.copy()
    rec["disp_margin"] = 0.25                         # far from a rounding boundary: never flagged at 1e-10
    assert not straddle_flags(rec, wl.tau).any()
    rec["disp_margin"] = 1e-9                         # closer than any fp64 implementation can resolve G: always
    assert straddle_flags(rec, wl.tau).all()
    # a displacement component that cancels to ~1e-6 has an fp32 ulp of ~1e-13: a 1e-10 error of G decides its rounding
    rec["disp_margin"] = 0.25
    rec["delta"][0, 0] = (1e-6, 0.1, -0.1)
    f = straddle_flags(rec, wl.tau)
    assert f[0, 0] and f.sum() == 1
    # the looser the tolerance on G, the more moves are undecided
    assert straddle_flags(log, wl.tau, 1e-8).sum() >= straddle_flags(log, wl.tau, 1e-10).sum()


def test_free_running_check_accepts_a_flagged_straddle_and_rejects_anything_else():
    wl, R0, R1, log = _oracle_sweep()
    W, N = log.shape
    chk = FreeRunningCheck(W, wl.tau)
    chk.sweep(R0, R1, R0, R1, log)                    # identical trajectories: every move exact
    assert chk.exact_moves == W * N and not chk.departed.any()
    acc = np.argwhere(log["accepted"] == 1)
    w, k = (int(x) for x in acc[len(acc) // 2])
    ulp = float(np.spacing(np.float32(abs(log[w, k]["delta"][0]))))
    Rg = R1.copy()
    Rg[w, k, 0] += ulp                                # the other rounding of that displacement
    with pytest.raises(AssertionError, match="rules out a straddle"):
        FreeRunningCheck(W, wl.tau).sweep(R0, Rg, R0, R1, log)
    rec = log.copy()
    rec["disp_margin"][w, k] = 1e-9                   # ... unless the oracle reports that rounding as undecided
    chk = FreeRunningCheck(W, wl.tau)
    chk.sweep(R0, Rg, R0, R1, rec)
    assert chk.departed[w] and chk.departed.sum() == 1 and chk.exact_moves == (W - 1) * N + k
    assert chk.inverse_tol(w) > chk.inverse_tol((w + 1) % W)
    # a walker that wanders off, or decides differently, fails even after it has departed
    Rbad = Rg.copy()
    Rbad[w, k] += 1e-3
    with pytest.raises(AssertionError):
        FreeRunningCheck(W, wl.tau).sweep(R0, Rbad, R0, R1, rec)
    rej = np.argwhere(log["accepted"] == 0)
    if len(rej):
        w2, k2 = (int(x) for x in rej[0])
        Rdec = R1.copy()
        Rdec[w2, k2] += 1e-9                          # "moved" where the oracle rejected
        with pytest.raises(AssertionError):
            FreeRunningCheck(W, wl.tau).sweep(R0, Rdec, R0, R1, log)


def _bench():
    sys.path.insert(0, str(ROOT))
    import bench
    return bench


def test_bench_byte_counts_at_cfg5():
    """bench.py's algorithmic bytes against the figures DESIGN.md section 6 derives by hand for cfg 5, k = 32."""
    b = _bench()
    wl = qi.WORKLOADS[5]
    a = b.algorithmic(wl, 4096, 32, 0.85, 4)
    per_walker = a["window"]["bytes"] / 4096
    # gather 3.146 MB + block rows 0.197 + V, Cp 0.167 + gradient caches 0.314 + positions 0.018 = 3.84 MB
    assert abs(per_walker - 3.842e6) < 0.01e6, per_walker
    assert abs(a["window"]["l2_plus_hbm_bytes"] / 4096 - 6.335e6) < 0.01e6
    assert a["flush"]["bytes"] == 4096 * 16 * 384 * 384
    assert abs(a["flush"]["flops"] / 4096 - (4 * 384 * 384 * 27.2 + 2 * 384 * 27.2 ** 2)) < 1.0
    assert a["rank1"]["bytes"] == pytest.approx(0.85 * 4096 * 16 * 384 * 384)
    assert abs(b.FP64_DMMA_CEILING_TFLOPS - 37.2) < 0.1
    assert len(b.csrc_digest()) == 16


def test_bench_gpus_2_starts_two_ranks_with_disjoint_walkers():
    """`python bench.py --gpus 2` outside torchrun starts the two ranks itself (the driver's own torchrun command
    line); --plan-only keeps it off the GPU: the ranks rendezvous over gloo and report their walker ranges."""
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--plan-only", "--walkers", "4096"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak"
    r0, r1 = line["ranks"]
    assert (r0["rank"], r0["walker_id0"], r0["walkers"]) == (0, 0, 4096)
    assert (r1["rank"], r1["walker_id0"], r1["walkers"]) == (1, 4096, 4096)
    assert r0["pid"] != r1["pid"]
