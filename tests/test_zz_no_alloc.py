"""qmc_spo_vgl_static (include/qmc_crowd.h): the orbital evaluation with its internal result buffer in a file-scope
static device array instead of a caller workspace -- for callers that cannot allocate device memory.

Checked against the existing path (qmc_spo_vgl on a crowd, teacher-forced to the same positions) within the tolerance the
step-parity tests use for orbitals (tests/test_gpu_step_parity.py: 1e-5 relative for an fp32 table, 1e-12 for fp64), on
two calls in a row that share the array (the second one smaller, so the array still holds the first call's results
beyond it), and against the oracle's plain definition (D:C1).  Collected last (pytest runs files in name order): the
run uses -x, a failure here hides nothing.
"""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu


def _existing_path(crowd, k, r):
    """qmc_spo_vgl with r' given for every walker: the path the library has had since round 1."""
    import torch
    return tuple(npy(x) for x in crowd.qmc_spo_vgl(k, rnew=torch.from_numpy(r).cuda(), want_outputs=True))


@pytest.mark.parametrize("dtype,n_elec,tol", [("f32", 40, 1e-5), ("f64", 24, 1e-12)])
def test_static_scratch_entry_point_matches_the_crowd_path_on_two_calls_in_a_row(dtype, n_elec, tol):
    import torch
    import paper_2209_14487_b200 as q
    W = 7
    wl = qi.small_workload(n_elec=n_elec, grid=8, box=5.0, coef_dtype=dtype, coef_dist="uniform" if dtype == "f64" else "normal",
                           n_walkers=W, tau=0.02, delay_rank=1, cfg=61)
    crowd, osys, coefs, pos = make_pair(wl)
    coefs_dev = torch.from_numpy(coefs).cuda()
    rng = np.random.default_rng(7)
    r1 = pos[:, 3] + rng.normal(0.0, 0.4, (W, 3))
    r2 = rng.uniform(-2.0 * wl.box, 3.0 * wl.box, (W, 3))            # outside the box: periodic images (D:C1)
    ref1 = _existing_path(crowd, 3, r1)
    ref2 = _existing_path(crowd, 3, r2)

    got1 = tuple(npy(x) for x in q.qmc_spo_vgl_static(coefs_dev, wl.box, torch.from_numpy(r1).cuda()))
    got2 = tuple(npy(x) for x in q.qmc_spo_vgl_static(coefs_dev, wl.box, torch.from_numpy(r2[:3]).cuda()))
    for g, r in zip(got1, ref1):
        assert g.shape == r.shape and g.dtype == r.dtype
        assert relerr(g, r) < tol
    for g, r in zip(got2, ref2):
        assert g.shape == r[:3].shape
        assert relerr(g, r[:3]) < tol
    # the same device function on the same inputs: in fact bit for bit
    assert all(np.array_equal(g, r) for g, r in zip(got1, ref1))
    # and the plain definition
    for w in (0, W - 1):
        p_ref, dp_ref, d2p_ref = osys.spo_vgl(r1[w])
        assert relerr(got1[0][w], p_ref) < tol and relerr(got1[1][w], dp_ref) < tol and relerr(got1[2][w], d2p_ref) < tol


def test_static_scratch_limit_is_enforced_and_nothing_is_allocated():
    import torch
    import paper_2209_14487_b200 as q
    wl = qi.small_workload(n_elec=32, grid=6, box=4.0, coef_dtype="f32", coef_dist="normal", n_walkers=2, cfg=62)
    coefs_dev = torch.from_numpy(qi.make_coefs(wl)).cuda()
    M, ns = 16, 16
    p_max = q.STATIC_SCRATCH_BYTES // (5 * ns * 4)
    r = torch.rand((p_max + 1, 3), dtype=torch.float64, device="cuda") * wl.box
    phi = torch.zeros((p_max + 1, M), dtype=torch.float32, device="cuda")
    dphi = torch.zeros((p_max + 1, 3, M), dtype=torch.float32, device="cuda")
    d2phi = torch.zeros((p_max + 1, M), dtype=torch.float32, device="cuda")
    with pytest.raises(q.QmcError) as e:
        q.qmc_spo_vgl_static(coefs_dev, wl.box, r, phi, dphi, d2phi)
    assert e.value.status == q.QMC_ERR_WORKSPACE and "static array holds" in str(e.value)
    torch.cuda.synchronize()
    assert not phi.any() and not dphi.any() and not d2phi.any()       # a refused call launches nothing
    # the largest accepted size, with caller-owned outputs: the driver's allocator is not touched by the call
    # (one small call first: the first launch of a kernel may make the driver load its code)
    q.qmc_spo_vgl_static(coefs_dev, wl.box, r[:1], phi[p_max:], dphi[p_max:], d2phi[p_max:])
    phi[p_max:].zero_()
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    q.qmc_spo_vgl_static(coefs_dev, wl.box, r[:p_max], phi[:p_max], dphi[:p_max], d2phi[:p_max])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, qi.make_coefs(wl), tau=wl.tau)
    for w in (0, p_max - 1):
        assert relerr(npy(phi[w]), osys.spo_vgl(npy(r[w]))[0]) < 1e-5
    assert not phi[p_max].any()
    # empty input: a no-op
    q.qmc_spo_vgl_static(coefs_dev, wl.box, r[:0])
