"""BASELINE.json configs 2, 3, 4 at their full sizes (the other bench-able shapes): one free-running sweep through
qmc_sweep in the launch configuration the library uses there, then properties that hold at any size and sampled
walkers the oracle can check one by one (P-inv protocol: the carried inverse inverts the Slater matrix rebuilt from
the CUDA spline at the final positions; the spline itself against the oracle on sampled electrons)."""
import numpy as np
import pytest

import qmc_inputs as qi
from gpu_util import make_pair, npy, relerr

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_full_config_sweep_properties_and_sampled_inverse(cfg):
    import torch
    wl = qi.WORKLOADS[cfg]
    W, N, n, kd = wl.n_walkers, wl.n_elec, wl.n, wl.delay_rank
    crowd, osys, _, pos = make_pair(wl)
    crowd.qmc_sweep(1)
    st = crowd.stats()
    assert st["proposed"] == W * N
    assert st["flushes"] == (0 if kd == 1 else 2 * (-(-n // kd)))
    alpha = st["accepted"] / st["proposed"]
    assert 0.5 < alpha < 0.999
    R1 = npy(crowd.positions())
    assert np.isfinite(R1).all()
    assert np.any(R1 != pos, axis=2).sum() == st["accepted"]
    sample = (0, W // 3, W - 1)
    idx = torch.tensor(sample, device="cuda")
    for spin in (0, 1):
        Bg = npy(crowd.inverse(spin)[idx])
        A = np.zeros((len(sample), n, n))
        for i in range(n):
            e = spin * n + i
            phi, _, _ = crowd.qmc_spo_vgl(e, rnew=torch.from_numpy(np.ascontiguousarray(R1[:, e])).cuda(), want_outputs=True)
            A[:, i] = npy(phi[idx]).astype(np.float64)
            if i % 61 == 0:
                for s, w in enumerate(sample):
                    assert relerr(A[s, i], osys.spo_vgl(R1[w, e])[0]) < 1e-5
        for s in range(len(sample)):
            res = np.abs(A[s] @ Bg[s].T - np.eye(n)).max()
            assert res < 1e-7, (cfg, spin, res)
    crowd.close()
