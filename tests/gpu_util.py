"""Shared helpers of the -m gpu parity tests: build the CUDA crowd and the oracle from one Workload."""
from __future__ import annotations

import numpy as np

import oracle
import qmc_inputs as qi


def make_pair(wl: qi.Workload, n_walkers=None, walker_id0=0, delay_rank=None, orb_pad=0, coefs=None, pos=None):
    """Returns (gpu_crowd, oracle_system, coefs_np, pos_np). orb_pad > 0 pads the table's orbital stride."""
    import torch
    import paper_2209_14487_b200 as q

    kd = wl.delay_rank if delay_rank is None else delay_rank
    coefs = qi.make_coefs(wl) if coefs is None else coefs
    pos = qi.make_positions(wl, n_walkers) if pos is None else pos
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, j2_a=wl.j2_a, j2_b=wl.j2_b,
                               tau=wl.tau, seed=wl.seed, delay_rank=kd)
    vw = 4 if coefs.dtype == np.float32 else 2
    M = coefs.shape[3]
    stride = -(-M // vw) * vw + orb_pad * vw
    tab = np.full(coefs.shape[:3] + (stride,), 777.0, dtype=coefs.dtype)  # garbage in the padding
    tab[..., :M] = coefs
    dev = torch.device("cuda:0")
    crowd = q.Crowd(torch.from_numpy(tab).to(dev), wl.box, torch.from_numpy(pos).to(dev), tau=wl.tau, delay_rank=kd,
                    j2_a=wl.j2_a, j2_b=wl.j2_b, seed=wl.seed, walker_id0=walker_id0, n_orb=M)
    return crowd, osys, coefs, pos


def relerr(x, y):
    """Norm-wise relative error max|x - y| / max|y| (reading A10)."""
    x, y = np.asarray(x, dtype=np.float64), np.asarray(y, dtype=np.float64)
    den = np.max(np.abs(y))
    return float(np.max(np.abs(x - y)) / (den if den > 0 else 1.0))


def npy(t):
    return t.detach().cpu().numpy()
