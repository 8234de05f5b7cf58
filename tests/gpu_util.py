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


def straddle_flags(log, tau, g_tol=1e-10):
    """Which logged moves have a displacement whose fp32 rounding (reading A7) is decided by less than a relative
    error g_tol of G_k(R)?  log: oracle move records [...]; returns a bool array of the same shape.

    Delta_c = fl32(x_c), x_c = tau G_c + sqrt(tau) chi_c.  Two correct fp64 implementations agree on G to g_tol
    (relative to max_c |G_c|; BASELINE.json: 1e-10) and on chi to a few ulp of libm, so their x_c differ by at most
    e = g_tol tau max|G| + 8 eps |x|; the roundings can differ only if x_c lies within e of a rounding boundary,
    i.e. if the oracle's margin (in fp32 ulps of Delta_c, minimum over components) is below e / ulp32(Delta_c)."""
    delta, g, margin = log["delta"], log["g_old"], log["disp_margin"]
    e = g_tol * tau * np.abs(g).max(axis=-1) + 8 * 2.0 ** -53 * np.abs(delta).max(axis=-1)
    ulp = np.spacing(np.abs(delta).astype(np.float32)).astype(np.float64)
    return margin < (e[..., None] / ulp).max(axis=-1)


class FreeRunningCheck:
    """P-free with classification: a free-running trajectory of the CUDA path against the
    oracle's, sweep by sweep, for crowds too long for "no rounding tie anywhere" to be a property of the inputs.

    Within a sweep every electron is proposed once, so the positions after the sweep show move by move where the two
    sides differ.  For every walker, all moves before its first difference agree bit for bit; that first difference
    must be a move whose fp32 displacement rounding the oracle itself reports as decided by less than the parity
    tolerance on G (straddle_flags) -- anything else is a bug and fails.  A walker that has met such a straddle has
    departed from the oracle's trajectory by one fp32 ulp of one displacement (~1e-8) and is from then on compared for
    closeness only (positions 1e-6, inverses 1e-5, same accept / reject decisions)."""

    def __init__(self, W, tau, g_tol=1e-10):
        self.tau, self.g_tol = tau, g_tol
        self.departed = np.zeros(W, dtype=bool)
        self.exact_moves = 0

    def sweep(self, Rg_prev, Rg, Ro_prev, Ro, log):
        """Rg_prev / Rg: CUDA positions before / after the sweep, Ro_prev / Ro: the oracle's; log: [W][N] records."""
        flags = straddle_flags(log, self.tau, self.g_tol)
        W, N = log.shape
        for w in range(W):
            diff = np.any(Rg[w] != Ro[w], axis=-1)
            if not self.departed[w]:
                if diff.any():
                    k = int(np.argmax(diff))
                    assert flags[w, k], (f"walker {w}, electron {k}: positions differ although the oracle's rounding "
                                         f"margin ({log[w, k]['disp_margin']:.3e} fp32 ulps) rules out a straddle")
                    self.departed[w] = True
                    self.exact_moves += k
                else:
                    self.exact_moves += N
            assert np.abs(Rg[w] - Ro[w]).max() < 1e-6, f"walker {w} left the oracle's trajectory"
            moved_g, moved_o = np.any(Rg[w] != Rg_prev[w], axis=-1), np.any(Ro[w] != Ro_prev[w], axis=-1)
            tie = np.abs(log[w]["u"] - log[w]["p"]) <= 1e-5 * np.abs(log[w]["p"])
            assert np.array_equal(moved_g[~tie], moved_o[~tie]), f"walker {w}: accept / reject decisions differ"

    def inverse_tol(self, w):
        return 1e-5 if self.departed[w] else 1e-10


def straddled_walkers(Ra, Rb, R_before, max_frac=2e-4, cascade=False, tau=0.02):
    """Two CUDA paths that evaluate the same move in different floating-point orders (qmc_sweep's eager-block form and
    the step calls' bordered form, R5) agree on G to ~1e-12, so they round a displacement to the two different
    neighbouring fp32 values only where the unrounded value sits on a rounding boundary to that accuracy (reading A7) --
    in practice a component that cancels to ~1e-6, whose fp32 ulp is ~1e-13.  Positions must be bit-identical except for
    at most a fraction max_frac of the components, each differing by exactly one fp32 ulp of its own displacement.
    Returns the walkers that contain such a component (their later moves see inputs that differ by that ulp)."""
    diff = Ra != Rb
    if not diff.any():
        return np.zeros(Ra.shape[0], dtype=bool)
    if cascade:
        # long sweeps (n = 384: 768 moves): a walker that met one straddle sees inputs that differ by that ulp in all its
        # later moves of the sweep, whose displacements then round differently every few moves.  Checked per walker: the
        # FIRST differing move (moves run in electron order) differs by one fp32 ulp of its displacement, or -- where the
        # component tau G + sqrt(tau) chi cancels to ~1e-5 and its fp32 ulp falls below the agreement of the two G's -- by
        # tau x 1e-8 (the two paths' G agree to 1e-10 of sum_j |b_j| |grad phi_j|, ~1e2 at n = 384 on random positions:
        # measured 1e-9 absolute); few walkers are affected, and they stay close.
        off = diff.any(axis=(1, 2))
        assert off.mean() <= 0.1, f"{off.sum()} of {off.size} walkers differ"
        for w in np.nonzero(off)[0]:
            k0 = int(np.argmax(diff[w].any(axis=1)))
            d = Ra[w, k0] - R_before[w, k0]
            ulp = np.spacing(np.abs(d).astype(np.float32)).astype(np.float64)
            assert (np.abs(Ra[w, k0] - Rb[w, k0]) <= 1.001 * ulp + tau * 1e-8).all(), (w, k0)
            assert np.abs(Ra[w] - Rb[w]).max() < 1e-5, w
        return off
    assert diff.mean() <= max_frac, f"{diff.sum()} position components differ"
    delta = np.where(diff, Ra - R_before, 1.0)
    ulp = np.spacing(np.abs(delta).astype(np.float32)).astype(np.float64)
    assert (np.abs(Ra - Rb)[diff] <= 1.001 * ulp[diff]).all(), "a position differs by more than one fp32 ulp of its displacement"
    return diff.any(axis=(1, 2))
