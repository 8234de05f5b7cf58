"""ORACLE -- test infrastructure, not the product.

Thin ctypes wrapper over ``oracle/qmc_oracle.c`` (plain fp64 C; see its header for what it
follows and what pins it).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing
from ``paper_2209_14487_b200`` and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "qmc_oracle.c"
_HDR = _HERE / "qmc_oracle.h"
_LIB = _HERE / "libqmc_oracle.so"


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2 -ffp-contract=off, OpenMP over walkers only)."""
    if (not force and _LIB.exists() and _LIB.stat().st_mtime >= _SRC.stat().st_mtime
            and _LIB.stat().st_mtime >= _HDR.stat().st_mtime):
        return _LIB
    tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-o", str(tmp), str(_SRC), "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


class System(C.Structure):
    _fields_ = [
        ("n_elec", C.c_int32), ("n_orb", C.c_int32), ("grid", C.c_int32 * 3), ("coef_dtype", C.c_int32),
        ("box", C.c_double * 3), ("coefs", C.c_void_p), ("j2_a", C.c_double), ("j2_b", C.c_double),
        ("tau", C.c_double), ("seed", C.c_uint64), ("delay_rank", C.c_int32), ("inverse_fp32", C.c_int32),
    ]


MOVE_LOG_DTYPE = np.dtype([
    ("rnew", "f8", 3), ("delta", "f8", 3), ("g_old", "f8", 3), ("g_new", "f8", 3),
    ("rho_d", "f8"), ("rho_j", "f8"), ("p", "f8"), ("u", "f8"), ("disp_margin", "f8"),
    ("accepted", "i4"), ("_pad", "i4"),
])

_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(str(build()))
    dp = C.POINTER(C.c_double)
    L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
    L.oracle_rng_gauss3.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, dp]
    L.oracle_rng_uniform.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
    L.oracle_rng_uniform.restype = C.c_double
    L.oracle_bspline_weights.argtypes = [C.c_double, dp, dp, dp]
    L.oracle_spo_vgl.argtypes = [C.POINTER(System), dp, dp, dp, dp]
    L.oracle_j2_logpsi.argtypes = [C.POINTER(System), dp]
    L.oracle_j2_logpsi.restype = C.c_double
    L.oracle_j2_usum_grad.argtypes = [C.POINTER(System), dp, C.c_int, dp, dp, dp]
    L.oracle_kinetic_energy.argtypes = [C.POINTER(System), dp, dp, dp, dp]
    L.oracle_kinetic_energy.restype = C.c_double
    L.oracle_lu_inverse_transpose.argtypes = [C.c_int, dp, dp, dp, C.POINTER(C.c_int)]
    L.oracle_sm_update.argtypes = [C.c_int, dp, C.c_int, dp, C.c_double]
    ip = C.POINTER(C.c_int32)
    L.oracle_delayed_row.argtypes = [C.c_int, dp, C.c_int, ip, dp, dp, C.c_int, dp]
    L.oracle_delayed_flush.argtypes = [C.c_int, dp, C.c_int, ip, dp, dp]
    L.oracle_move_propose.argtypes = [C.c_double, dp, dp, dp, dp, dp, dp]
    L.oracle_move_accept.argtypes = [C.c_double, dp, dp, dp, C.c_double, C.c_double, C.c_double, dp]
    L.oracle_crowd_create.argtypes = [C.POINTER(System), C.c_int, C.c_int, dp, C.POINTER(C.c_int)]
    L.oracle_crowd_create.restype = C.c_void_p
    L.oracle_crowd_destroy.argtypes = [C.c_void_p]
    L.oracle_crowd_sweep.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
    L.oracle_crowd_sweep.restype = C.c_int64
    L.oracle_crowd_set_sweep_index.argtypes = [C.c_void_p, C.c_uint32]
    L.oracle_crowd_recompute.argtypes = [C.c_void_p]
    L.oracle_crowd_recompute.restype = C.c_int
    L.oracle_round_to_fp32.argtypes = [C.c_int, dp]
    L.oracle_crowd_branch.argtypes = [C.c_void_p, C.c_void_p]
    L.oracle_crowd_branch.restype = C.c_int
    L.oracle_crowd_get_positions.argtypes = [C.c_void_p, dp]
    L.oracle_crowd_get_inverse.argtypes = [C.c_void_p, C.c_int, dp]
    L.oracle_num_threads.restype = C.c_int
    _lib = L
    return L


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a: np.ndarray):
    assert a.dtype == np.int32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


# ----------------------------------------------------------------------------- random numbers
def philox4x32_10(ctr, key) -> np.ndarray:
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def rng_gauss3(seed: int, walker: int, k: int, sweep: int) -> np.ndarray:
    out = np.zeros(3)
    lib().oracle_rng_gauss3(seed, walker, k, sweep, _dp(out))
    return out


def rng_uniform(seed: int, walker: int, k: int, sweep: int) -> float:
    return float(lib().oracle_rng_uniform(seed, walker, k, sweep))


# ----------------------------------------------------------------------------- system
class OracleSystem:
    """Owns a ``System`` struct and keeps the coefficient array alive."""

    def __init__(self, n_elec: int, grid, box, coefs: np.ndarray, j2_a=0.5, j2_b=1.0, tau=0.01,
                 seed=1, delay_rank=1, inverse_fp32=False):
        n_orb = n_elec // 2
        grid = [int(g) for g in grid]
        assert coefs.dtype in (np.float32, np.float64)
        assert coefs.shape == (grid[0], grid[1], grid[2], n_orb), coefs.shape
        self.coefs = np.ascontiguousarray(coefs)
        self.n_elec, self.n_orb, self.n = n_elec, n_orb, n_elec // 2
        self.grid, self.box = grid, [float(b) for b in box]
        s = System()
        s.n_elec, s.n_orb = n_elec, n_orb
        s.grid = (C.c_int32 * 3)(*grid)
        s.coef_dtype = 0 if self.coefs.dtype == np.float32 else 1
        s.box = (C.c_double * 3)(*self.box)
        s.coefs = self.coefs.ctypes.data
        s.j2_a, s.j2_b, s.tau, s.seed, s.delay_rank = j2_a, j2_b, tau, seed, delay_rank
        s.inverse_fp32 = 1 if inverse_fp32 else 0
        self.struct = s

    @property
    def ref(self):
        return C.byref(self.struct)

    def spo_vgl(self, r):
        M = self.n_orb
        r = _f64(r)
        phi, dphi, d2phi = np.zeros(M), np.zeros((3, M)), np.zeros(M)
        lib().oracle_spo_vgl(self.ref, _dp(r), _dp(phi), _dp(dphi), _dp(d2phi))
        return phi, dphi, d2phi

    def j2_logpsi(self, R) -> float:
        R = _f64(R)
        assert R.shape == (self.n_elec, 3)
        return float(lib().oracle_j2_logpsi(self.ref, _dp(R)))

    def j2_usum_grad(self, R, k: int, rk):
        R, rk = _f64(R), _f64(rk)
        us, g = C.c_double(), np.zeros(3)
        lib().oracle_j2_usum_grad(self.ref, _dp(R), k, _dp(rk), C.byref(us), _dp(g))
        return us.value, g


    def kinetic_energy(self, R, B_up, B_dn):
        """(T, per-electron terms): -1/2 sum_k lap_k Psi / Psi at R with the transposed inverses B_up, B_dn."""
        R, B_up, B_dn = _f64(R), _f64(B_up), _f64(B_dn)
        n = self.n_elec // 2
        assert R.shape == (self.n_elec, 3) and B_up.shape == (n, n) and B_dn.shape == (n, n)
        e = np.zeros(self.n_elec)
        t = lib().oracle_kinetic_energy(self.ref, _dp(R), _dp(B_up), _dp(B_dn), _dp(e))
        return float(t), e


def bspline_weights(t: float):
    a, da, d2a = np.zeros(4), np.zeros(4), np.zeros(4)
    lib().oracle_bspline_weights(t, _dp(a), _dp(da), _dp(d2a))
    return a, da, d2a


# ----------------------------------------------------------------------------- linear algebra
def lu_inverse_transpose(A):
    A = _f64(A)
    n = A.shape[0]
    B = np.zeros((n, n))
    la, sg = C.c_double(), C.c_int()
    st = lib().oracle_lu_inverse_transpose(n, _dp(A), _dp(B), C.byref(la), C.byref(sg))
    return st, B, la.value, sg.value


def sm_update(B, k: int, phi, rho_d: float) -> np.ndarray:
    B = _f64(B).copy()
    phi = _f64(phi)
    lib().oracle_sm_update(B.shape[0], _dp(B), k, _dp(phi), rho_d)
    return B


def round_to_fp32(B) -> np.ndarray:
    B = _f64(B).copy()
    lib().oracle_round_to_fp32(B.shape[0], _dp(B))
    return B


def delayed_row(B0, rows, V, Cm, k: int) -> np.ndarray:
    B0, V, Cm = _f64(B0), _f64(V), _f64(Cm)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    n, m = B0.shape[0], len(rows)
    b = np.zeros(n)
    st = lib().oracle_delayed_row(n, _dp(B0), m, _ip(rows), _dp(V), _dp(Cm), k, _dp(b))
    assert st == 0, "singular window"
    return b


def delayed_flush(B0, rows, V, Cm) -> np.ndarray:
    B = _f64(B0).copy()
    V, Cm = _f64(V), _f64(Cm)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    st = lib().oracle_delayed_flush(B.shape[0], _dp(B), len(rows), _ip(rows), _dp(V), _dp(Cm))
    assert st == 0, "singular window"
    return B


# ----------------------------------------------------------------------------- the move
def move_propose(tau: float, rk, g_old, chi):
    rk, g_old, chi = _f64(rk), _f64(g_old), _f64(chi)
    delta, rnew, mg = np.zeros(3), np.zeros(3), C.c_double()
    lib().oracle_move_propose(tau, _dp(rk), _dp(g_old), _dp(chi), _dp(delta), _dp(rnew), C.byref(mg))
    return delta, rnew, mg.value


def move_accept(tau: float, delta, g_old, g_new, rho_d: float, rho_j: float, u: float):
    delta, g_old, g_new = _f64(delta), _f64(g_old), _f64(g_new)
    p = C.c_double()
    acc = lib().oracle_move_accept(tau, _dp(delta), _dp(g_old), _dp(g_new), rho_d, rho_j, u, C.byref(p))
    return bool(acc), p.value


# ----------------------------------------------------------------------------- crowd
class OracleCrowd:
    def __init__(self, system: OracleSystem, pos, walker_id0: int = 0):
        pos = _f64(pos)
        assert pos.ndim == 3 and pos.shape[1:] == (system.n_elec, 3)
        self.sys, self.W = system, pos.shape[0]
        st = C.c_int()
        self._h = lib().oracle_crowd_create(system.ref, self.W, walker_id0, _dp(pos), C.byref(st))
        if not self._h or st.value != 0:
            raise RuntimeError(f"oracle_crowd_create failed, status {st.value}")

    def sweep(self, n_sweeps: int = 1, log: bool = False):
        rec = None
        if log:
            rec = np.zeros((n_sweeps, self.W, self.sys.n_elec), dtype=MOVE_LOG_DTYPE)
        acc = lib().oracle_crowd_sweep(self._h, n_sweeps, rec.ctypes.data if log else None)
        return (int(acc), rec) if log else int(acc)

    def set_sweep_index(self, s: int):
        lib().oracle_crowd_set_sweep_index(self._h, s)

    def recompute(self):
        st = lib().oracle_crowd_recompute(self._h)
        if st != 0:
            raise RuntimeError(f"oracle_crowd_recompute: status {st}")

    def branch(self, src):
        src = np.ascontiguousarray(src, dtype=np.int32)
        assert src.shape == (self.W,)
        st = lib().oracle_crowd_branch(self._h, src.ctypes.data)
        if st != 0:
            raise ValueError(f"oracle_crowd_branch: status {st}")

    def positions(self) -> np.ndarray:
        out = np.zeros((self.W, self.sys.n_elec, 3))
        lib().oracle_crowd_get_positions(self._h, _dp(out))
        return out

    def inverse(self, spin: int) -> np.ndarray:
        n = self.sys.n
        out = np.zeros((self.W, n, n))
        lib().oracle_crowd_get_inverse(self._h, spin, _dp(out))
        return out

    def close(self):
        if self._h:
            lib().oracle_crowd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def num_threads() -> int:
    return int(lib().oracle_num_threads())
