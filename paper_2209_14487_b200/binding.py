"""ctypes binding of libqmc_crowd.so (include/qmc_crowd.h): argument marshalling only.

PyTorch is used here for device memory (workspace, table, outputs) and for the CUDA stream; every
step of the path runs in the library's kernels.  There is no CPU fallback: if the library is
missing or no CUDA device exists, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

from . import build as _build

_lib = None

QMC_OK, QMC_ERR_INVALID_ARG, QMC_ERR_CUDA, QMC_ERR_WORKSPACE, QMC_ERR_SINGULAR, QMC_ERR_STATE = range(6)
QMC_OPT_GRAPH = 0
QMC_OPT_PROFILE = 1
QMC_OPT_SUBCROWDS = 2
QMC_OPT_RECOMPUTE_EVERY = 3
QMC_OPT_STRIP_ROWS = 4
KERNEL_CLASSES = ("row_propose", "spline_vgl", "ratio_grad", "accept", "rank1", "flush", "ratio_accept",
                  "window", "kinetic", "branch")

EXPORTS = [
    "qmc_crowd_workspace_bytes", "qmc_crowd_create", "qmc_crowd_destroy", "qmc_spo_vgl", "qmc_ratio_grad",
    "qmc_accept_reject", "qmc_flush_delayed", "qmc_sweep", "qmc_sweep_host", "qmc_kinetic_energy", "qmc_recompute_inverse", "qmc_crowd_branch", "qmc_crowd_walker_state_bytes", "qmc_crowd_export_walkers",
    "qmc_crowd_import_walkers", "qmc_crowd_get_positions",
    "qmc_crowd_set_positions", "qmc_crowd_get_inverse", "qmc_crowd_set_inverse", "qmc_crowd_get_caches",
    "qmc_crowd_get_window", "qmc_crowd_get_move", "qmc_crowd_set_sweep_index", "qmc_crowd_stats",
    "qmc_crowd_launch_count", "qmc_crowd_set_option", "qmc_crowd_get_profile", "qmc_last_error", "qmc_version",
    "qmc_spo_vgl_static",
]
STATIC_SCRATCH_BYTES = 4 << 20      # QMC_STATIC_SCRATCH_BYTES of include/qmc_crowd.h


class QmcError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"qmc status {status}: {msg}")
        self.status = status


class CrowdDesc(C.Structure):
    _fields_ = [
        ("n_elec", C.c_int32), ("n_orb", C.c_int32), ("grid", C.c_int32 * 3), ("coef_dtype", C.c_int32),
        ("box", C.c_double * 3), ("coefs", C.c_void_p), ("orb_stride", C.c_int64),
        ("j2_a", C.c_double), ("j2_b", C.c_double), ("tau", C.c_double),
        ("n_walkers", C.c_int32), ("walker_id0", C.c_int32), ("delay_rank", C.c_int32), ("inverse_dtype", C.c_int32),
        ("seed", C.c_uint64), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("stream", C.c_void_p),
    ]


def lib_path() -> Path:
    return _build.LIB


def load():
    """Load libqmc_crowd.so (building it in-tree first if sources are newer and nvcc exists)."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        _build.build()
    except (FileNotFoundError, OSError):
        pass  # no nvcc on this box: use the shipped .so
    if not _build.LIB.exists():
        raise ImportError(f"{_build.LIB} is missing: run `python -m paper_2209_14487_b200.build` (needs nvcc). "
                          "There is no fallback path.")
    L = C.CDLL(str(_build.LIB))
    vp, ip, dp = C.c_void_p, C.c_int, C.c_void_p
    L.qmc_crowd_workspace_bytes.argtypes = [C.POINTER(CrowdDesc)]
    L.qmc_crowd_workspace_bytes.restype = C.c_size_t
    L.qmc_crowd_create.argtypes = [C.POINTER(CrowdDesc), dp, C.POINTER(vp)]
    L.qmc_crowd_destroy.argtypes = [vp]
    L.qmc_spo_vgl.argtypes = [vp, ip, dp, vp, vp, vp]
    L.qmc_ratio_grad.argtypes = [vp, ip, dp, dp]
    L.qmc_accept_reject.argtypes = [vp, ip, vp]
    L.qmc_flush_delayed.argtypes = [vp]
    L.qmc_recompute_inverse.argtypes = [vp]
    L.qmc_crowd_branch.argtypes = [vp, vp, C.POINTER(C.c_int)]
    L.qmc_crowd_walker_state_bytes.argtypes = [vp]
    L.qmc_crowd_walker_state_bytes.restype = C.c_size_t
    L.qmc_crowd_export_walkers.argtypes = [vp, ip, vp, vp]
    L.qmc_crowd_import_walkers.argtypes = [vp, ip, vp, vp]
    L.qmc_sweep.argtypes = [vp, ip]
    L.qmc_sweep_host.argtypes = [vp, vp, ip, vp]
    L.qmc_kinetic_energy.argtypes = [vp, dp, dp]
    L.qmc_crowd_get_positions.argtypes = [vp, dp]
    L.qmc_crowd_set_positions.argtypes = [vp, dp]
    L.qmc_crowd_get_inverse.argtypes = [vp, ip, dp]
    L.qmc_crowd_set_inverse.argtypes = [vp, ip, dp]
    L.qmc_crowd_get_caches.argtypes = [vp, vp, vp]
    L.qmc_crowd_get_window.argtypes = [vp, vp, vp, dp, dp, dp]
    L.qmc_crowd_get_move.argtypes = [vp] + [dp] * 9
    L.qmc_crowd_set_sweep_index.argtypes = [vp, C.c_uint32]
    L.qmc_crowd_stats.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.qmc_crowd_launch_count.argtypes = [vp]
    L.qmc_crowd_launch_count.restype = C.c_uint64
    L.qmc_crowd_set_option.argtypes = [vp, ip, ip]
    L.qmc_crowd_get_profile.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
    L.qmc_spo_vgl_static.argtypes = [ip, C.POINTER(C.c_int32), C.POINTER(C.c_double), ip, vp, C.c_int64, ip, dp, vp, vp, vp, vp]
    L.qmc_last_error.restype = C.c_char_p
    L.qmc_version.restype = C.c_char_p
    _lib = L
    return L


def _check(st: int):
    if st != QMC_OK:
        raise QmcError(st, load().qmc_last_error().decode())


def _ptr(t, dtype=None):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    return t.data_ptr()


def qmc_spo_vgl_static(coefs, box, r, phi=None, dphi=None, d2phi=None):
    """include/qmc_crowd.h qmc_spo_vgl_static: orbitals at the positions r [P][3] (CUDA fp64) from the table coefs
    [gx][gy][gz][orb_stride] (CUDA fp32 / fp64, n_orb = orb_stride), no crowd, no workspace, no allocation inside the
    library.  phi [P][M], dphi [P][3][M], d2phi [P][M]: caller-owned CUDA outputs of the table's dtype (allocated here
    when None -- by the caller's allocator, outside the library).  Runs on the current stream."""
    import torch
    assert coefs.is_cuda and coefs.is_contiguous() and coefs.dim() == 4 and r.is_cuda and r.dtype == torch.float64
    r = r.contiguous()
    P, M = int(r.shape[0]), int(coefs.shape[3])
    grid = (C.c_int32 * 3)(*[int(x) for x in coefs.shape[:3]])
    bx = (C.c_double * 3)(*([float(box)] * 3 if not hasattr(box, "__len__") else [float(x) for x in box]))
    if phi is None:
        phi = torch.empty((P, M), dtype=coefs.dtype, device=coefs.device)
    if dphi is None:
        dphi = torch.empty((P, 3, M), dtype=coefs.dtype, device=coefs.device)
    if d2phi is None:
        d2phi = torch.empty((P, M), dtype=coefs.dtype, device=coefs.device)
    for o in (phi, dphi, d2phi):
        assert o.is_cuda and o.is_contiguous() and o.dtype == coefs.dtype
    stream = torch.cuda.current_stream(coefs.device).cuda_stream
    _check(load().qmc_spo_vgl_static(M, grid, bx, 1 if coefs.dtype == torch.float64 else 0, coefs.data_ptr(), M, P,
                                     r.data_ptr() if P else None, phi.data_ptr() if P else None,
                                     dphi.data_ptr() if P else None, d2phi.data_ptr() if P else None, stream))
    return phi, dphi, d2phi


class Crowd:
    """A crowd of walkers advanced in lock-step.  Methods carry the C names."""

    def __init__(self, coefs, box, positions, *, tau, delay_rank=1, j2_a=0.5, j2_b=1.0, seed=1, walker_id0=0,
                 n_orb=None, stream=None, inverse_fp32=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("qmc crowd needs a CUDA device; there is no CPU fallback")
        L = load()
        assert coefs.is_cuda and coefs.is_contiguous() and coefs.dim() == 4
        assert coefs.dtype in (torch.float32, torch.float64)
        assert positions.is_cuda and positions.dtype == torch.float64 and positions.dim() == 3
        positions = positions.contiguous()
        W, N, _ = positions.shape
        self.torch = torch
        self.coefs = coefs                      # keep alive (BORROWED by the library)
        self.dtype = coefs.dtype
        self.W, self.N, self.n = W, N, N // 2
        self.M = N // 2 if n_orb is None else n_orb
        self.delay_rank = delay_rank
        self.device = coefs.device
        self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
        d = CrowdDesc()
        d.n_elec, d.n_orb = N, self.M
        d.grid = (C.c_int32 * 3)(*coefs.shape[:3])
        d.coef_dtype = 0 if coefs.dtype == torch.float32 else 1
        box = [float(box)] * 3 if not hasattr(box, "__len__") else [float(b) for b in box]
        d.box = (C.c_double * 3)(*box)
        d.coefs = coefs.data_ptr()
        d.orb_stride = coefs.shape[3]
        d.j2_a, d.j2_b, d.tau = j2_a, j2_b, tau
        d.n_walkers, d.walker_id0, d.delay_rank = W, walker_id0, delay_rank
        d.inverse_dtype = 1 if inverse_fp32 else 0
        d.seed = seed
        d.stream = self.stream.cuda_stream
        need = L.qmc_crowd_workspace_bytes(C.byref(d))
        if need == 0:
            raise QmcError(QMC_ERR_INVALID_ARG, L.qmc_last_error().decode())
        self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
        d.workspace, d.workspace_bytes = self.workspace.data_ptr(), need
        self.desc = d
        h = C.c_void_p()
        with torch.cuda.stream(self.stream):
            _check(L.qmc_crowd_create(C.byref(d), positions.data_ptr(), C.byref(h)))
        self._h = h

    # -- the six calls of the boundary -----------------------------------------------------
    # Outputs are allocated with the crowd's stream current (so the caching allocator ties the block to the stream the
    # library writes it on) and the caller's current stream is made to wait for the kernels that fill them: a consumer
    # on another stream never reads an output early when the crowd was built with its own stream (multi-crowd mode).
    def _on_stream(self):
        return self.torch.cuda.stream(self.stream)

    def _publish(self, caller_stream):
        if caller_stream != self.stream:
            caller_stream.wait_stream(self.stream)

    def qmc_spo_vgl(self, k, rnew=None, want_outputs=False):
        t = self.torch
        phi = dphi = d2phi = None
        caller = t.cuda.current_stream(self.device)
        if rnew is not None and caller != self.stream:
            self.stream.wait_stream(caller)            # rnew was produced on the caller's stream
        with self._on_stream():
            if want_outputs:
                phi = t.empty((self.W, self.M), dtype=self.dtype, device=self.device)
                dphi = t.empty((self.W, 3, self.M), dtype=self.dtype, device=self.device)
                d2phi = t.empty((self.W, self.M), dtype=self.dtype, device=self.device)
            _check(load().qmc_spo_vgl(self._h, k, _ptr(rnew, t.float64), _ptr(phi), _ptr(dphi), _ptr(d2phi)))
        if want_outputs:
            self._publish(caller)
        return (phi, dphi, d2phi) if want_outputs else None

    def qmc_ratio_grad(self, k):
        t = self.torch
        caller = t.cuda.current_stream(self.device)
        with self._on_stream():
            ratio = t.empty(self.W, dtype=t.float64, device=self.device)
            grad = t.empty((self.W, 3), dtype=t.float64, device=self.device)
            _check(load().qmc_ratio_grad(self._h, k, ratio.data_ptr(), grad.data_ptr()))
        self._publish(caller)
        return ratio, grad

    def qmc_accept_reject(self, k):
        t = self.torch
        caller = t.cuda.current_stream(self.device)
        with self._on_stream():
            acc = t.empty(self.W, dtype=t.uint8, device=self.device)
            _check(load().qmc_accept_reject(self._h, k, acc.data_ptr()))
        self._publish(caller)
        return acc

    def qmc_flush_delayed(self):
        _check(load().qmc_flush_delayed(self._h))

    def qmc_recompute_inverse(self):
        _check(load().qmc_recompute_inverse(self._h))

    def walker_state_bytes(self):
        return int(load().qmc_crowd_walker_state_bytes(self._h))

    def qmc_crowd_export_walkers(self, slots):
        """slots: int32 CUDA tensor [n]. Returns a uint8 CUDA tensor [n, walker_state_bytes] of packed states."""
        import torch
        assert slots.dtype == torch.int32 and slots.is_cuda and slots.is_contiguous()
        n = slots.numel()
        buf = torch.empty((n, self.walker_state_bytes()), dtype=torch.uint8, device=self.device)
        with torch.cuda.stream(self.stream):
            _check(load().qmc_crowd_export_walkers(self._h, n, slots.data_ptr(), buf.data_ptr()))
        return buf

    def qmc_crowd_import_walkers(self, slots, buf):
        import torch
        assert slots.dtype == torch.int32 and slots.is_cuda and slots.is_contiguous()
        n = slots.numel()
        assert buf.dtype == torch.uint8 and buf.is_cuda and buf.is_contiguous()
        assert buf.numel() == n * self.walker_state_bytes()
        with torch.cuda.stream(self.stream):
            _check(load().qmc_crowd_import_walkers(self._h, n, slots.data_ptr(), buf.data_ptr()))

    def qmc_crowd_branch(self, src):
        """src: int32 CUDA tensor [W]; slot w takes over the state of slot src[w]. Returns the number of copied slots."""
        import torch
        assert src.dtype == torch.int32 and src.is_cuda and src.is_contiguous() and src.numel() == self.W
        n = C.c_int(0)
        with torch.cuda.stream(self.stream):
            _check(load().qmc_crowd_branch(self._h, src.data_ptr(), C.byref(n)))
        return n.value

    def qmc_sweep(self, n_sweeps=1):
        _check(load().qmc_sweep(self._h, n_sweeps))

    def qmc_sweep_host(self, pos_host, n_sweeps=1):
        """pos_host: pinned (or plain) CPU float64 tensor [W][N][3], updated in place. Returns stats."""
        assert (not pos_host.is_cuda) and pos_host.is_contiguous() and pos_host.dtype == self.torch.float64
        assert tuple(pos_host.shape) == (self.W, self.N, 3)
        stats = (C.c_uint64 * 3)()
        _check(load().qmc_sweep_host(self._h, pos_host.data_ptr(), n_sweeps, stats))
        return {"proposed": stats[0], "accepted": stats[1], "flushes": stats[2]}

    def qmc_kinetic_energy(self, per_electron=False):
        """Kinetic energy of every walker, device fp64 [W] (and the per-electron terms [W][N] if asked)."""
        t = self.torch
        caller = t.cuda.current_stream(self.device)
        with self._on_stream():
            ekin = t.empty((self.W,), dtype=t.float64, device=self.device)
            e = t.empty((self.W, self.N), dtype=t.float64, device=self.device) if per_electron else None
            _check(load().qmc_kinetic_energy(self._h, ekin.data_ptr(), e.data_ptr() if per_electron else None))
        self._publish(caller)
        return (ekin, e) if per_electron else ekin

    # -- state access ------------------------------------------------------------------------
    def positions(self):
        t = self.torch
        out = t.empty((self.W, self.N, 3), dtype=t.float64, device=self.device)
        _check(load().qmc_crowd_get_positions(self._h, out.data_ptr()))
        return out

    def set_positions(self, pos):
        _check(load().qmc_crowd_set_positions(self._h, _ptr(pos.contiguous(), self.torch.float64)))

    def inverse(self, spin):
        t = self.torch
        out = t.empty((self.W, self.n, self.n), dtype=t.float64, device=self.device)
        _check(load().qmc_crowd_get_inverse(self._h, spin, out.data_ptr()))
        return out

    def set_inverse(self, spin, binv):
        assert tuple(binv.shape) == (self.W, self.n, self.n)
        _check(load().qmc_crowd_set_inverse(self._h, spin, _ptr(binv.contiguous(), self.torch.float64)))

    def caches(self):
        t = self.torch
        dphi = t.empty((self.W, self.N, 3, self.M), dtype=self.dtype, device=self.device)
        d2phi = t.empty((self.W, self.N, self.M), dtype=self.dtype, device=self.device)
        _check(load().qmc_crowd_get_caches(self._h, dphi.data_ptr(), d2phi.data_ptr()))
        return dphi, d2phi

    def window(self):
        t, k = self.torch, self.delay_rank
        m = t.empty(self.W, dtype=t.int32, device=self.device)
        rows = t.empty((self.W, k), dtype=t.int32, device=self.device)
        V = t.empty((self.W, k, self.n), dtype=t.float64, device=self.device)
        Cm = t.empty((self.W, k, self.n), dtype=t.float64, device=self.device)
        Sinv = t.empty((self.W, k, k), dtype=t.float64, device=self.device)
        _check(load().qmc_crowd_get_window(self._h, m.data_ptr(), rows.data_ptr(), V.data_ptr(), Cm.data_ptr(),
                                           Sinv.data_ptr()))
        return m, rows, V, Cm, Sinv

    def move(self):
        t = self.torch
        f = lambda *s: t.empty(s, dtype=t.float64, device=self.device)
        out = {"rnew": f(self.W, 3), "delta": f(self.W, 3), "g_old": f(self.W, 3), "g_new": f(self.W, 3),
               "rho_d": f(self.W), "rho_j": f(self.W), "p": f(self.W), "u": f(self.W), "brow": f(self.W, self.n)}
        _check(load().qmc_crowd_get_move(self._h, *[out[k].data_ptr() for k in
                                                    ("rnew", "delta", "g_old", "g_new", "rho_d", "rho_j", "p", "u",
                                                     "brow")]))
        return out

    def set_sweep_index(self, s):
        _check(load().qmc_crowd_set_sweep_index(self._h, s))

    def stats(self):
        a, b, c = C.c_uint64(), C.c_uint64(), C.c_uint64()
        _check(load().qmc_crowd_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return {"proposed": a.value, "accepted": b.value, "flushes": c.value}

    def launch_count(self):
        return int(load().qmc_crowd_launch_count(self._h))

    def profile(self):
        """{kernel class: (total ms, launches)} recorded in QMC_OPT_PROFILE mode since the last call."""
        ms, cnt = (C.c_double * len(KERNEL_CLASSES))(), (C.c_uint64 * len(KERNEL_CLASSES))()
        _check(load().qmc_crowd_get_profile(self._h, ms, cnt))
        return {name: (ms[i], int(cnt[i])) for i, name in enumerate(KERNEL_CLASSES)}

    def set_option(self, option, value):
        _check(load().qmc_crowd_set_option(self._h, option, value))

    def close(self):
        if getattr(self, "_h", None):
            load().qmc_crowd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
