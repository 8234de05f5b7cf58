"""CPU-side checks of the boundary: libqmc_crowd.so loads and exports every symbol that
include/qmc_crowd.h declares; descriptor validation and workspace sizing (host logic, no kernels)."""
import ctypes as C
import re
from pathlib import Path

import pytest

import paper_2209_14487_b200 as q

ROOT = Path(__file__).resolve().parent.parent


def declared_symbols():
    txt = (ROOT / "include" / "qmc_crowd.h").read_text()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(qmc_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    lib = q.load()
    names = declared_symbols()
    assert len(names) >= 20 and "qmc_sweep" in names and "qmc_flush_delayed" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in qmc_crowd.h but not exported"
    assert sorted(q.EXPORTS) == names
    assert b"sm_100a" in lib.qmc_version()


def test_no_oracle_or_torch_types_cross_the_boundary():
    txt = (ROOT / "include" / "qmc_crowd.h").read_text()
    assert "torch" not in txt.replace("PyTorch", "") and "at::" not in txt and "std::" not in txt
    for p in (ROOT / "paper_2209_14487_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            body = p.read_text()
            assert "import oracle" not in body and "qmc_oracle" not in body, f"{p} touches the oracle"


def _desc(**kw):
    d = q.CrowdDesc()
    d.n_elec, d.n_orb = kw.get("n_elec", 768), kw.get("n_orb", kw.get("n_elec", 768) // 2)
    d.grid = (C.c_int32 * 3)(*([kw.get("grid", 80)] * 3))
    d.coef_dtype = kw.get("coef_dtype", 0)
    d.box = (C.c_double * 3)(*([kw.get("box", 23.0)] * 3))
    d.orb_stride = kw.get("orb_stride", d.n_orb)
    d.j2_a, d.j2_b, d.tau = 0.5, 1.0, kw.get("tau", 0.01)
    d.n_walkers, d.delay_rank = kw.get("n_walkers", 4096), kw.get("delay_rank", 32)
    return d


def test_workspace_bytes_matches_the_documented_layout():
    lib = q.load()
    W, N, n, k = 4096, 768, 384, 32
    need = lib.qmc_crowd_workspace_bytes(C.byref(_desc()))
    inverses = W * 2 * n * n * 8
    caches = W * N * 4 * n * 4
    window = 2 * W * k * n * 8
    lower = inverses + caches + window + W * N * 24
    assert lower <= need <= lower * 1.02, (need, lower)
    # padding of n to 16 and of the delay rank to 8/16/32/64
    small = lib.qmc_crowd_workspace_bytes(C.byref(_desc(n_elec=8, grid=16, coef_dtype=1, n_walkers=4, delay_rank=1)))
    assert small >= 4 * 2 * 16 * 16 * 8


@pytest.mark.parametrize("bad", [dict(n_elec=7), dict(n_orb=5), dict(n_walkers=0), dict(delay_rank=0),
                                 dict(delay_rank=65), dict(coef_dtype=2), dict(orb_stride=383), dict(orb_stride=386),
                                 dict(tau=0.0), dict(box=-1.0), dict(grid=0), dict(grid=4000, orb_stride=4 * 384)])
def test_bad_descriptors_are_refused(bad):
    lib = q.load()
    assert lib.qmc_crowd_workspace_bytes(C.byref(_desc(**bad))) == 0
    assert len(lib.qmc_last_error()) > 0


def test_null_handles_are_errors_not_crashes():
    lib = q.load()
    assert lib.qmc_sweep(None, 1) == q.QMC_ERR_INVALID_ARG
    assert lib.qmc_flush_delayed(None) == q.QMC_ERR_INVALID_ARG
    assert lib.qmc_spo_vgl(None, 0, None, None, None, None) == q.QMC_ERR_INVALID_ARG
    assert lib.qmc_crowd_destroy(None) == q.QMC_OK
    out = C.c_void_p()
    assert lib.qmc_crowd_create(None, None, C.byref(out)) == q.QMC_ERR_INVALID_ARG


def test_binding_constants_match_the_header():
    """Option numbers, status codes and the static scratch size are typed twice (header and binding): keep them equal."""
    txt = (ROOT / "include" / "qmc_crowd.h").read_text()
    for name in ("QMC_OPT_GRAPH", "QMC_OPT_PROFILE", "QMC_OPT_SUBCROWDS", "QMC_OPT_RECOMPUTE_EVERY", "QMC_OPT_STRIP_ROWS"):
        m = re.search(rf"#define\s+{name}\s+(\d+)", txt)
        assert m and int(m.group(1)) == getattr(q, name), name
    m = re.search(r"#define\s+QMC_STATIC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", txt)
    assert m and (int(m.group(1)) << int(m.group(2))) == q.STATIC_SCRATCH_BYTES
    for name in ("QMC_OK", "QMC_ERR_INVALID_ARG", "QMC_ERR_CUDA", "QMC_ERR_WORKSPACE", "QMC_ERR_SINGULAR", "QMC_ERR_STATE"):
        m = re.search(rf"\b{name}\s*=\s*(\d+)", txt)
        assert m and int(m.group(1)) == getattr(q, name), name
