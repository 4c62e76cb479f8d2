"""CPU-side checks of the boundary: the library builds/loads, exports every symbol of include/md.h,
validates arguments on the host, and fails loudly (no fallback) without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

from paper_1812_07993_b200 import build as B
from paper_1812_07993_b200 import inputs as I
from paper_1812_07993_b200 import md

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return md.load_library()


def test_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "md.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(md_[a-z_]+)\s*\(", header))
    assert declared == set(md.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_sizes_match_header_layout():
    assert C.sizeof(md.md_box) == 48 and C.sizeof(md.md_lj) == 48 and C.sizeof(md.md_opts) == 56
    assert C.sizeof(md.md_energy_out) == 64 and C.sizeof(md.md_kernel_times) == 136 and C.sizeof(md.md_peaks) == 24


def test_workspace_bytes_scale_and_reject(lib):
    small, big = I.config4(10), I.config4(14)
    a, b = md.workspace_bytes(small), md.workspace_bytes(big)
    assert 0 < a < b < 64 << 20
    assert md.workspace_bytes(big, precision=32) < b
    bad = dict(small)
    bad["dim"] = 4
    assert md.workspace_bytes(bad) == 0
    thin = I.small_case(2, 10, (6.0, 20.0), (0, 0), seed=2)
    assert md.workspace_bytes(thin, algo="cells") == 0        # < 3 cells in a periodic dimension
    assert md.workspace_bytes(thin, algo="auto") > 0          # AUTO falls back to all-pairs


def _create_raw(lib, cfg, ws_ptr=256, ws_bytes=1 << 30, **kw):
    box, lj, opts = md._structs(cfg, kw.get("precision", 64), kw.get("algo"))
    h = C.c_void_p()
    pos = np.ascontiguousarray(cfg["pos"])
    vel = np.ascontiguousarray(cfg["vel"])
    wall = np.ascontiguousarray(cfg["wall"])
    rc = lib.md_create(C.byref(h), C.byref(box), None, C.byref(lj), C.byref(opts), pos.shape[0], md._dptr(pos),
                       md._dptr(vel), wall.shape[0], md._dptr(wall) if wall.shape[0] else None, ws_ptr, ws_bytes, None)
    return rc, (lib.md_last_error(None) or b"").decode(), h


def test_host_validation_errors(lib):
    cfg = I.small_case(3, 20, (8.0, 8.0, 8.0), (0, 0, 1), n_wall=3, seed=1)
    for key, val, frag in (("dt", 0.0, "dt"), ("mass", -1.0, "mass"), ("r_cut", 0.0, "r_cut"), ("dim", 5, "dim")):
        bad = dict(cfg)
        bad[key] = val
        rc, msg, h = _create_raw(lib, bad)
        assert rc == md.MD_ERR_INVALID_ARG and frag in msg and not h.value
    bad = dict(cfg)
    bad["pos"] = cfg["pos"].copy()
    bad["pos"][3, 1] = 8.5
    rc, msg, _ = _create_raw(lib, bad)
    assert rc == md.MD_ERR_INVALID_ARG and "outside" in msg
    bad["pos"][3, 1] = np.nan
    assert _create_raw(lib, bad)[0] == md.MD_ERR_INVALID_ARG
    bad = dict(cfg)
    bad["box_len"] = [4.0, 8.0, 8.0]
    bad["pos"] = cfg["pos"] * np.array([0.5, 1, 1])
    rc, msg, _ = _create_raw(lib, bad)
    assert rc == md.MD_ERR_INVALID_ARG and "2 r_cut" in msg
    bad = dict(cfg, tau_b=0.001, t_target=1.0)               # tau_B < dt: lambda^2 could go negative
    rc, msg, _ = _create_raw(lib, bad)
    assert rc == md.MD_ERR_INVALID_ARG and "thermostat" in msg
    thin = I.small_case(2, 10, (6.0, 20.0), (0, 0), seed=2)
    rc, msg, _ = _create_raw(lib, thin, algo="cells")
    assert rc == md.MD_ERR_UNSUPPORTED
    rc, msg, _ = _create_raw(lib, cfg, ws_ptr=0)
    assert rc == md.MD_ERR_INVALID_ARG and "workspace" in msg
    assert lib.md_step(None, 1) == md.MD_ERR_INVALID_ARG


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_fails_loudly_without_fallback(lib):
    cfg = I.small_case(3, 20, (8.0, 8.0, 8.0), (0, 0, 1), seed=1)
    rc, msg, h = _create_raw(lib, cfg)
    assert rc == md.MD_ERR_CUDA and "no CPU fallback" in msg and not h.value
    with pytest.raises(md.MDError):
        md.Simulation(cfg)
    with pytest.raises(md.MDError):
        md.measure_peaks()


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1812_07993_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("CPU oracle", "").replace("the oracle", ""), f
