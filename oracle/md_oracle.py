"""ctypes binding of oracle/libmd_oracle.so -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  See md_oracle.c for the citations.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build


class OrcParams(C.Structure):
    _fields_ = [("dim", C.c_int), ("L", C.c_double * 3), ("bc", C.c_int * 3), ("eps", C.c_double),
                ("sigma", C.c_double), ("eps_w", C.c_double), ("sigma_w", C.c_double), ("r_cut", C.c_double),
                ("shift_energy", C.c_int), ("dt", C.c_double), ("mass", C.c_double), ("tau_b", C.c_double),
                ("t_target", C.c_double), ("prism", C.c_int), ("prism_axis", C.c_int), ("prism_c", C.c_double * 3),
                ("prism_h", C.c_double * 3)]


_lib = None
_DP = C.POINTER(C.c_double)
_LP = C.POINTER(C.c_longlong)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        assert _lib.orc_sizeof_params() == C.sizeof(OrcParams)
        sig = [C.POINTER(OrcParams), C.c_long, _DP, C.c_long, _DP, _DP, _DP, _DP, _DP, _LP]
        _lib.orc_forces_brute.argtypes = sig
        _lib.orc_forces_brute.restype = None
        _lib.orc_forces_cells.argtypes = sig
        _lib.orc_forces_cells.restype = C.c_int
        _lib.orc_kinetic.argtypes = [C.POINTER(OrcParams), C.c_long, _DP]
        _lib.orc_kinetic.restype = C.c_double
        _lib.orc_run.argtypes = [C.POINTER(OrcParams), C.c_int, C.c_long, _DP, _DP, C.c_long, _DP, C.c_long,
                                 _DP, _DP, _DP, _DP, _DP]
        _lib.orc_run.restype = C.c_int
    return _lib


def params(cfg) -> OrcParams:
    p = OrcParams()
    p.dim = int(cfg["dim"])
    for a in range(3):
        p.L[a] = float(cfg["box_len"][a])
        p.bc[a] = int(cfg["bc"][a])
    p.eps, p.sigma = float(cfg["eps"]), float(cfg["sigma"])
    p.eps_w, p.sigma_w = float(cfg["eps_w"]), float(cfg["sigma_w"])
    p.r_cut = float(cfg["r_cut"])
    p.shift_energy = int(cfg.get("shift_energy", 1))
    p.dt, p.mass = float(cfg["dt"]), float(cfg["mass"])
    p.tau_b, p.t_target = float(cfg.get("tau_b", 0.0)), float(cfg.get("t_target", 1.0))
    pd = cfg.get("pore")
    if pd and pd["kind"] == "prism":         # geometric walls: centre, length along axis, width across
        p.prism, p.prism_axis = 1, int(pd["axis"])
        for a in range(p.dim):
            p.prism_c[a] = float(pd["center"][a])
            p.prism_h[a] = 0.5 * float(pd["length"] if a == p.prism_axis else pd["width"])
    return p


def _ptr(a):
    return a.ctypes.data_as(_DP)


def _arr(x, dim):
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(-1, dim))


def forces(cfg, pos=None, cells=False):
    """Forces/energies of cfg (or of `pos` in cfg's box). Returns a dict."""
    p = params(cfg)
    dim = p.dim
    pos = _arr(cfg["pos"] if pos is None else pos, dim)
    wall = _arr(cfg["wall"], dim)
    nv, nw = pos.shape[0], wall.shape[0]
    f = np.zeros((nv, dim))
    pe, pe_w, vir = np.zeros(nv), np.zeros(nv), np.zeros(nv)
    cnt = np.zeros(2, dtype=np.int64)
    cp = cnt.ctypes.data_as(_LP)
    if cells:
        rc = lib().orc_forces_cells(C.byref(p), nv, _ptr(pos), nw, _ptr(wall), _ptr(f), _ptr(pe), _ptr(pe_w),
                                    _ptr(vir), cp)
        if rc != 0:
            raise ValueError("oracle cell grid invalid (periodic dimension with < 3 cells)")
    else:
        lib().orc_forces_brute(C.byref(p), nv, _ptr(pos), nw, _ptr(wall), _ptr(f), _ptr(pe), _ptr(pe_w),
                               _ptr(vir), cp)
    assert cnt[0] % 2 == 0
    return dict(f=f, pe=pe, pe_w=pe_w, vir=vir, pairs_vv=int(cnt[0]) // 2, pairs_vw=int(cnt[1]),
                U=float(pe.sum()), U_vw=float(pe_w.sum()), U_vv=float(pe.sum() - pe_w.sum()))


def kinetic(cfg, vel):
    p = params(cfg)
    v = _arr(vel, p.dim)
    return float(lib().orc_kinetic(C.byref(p), v.shape[0], _ptr(v)))


def run(cfg, n_steps, pos=None, vel=None, cells=False, history=False):
    """n_steps of velocity Verlet from (pos, vel) (default: cfg's). Returns a dict with copies."""
    p = params(cfg)
    dim = p.dim
    pos = _arr(cfg["pos"] if pos is None else pos, dim).copy()
    vel = _arr(cfg["vel"] if vel is None else vel, dim).copy()
    wall = _arr(cfg["wall"], dim)
    nv, nw = pos.shape[0], wall.shape[0]
    f = np.zeros((nv, dim))
    pe, pe_w, vir = np.zeros(nv), np.zeros(nv), np.zeros(nv)
    hist = np.zeros((n_steps + 1, 5)) if history else None
    rc = lib().orc_run(C.byref(p), int(cells), nv, _ptr(pos), _ptr(vel), nw, _ptr(wall), int(n_steps), _ptr(f),
                       _ptr(pe), _ptr(pe_w), _ptr(vir), _ptr(hist) if history else None)
    if rc != 0:
        raise RuntimeError("oracle run failed with code %d" % rc)
    out = dict(pos=pos, vel=vel, f=f, pe=pe, pe_w=pe_w, vir=vir, K=kinetic(cfg, vel), U=float(pe.sum()),
               U_vw=float(pe_w.sum()))
    if history:
        out["hist"] = hist
    return out


def n_threads() -> int:
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
