"""Thin Python binding of include/md.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libmd_b200.so; PyTorch is
used for the device workspace (`torch.empty(uint8, device="cuda")`) and the stream.
There is no CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmd_b200.so")

MD_OK = 0
MD_ERR_INVALID_ARG, MD_ERR_UNSUPPORTED, MD_ERR_CUDA, MD_ERR_WORKSPACE, MD_ERR_NONFINITE, MD_ERR_STATE = -1, -2, -3, -4, -5, -6
MD_BC_PERIODIC, MD_BC_REFLECT = 0, 1
MD_FORCE_AUTO, MD_FORCE_ALLPAIRS, MD_FORCE_CELLS, MD_FORCE_VERLET = 0, 1, 2, 3
_ALGO = {"auto": MD_FORCE_AUTO, "allpairs": MD_FORCE_ALLPAIRS, "cells": MD_FORCE_CELLS, "verlet": MD_FORCE_VERLET}

EXPORTS = ["md_workspace_bytes", "md_create", "md_step", "md_get_state", "md_energy", "md_pressure", "md_density_profile", "md_profile_step",
           "md_pair_tests", "md_info", "md_measure_peaks", "md_destroy", "md_last_error", "md_kinetic_energy_noalloc"]
NOALLOC_MAX_PARTICLES = 4194304


class md_box(C.Structure):
    _fields_ = [("dim", C.c_int), ("len", C.c_double * 3), ("bc", C.c_int * 3)]


class md_pore(C.Structure):
    _fields_ = [("kind", C.c_int), ("axis", C.c_int), ("center", C.c_double * 3), ("length", C.c_double),
                ("r0", C.c_double), ("r1", C.c_double), ("neck_len", C.c_double), ("width", C.c_double)]


class md_lj(C.Structure):
    _fields_ = [("eps", C.c_double), ("sigma", C.c_double), ("eps_w", C.c_double), ("sigma_w", C.c_double),
                ("r_cut", C.c_double), ("shift_energy", C.c_int)]


class md_opts(C.Structure):
    _fields_ = [("dt", C.c_double), ("mass", C.c_double), ("precision", C.c_int), ("force_algo", C.c_int),
                ("skin", C.c_double), ("tau_b", C.c_double), ("t_target", C.c_double), ("heavy_list", C.c_int), ("list_prunes", C.c_int)]


class md_energy_out(C.Structure):
    _fields_ = [("kinetic", C.c_double), ("potential", C.c_double), ("potential_vv", C.c_double),
                ("potential_vw", C.c_double), ("virial", C.c_double), ("pairs_vv", C.c_longlong),
                ("pairs_vw", C.c_longlong), ("step", C.c_longlong)]


class md_pressure_out(C.Structure):
    _fields_ = [("pressure_box", C.c_double), ("volume_box", C.c_double), ("pressure_pore", C.c_double),
                ("volume_pore", C.c_double), ("kinetic_pore", C.c_double), ("virial_pore", C.c_double),
                ("n_pore", C.c_longlong), ("step", C.c_longlong)]


class md_kernel_times(C.Structure):
    _fields_ = [("ms", C.c_double * 4), ("launches", C.c_longlong * 4), ("total_ms", C.c_double),
                ("steps", C.c_longlong), ("rebuilds", C.c_longlong), ("rebuild_ms", C.c_double * 4), ("prunes", C.c_longlong), ("prune_ms", C.c_double)]


class md_peaks(C.Structure):
    _fields_ = [("fp64_tflops", C.c_double), ("fp32_tflops", C.c_double), ("copy_gbs", C.c_double)]


class MDError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("md error %d: %s" % (code, msg))
        self.code = code


_lib = None
_DP = C.POINTER(C.c_double)


def load_library():
    """Loads libmd_b200.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_1812_07993_b200.build` (there is no fallback)"
                              % LIB_PATH)
        lib = C.CDLL(LIB_PATH)
        lib.md_workspace_bytes.restype = C.c_size_t
        lib.md_workspace_bytes.argtypes = [C.POINTER(md_box), C.POINTER(md_lj), C.POINTER(md_opts), C.c_longlong,
                                           C.c_longlong]
        lib.md_create.restype = C.c_int
        lib.md_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(md_box), C.POINTER(md_pore), C.POINTER(md_lj),
                                  C.POINTER(md_opts), C.c_longlong, _DP, _DP, C.c_longlong, _DP, C.c_void_p,
                                  C.c_size_t, C.c_void_p]
        lib.md_step.restype = C.c_int
        lib.md_step.argtypes = [C.c_void_p, C.c_longlong]
        lib.md_get_state.restype = C.c_int
        lib.md_get_state.argtypes = [C.c_void_p, _DP, _DP, _DP, _DP, C.POINTER(C.c_longlong)]
        lib.md_energy.restype = C.c_int
        lib.md_energy.argtypes = [C.c_void_p, C.POINTER(md_energy_out)]
        lib.md_pressure.restype = C.c_int
        lib.md_pressure.argtypes = [C.c_void_p, C.POINTER(md_pressure_out)]
        lib.md_density_profile.restype = C.c_int
        lib.md_density_profile.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_longlong), C.c_int, C.c_double,
                                           C.POINTER(C.c_longlong)]
        lib.md_profile_step.restype = C.c_int
        lib.md_profile_step.argtypes = [C.c_void_p, C.c_longlong, C.POINTER(md_kernel_times)]
        lib.md_pair_tests.restype = C.c_int
        lib.md_pair_tests.argtypes = [C.c_void_p, C.POINTER(C.c_longlong)]
        lib.md_info.restype = C.c_int
        lib.md_info.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int * 3), C.POINTER(C.c_int)]
        lib.md_measure_peaks.restype = C.c_int
        lib.md_measure_peaks.argtypes = [C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(md_peaks)]
        lib.md_destroy.restype = C.c_int
        lib.md_destroy.argtypes = [C.c_void_p]
        lib.md_last_error.restype = C.c_char_p
        lib.md_last_error.argtypes = [C.c_void_p]
        lib.md_kinetic_energy_noalloc.restype = C.c_int
        lib.md_kinetic_energy_noalloc.argtypes = [C.c_void_p, C.c_longlong, C.c_int, C.c_double, C.c_void_p, C.c_void_p,
                                                  C.c_char_p, C.c_size_t]
        _lib = lib
    return _lib


def _structs(cfg, precision=64, algo=None):
    box, lj, opts = md_box(), md_lj(), md_opts()
    box.dim = int(cfg["dim"])
    for a in range(3):
        box.len[a] = float(cfg["box_len"][a])
        box.bc[a] = int(cfg["bc"][a])
    lj.eps, lj.sigma, lj.eps_w, lj.sigma_w = (float(cfg[k]) for k in ("eps", "sigma", "eps_w", "sigma_w"))
    lj.r_cut, lj.shift_energy = float(cfg["r_cut"]), int(cfg.get("shift_energy", 1))
    opts.dt, opts.mass, opts.precision = float(cfg["dt"]), float(cfg["mass"]), int(precision)
    opts.force_algo = _ALGO[algo if algo is not None else cfg.get("algo", "auto")]
    opts.skin = float(cfg.get("skin", 0.0))
    opts.tau_b, opts.t_target = float(cfg.get("tau_b", 0.0)), float(cfg.get("t_target", 1.0))
    opts.heavy_list = int(cfg.get("heavy_list", 0))
    opts.list_prunes = int(cfg.get("list_prunes", 0))
    return box, lj, opts


def _dptr(a):
    return a.ctypes.data_as(_DP) if a is not None else None


def workspace_bytes(cfg, precision=64, algo=None) -> int:
    box, lj, opts = _structs(cfg, precision, algo)
    return int(load_library().md_workspace_bytes(C.byref(box), C.byref(lj), C.byref(opts), int(cfg["n_vapor"]),
                                                 int(cfg["n_wall"])))


class Simulation:
    """md_create / md_step / md_get_state / md_energy on one GPU."""

    def __init__(self, cfg, precision=64, algo=None, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise MDError(MD_ERR_CUDA, "no CUDA device (there is no CPU fallback)")
        self._lib = load_library()
        self.dim = int(cfg["dim"])
        self.n_vapor = int(cfg["n_vapor"])
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        box, lj, opts = _structs(cfg, precision, algo)
        pos = np.ascontiguousarray(cfg["pos"], dtype=np.float64).reshape(-1, self.dim)
        vel = np.ascontiguousarray(cfg["vel"], dtype=np.float64).reshape(-1, self.dim)
        wall = np.ascontiguousarray(cfg["wall"], dtype=np.float64).reshape(-1, self.dim)
        n_wall = wall.shape[0]
        nbytes = self._lib.md_workspace_bytes(C.byref(box), C.byref(lj), C.byref(opts), self.n_vapor, n_wall)
        self.workspace = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=self.device)
        self.workspace.record_stream(self.stream)  # allocated on the current stream, used on self.stream
        torch.cuda.synchronize(self.device)
        self._h = C.c_void_p()
        pore = None
        if cfg.get("pore"):                       # dict(kind="cylinder"|"slit", axis, center, length, r0 | width)
            pd = cfg["pore"]
            pore = md_pore()
            pore.kind = {"slit": 1, "cylinder": 2, "prism": 5}[pd["kind"]]
            pore.axis = int(pd["axis"])
            for a, c in enumerate(pd["center"]):
                pore.center[a] = float(c)
            pore.length, pore.r0, pore.width = float(pd["length"]), float(pd.get("r0", 0.0)), float(pd.get("width", 0.0))
        rc = self._lib.md_create(C.byref(self._h), C.byref(box), C.byref(pore) if pore else None, C.byref(lj), C.byref(opts), self.n_vapor,
                                 _dptr(pos), _dptr(vel), n_wall, _dptr(wall) if n_wall else None,
                                 self.workspace.data_ptr(), self.workspace.numel(), self.stream.cuda_stream)
        if rc != MD_OK:
            self._h = C.c_void_p()
            raise MDError(rc, (self._lib.md_last_error(None) or b"").decode())

    def _check(self, rc):
        if rc != MD_OK:
            raise MDError(rc, (self._lib.md_last_error(self._h) or b"").decode())

    def step(self, n_steps: int):
        self._check(self._lib.md_step(self._h, int(n_steps)))

    def get_state(self, pos=True, vel=True, force=True, pe=True):
        n, d = self.n_vapor, self.dim
        out = {}
        bufs = [np.empty((n, d)) if f else None for f in (pos, vel, force)] + [np.empty(n) if pe else None]
        step = C.c_longlong()
        self._check(self._lib.md_get_state(self._h, *[_dptr(b) for b in bufs], C.byref(step)))
        for k, b in zip(("pos", "vel", "f", "pe"), bufs):
            if b is not None:
                out[k] = b
        out["step"] = step.value
        return out

    def energy(self):
        e = md_energy_out()
        self._check(self._lib.md_energy(self._h, C.byref(e)))
        return dict(K=e.kinetic, U=e.potential, U_vv=e.potential_vv, U_vw=e.potential_vw, virial=e.virial,
                    pairs_vv=e.pairs_vv, pairs_vw=e.pairs_vw, step=e.step)

    def pressure(self):
        o = md_pressure_out()
        self._check(self._lib.md_pressure(self._h, C.byref(o)))
        return dict(P_box=o.pressure_box, V_box=o.volume_box, P_pore=o.pressure_pore, V_pore=o.volume_pore,
                    K_pore=o.kinetic_pore, W_pore=o.virial_pore, n_pore=o.n_pore, step=o.step)

    def density_profile(self, n_axial: int, n_radial: int, r_max: float):
        """(axial counts, radial counts) about the pore of cfg["pore"], histogrammed on the device."""
        ax = np.zeros(max(n_axial, 1), dtype=np.int64)
        ra = np.zeros(max(n_radial, 1), dtype=np.int64)
        lp = C.POINTER(C.c_longlong)
        self._check(self._lib.md_density_profile(self._h, int(n_axial), ax.ctypes.data_as(lp), int(n_radial), float(r_max),
                                                 ra.ctypes.data_as(lp)))
        return ax[:n_axial], ra[:n_radial]

    def profile_step(self, n_steps: int):
        t = md_kernel_times()
        self._check(self._lib.md_profile_step(self._h, int(n_steps), C.byref(t)))
        return dict(ms=list(t.ms), launches=list(t.launches), total_ms=t.total_ms, steps=t.steps, rebuilds=t.rebuilds,
                    rebuild_ms=list(t.rebuild_ms), prunes=t.prunes, prune_ms=t.prune_ms)

    def pair_tests(self) -> int:
        v = C.c_longlong()
        self._check(self._lib.md_pair_tests(self._h, C.byref(v)))
        return v.value

    def info(self):
        algo, nc, kps = C.c_int(), (C.c_int * 3)(), C.c_int()
        self._check(self._lib.md_info(self._h, C.byref(algo), C.byref(nc), C.byref(kps)))
        return dict(algo={1: "allpairs", 2: "cells", 3: "verlet"}[algo.value], n_cells=list(nc), kernels_per_step=kps.value)

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.md_destroy(self._h)          # synchronises the stream: nothing runs on the workspace afterwards
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def measure_peaks(device="cuda:0", scratch_mib=512):
    import torch

    if not torch.cuda.is_available():
        raise MDError(MD_ERR_CUDA, "no CUDA device")
    lib = load_library()
    torch.cuda.set_device(device)
    buf = torch.empty(scratch_mib << 20, dtype=torch.uint8, device=device)
    st = torch.cuda.Stream(device=device)
    out = md_peaks()
    rc = lib.md_measure_peaks(buf.data_ptr(), buf.numel(), st.cuda_stream, C.byref(out))
    if rc != MD_OK:
        raise MDError(rc, "md_measure_peaks failed")
    return dict(fp64_tflops=out.fp64_tflops, fp32_tflops=out.fp32_tflops, copy_gbs=out.copy_gbs)


def kinetic_energy_noalloc(vel, mass, out, stream=None, n=None):
    """md_kinetic_energy_noalloc: K of the fp64 CUDA tensor `vel` [n, dim] into the one-element fp64 CUDA tensor `out`,
    asynchronously on `stream` (a torch.cuda.Stream; None = the legacy default stream).  Allocates nothing on the device:
    the reduction's scratch is a static array inside the library (at most NOALLOC_MAX_PARTICLES particles).  `n` overrides
    the particle count (argument checks)."""
    import torch

    if not (vel.is_cuda and out.is_cuda and vel.dtype == torch.float64 and out.dtype == torch.float64 and vel.is_contiguous()):
        raise ValueError("vel and out must be contiguous fp64 CUDA tensors")
    err = C.create_string_buffer(256)
    rc = load_library().md_kinetic_energy_noalloc(vel.data_ptr(), int(vel.shape[0] if n is None else n), int(vel.shape[1]),
                                                  float(mass), out.data_ptr(), stream.cuda_stream if stream is not None else None,
                                                  err, len(err))
    if rc != MD_OK:
        raise MDError(rc, err.value.decode())
