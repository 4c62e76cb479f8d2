"""Error metrics of DESIGN.md "Tolerances" shared by the parity tests."""
import numpy as np


def force_error(f_gpu, f_cpu):
    """max_i ||f_gpu_i - f_cpu_i||_inf / max(||f_cpu_i||_inf, 1e-3 f_rms); zero-force particles must be exactly zero."""
    mag = np.abs(f_cpu).max(axis=1)
    nz = mag > 0
    frms = np.sqrt((f_cpu[nz] ** 2).sum(axis=1).mean()) if nz.any() else 1.0
    err = np.abs(f_gpu - f_cpu).max(axis=1) / np.maximum(mag, 1e-3 * frms)
    assert (f_gpu[~nz] == 0).all(), "a particle with no neighbour has a non-zero force"
    return float(err.max())


def scalar_error(a_gpu, a_cpu):
    mag = np.abs(a_cpu)
    nz = mag > 0
    rms = np.sqrt((a_cpu[nz] ** 2).mean()) if nz.any() else 1.0
    return float((np.abs(a_gpu - a_cpu) / np.maximum(mag, 1e-3 * rms)).max())


def traj_error(p_gpu, p_cpu, box_len, bc):
    d = p_gpu - p_cpu
    for a in range(d.shape[1]):
        if bc[a] == 0:
            d[:, a] -= box_len[a] * np.rint(d[:, a] / box_len[a])
    return float(np.abs(d).max())
