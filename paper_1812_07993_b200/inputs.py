"""Seeded synthetic input generators for the five pore configurations.

This module serves BOTH the CUDA path and the CPU oracle as *data*: it holds
none of the method's arithmetic (no Lennard-Jones term, no integrator, no cell
list).  It only places particles and draws velocities.

Recipe (stands in for the paper's workloads,
PAPER.md:115-125 (2D, 2184 molecules) and PAPER.md:186-188 (3D, 2800
molecules); the concrete sizes come from BASELINE.json configs[0..4]):

* RNG: counter-based splitmix64; k-th 64-bit output of a stream is
  mix(seed + (k+1)*GAMMA); uniform = top 53 bits / 2^53.
* wall particles: fixed lattices described per config below, centred in the box.
* vapor: cubic/square lattice over the whole box (n sites per side, the
  smallest n whose surviving sites number >= N_v), uniform jitter, sites whose
  jittered position is closer than 1.5 sigma to a wall particle rejected,
  N_v survivors chosen by sorting seeded random keys.
* velocities: Box-Muller normals, mean removed, rescaled so that
  2K / (d*N_v - d) = T* exactly.
"""
from __future__ import annotations

import math

import numpy as np

BASE_SEED = 181207993
_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

BC_PERIODIC = 0
BC_REFLECT = 1


class SplitMix64:
    """Counter-based splitmix64 stream (vectorised)."""

    def __init__(self, seed: int):
        self.seed = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)
        self.k = 0

    def bits(self, n: int) -> np.ndarray:
        with np.errstate(over="ignore"):
            ctr = np.arange(self.k + 1, self.k + n + 1, dtype=np.uint64)
            z = self.seed + ctr * _GAMMA
            z = (z ^ (z >> np.uint64(30))) * _M1
            z = (z ^ (z >> np.uint64(27))) * _M2
            z = z ^ (z >> np.uint64(31))
        self.k += n
        return z

    def uniform(self, n: int) -> np.ndarray:
        return (self.bits(n) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)

    def normal(self, n: int) -> np.ndarray:
        m = (n + 1) // 2
        u1 = self.uniform(m)
        u2 = self.uniform(m)
        r = np.sqrt(-2.0 * np.log(1.0 - u1))
        out = np.concatenate([r * np.cos(2.0 * math.pi * u2), r * np.sin(2.0 * math.pi * u2)])
        return out[:n]


# --------------------------------------------------------------------------
# wall lattices (all return arrays [N_w, dim], centred on `c`)
# --------------------------------------------------------------------------
def wall_slit2d_rows(c, n_per_row, n_per_wall, half_gap):
    """Two walls along x; rows filled outward from the slit faces at 1 sigma."""
    pts = []
    for sgn in (-1.0, 1.0):
        k = 0
        row = 0
        while k < n_per_wall:
            m = min(n_per_row, n_per_wall - k)
            x = c[0] - 0.5 * (n_per_row - 1) + np.arange(m)
            y = np.full(m, c[1] + sgn * (half_gap + row))
            pts.append(np.stack([x, y], axis=1))
            k += m
            row += 1
    return np.concatenate(pts)


def _ring(radius, n, phase, z, c):
    a = 2.0 * math.pi * (np.arange(n) + phase) / n
    return np.stack([c[0] + radius * np.cos(a), c[1] + radius * np.sin(a), np.full(n, z)], axis=1)


def wall_cylinder(c, radius, length, per_ring=31):
    """`length` rings 1 sigma apart along z, alternate rings rotated half a step."""
    nr = int(length)
    if nr <= 0:
        return np.zeros((0, 3))
    z0 = c[2] - 0.5 * (nr - 1)
    return np.concatenate([_ring(radius, per_ring, 0.5 * (k % 2), z0 + k, c) for k in range(nr)])


def wall_cone(c, r_a, r_b, length):
    nr = int(length)
    z0 = c[2] - 0.5 * (nr - 1)
    out = []
    for k in range(nr):
        rad = r_a + (r_b - r_a) * k / (nr - 1)
        out.append(_ring(rad, int(round(2.0 * math.pi * rad)), 0.5 * (k % 2), z0 + k, c))
    return np.concatenate(out)


def wall_inkbottle(c, r_neck, len_neck, r_body, len_body):
    """Neck (open top) -> shoulder annulus -> body -> closed bottom disc."""
    total = len_neck + len_body
    z0 = c[2] - 0.5 * (total - 1)
    out = []
    n_neck = int(round(2.0 * math.pi * r_neck))
    n_body = int(round(2.0 * math.pi * r_body))
    for k in range(len_neck):
        out.append(_ring(r_neck, n_neck, 0.5 * (k % 2), z0 + k, c))
    zs = z0 + len_neck - 0.5
    for rad in range(int(r_neck) + 1, int(r_body)):
        out.append(_ring(float(rad), int(round(2.0 * math.pi * rad)), 0.0, zs, c))
    for k in range(len_body):
        out.append(_ring(r_body, n_body, 0.5 * (k % 2), z0 + len_neck + k, c))
    zb = z0 + total
    out.append(np.array([[c[0], c[1], zb]]))
    for rad in range(1, int(r_body)):
        out.append(_ring(float(rad), int(round(2.0 * math.pi * rad)), 0.0, zb, c))
    return np.concatenate(out)


def wall_slit3d(c, gap, side=40):
    g = np.arange(side) - 0.5 * (side - 1)
    yy, zz = np.meshgrid(c[1] + g, c[2] + g, indexing="ij")
    out = []
    for sgn in (-1.0, 1.0):
        out.append(np.stack([np.full(yy.size, c[0] + sgn * 0.5 * gap), yy.ravel(), zz.ravel()], axis=1))
    return np.concatenate(out)


# --------------------------------------------------------------------------
# vapor placement and velocities
# --------------------------------------------------------------------------
def _min_wall_distance(pos, wall):
    if wall.shape[0] == 0:
        return np.full(pos.shape[0], np.inf)
    from scipy.spatial import cKDTree  # neighbour query for rejection only

    d, _ = cKDTree(wall).query(pos, k=1)
    return d


def place_vapor(rng, n_vapor, box_len, dim, wall, jitter, n_side=None, jitter_is_fraction=True, reject=1.5):
    """Jittered lattice over the whole box with wall rejection (module docstring)."""
    n = n_side if n_side is not None else int(math.ceil(n_vapor ** (1.0 / dim) - 1e-9))
    while True:
        a = np.array([box_len[d] / n for d in range(dim)])
        idx = np.indices((n,) * dim).reshape(dim, -1).T.astype(np.float64)
        sub = SplitMix64(int(rng.seed) ^ (0xA5A5A5A5 + n))
        u = sub.uniform(idx.shape[0] * dim).reshape(-1, dim)
        amp = jitter * a if jitter_is_fraction else np.full(dim, jitter)
        pos = (idx + 0.5) * a + (2.0 * u - 1.0) * amp
        keep = _min_wall_distance(pos, wall) >= reject
        if int(keep.sum()) >= n_vapor:
            break
        n += 1
    pos = pos[keep]
    keys = sub.uniform(pos.shape[0])
    pick = np.sort(np.argsort(keys, kind="stable")[:n_vapor])
    pos = np.ascontiguousarray(pos[pick])
    for d in range(dim):  # jitter never leaves the box (amp < a/2) but be safe
        np.clip(pos[:, d], 0.0, np.nextafter(box_len[d], 0.0), out=pos[:, d])
    return pos, n


def maxwell_boltzmann(rng, n, dim, t_star=1.0, mass=1.0):
    v = rng.normal(n * dim).reshape(n, dim) * math.sqrt(t_star / mass)
    if n > 1:
        v -= v.mean(axis=0)
        dof = dim * n - dim
        t_now = mass * float((v * v).sum()) / dof
        v *= math.sqrt(t_star / t_now)
    return np.ascontiguousarray(v)


def _finish(name, seed, dim, box_len, bc, wall, n_vapor, jitter, steps, algo, jit_frac=True, n_side=None, **extra):
    rng = SplitMix64(seed)
    L = [float(x) for x in box_len] + [1.0] * (3 - dim)
    bcs = list(bc) + [BC_PERIODIC] * (3 - dim)
    wall = np.ascontiguousarray(wall, dtype=np.float64).reshape(-1, dim)
    pos, n_side = place_vapor(rng, n_vapor, L, dim, wall, jitter, n_side=n_side, jitter_is_fraction=jit_frac)
    vel = maxwell_boltzmann(rng, n_vapor, dim)
    cfg = dict(name=name, seed=seed, dim=dim, box_len=L, bc=bcs, eps=1.0, sigma=1.0, eps_w=2.0, sigma_w=1.0,
               r_cut=2.5, shift_energy=1, dt=0.005, mass=1.0, pos=pos, vel=vel, wall=wall,
               n_vapor=n_vapor, n_wall=int(wall.shape[0]), lattice_side=n_side, steps=steps, algo=algo)
    cfg.update(extra)
    return cfg


# --------------------------------------------------------------------------
# the five configurations (BASELINE.json configs[0..4]; readings A18-A23 of DESIGN.md)
# --------------------------------------------------------------------------
def config0(seed=BASE_SEED):
    """2D slit, 1024 vapor + 2x(4 rows x 32) wall, 64x64 periodic, all-pairs, 200 steps."""
    c = (32.0, 32.0)
    wall = wall_slit2d_rows(c, 32, 128, 5.0)
    return _finish("cfg0_slit2d_1k", seed, 2, (64.0, 64.0), (BC_PERIODIC, BC_PERIODIC), wall, 1024, 0.2,
                   200, "allpairs", jit_frac=False, n_side=42)


def config1(seed=BASE_SEED + 1, n_vapor=16384):
    """2D slit 10 x 200 sigma, 16384 vapor + 4096 wall, 600x600, periodic x / reflecting y."""
    c = (300.0, 300.0)
    wall = wall_slit2d_rows(c, 200, 2048, 5.0)
    return _finish("cfg1_slit2d_16k", seed, 2, (600.0, 600.0), (BC_PERIODIC, BC_REFLECT), wall, n_vapor, 0.3,
                   10000, "cells", pore=dict(kind="slit", axis=1, center=c, length=200.0, width=10.0))


def cylinder_config(n_vapor, seed, name, steps=1000, algo="cells", density=0.05, box=None, length=None):
    """3D cylinder R=5 along z; box from density unless given; pore length min(40, floor(0.36 L))."""
    L = box if box is not None else (n_vapor / density) ** (1.0 / 3.0)
    length = length if length is not None else min(40, int(math.floor(0.36 * L)))
    c = (0.5 * L, 0.5 * L, 0.5 * L)
    wall = wall_cylinder(c, 5.0, length)
    return _finish(name, seed, 3, (L, L, L), (BC_PERIODIC, BC_PERIODIC, BC_REFLECT), wall, n_vapor, 0.3,
                   steps, algo, pore_length=length,
                   pore=dict(kind="cylinder", axis=2, center=c, length=float(length), r0=5.0) if length > 0 else None)


def config2(seed=BASE_SEED + 2):
    """3D cylindrical pore, 65536 vapor + 1240 wall, 110^3, periodic x,y / reflecting z."""
    return cylinder_config(65536, seed, "cfg2_cyl3d_64k", steps=10000, box=110.0, length=40)


def condense(cfg, side=12.0, density=0.6, corner=(14.0, 14.0, 14.0), name=None):
    """A 3D configuration with part of its vapor condensed: the vapor particles inside a cube of `side` at `corner` (far
    from the pore) are replaced, one for one, by a jittered simple-cubic lattice at liquid `density` filling the cube (the
    rest of the replaced particles come from the end of the array).  About 1,000 particles then have 60-90 neighbours within
    r_c + skin -- the state a long run reaches on the pore wall -- while N_v stays the same.  Velocities unchanged."""
    cfg = dict(cfg)
    rng = SplitMix64(cfg["seed"] + 77)
    a = density ** (-1.0 / 3.0)
    m = int(math.floor(side / a))
    grid = np.array([(i, j, k) for i in range(m) for j in range(m) for k in range(m)], dtype=np.float64)
    drop = np.array(corner) + 0.5 * a + a * grid + 0.1 * a * (rng.uniform(3 * len(grid)).reshape(-1, 3) * 2.0 - 1.0)
    pos = cfg["pos"].copy()
    lo, hi = np.array(corner) - 1.0, np.array(corner) + m * a + 1.0         # 1 sigma clear of the remaining vapor
    inside = np.nonzero(np.all((pos > lo) & (pos < hi), axis=1))[0]
    n = len(drop)
    assert len(inside) <= n < len(pos)
    taken = set(inside.tolist())
    outside_tail = [i for i in range(len(pos) - 1, -1, -1) if i not in taken][: n - len(inside)]
    idx = np.concatenate([inside, np.array(outside_tail, dtype=np.int64)])
    pos[idx] = drop
    cfg.update(name=name or cfg["name"] + "_condensed", pos=np.ascontiguousarray(pos), n_droplet=n)
    return cfg


def config2_condensed(seed=BASE_SEED + 2):
    """config 2 with 1,000 of its 65,536 vapor particles condensed into a droplet (see condense)."""
    return condense(config2(seed), name="cfg2_condensed")


def config3(shape, seed=None, n_vapor=262144):
    """3D pore-shape variants: shape in {'cone', 'inkbottle', 'slit'}."""
    k = ("cone", "inkbottle", "slit").index(shape)
    seed = BASE_SEED + 3 + 1000 * k if seed is None else seed
    L = (n_vapor / 0.05) ** (1.0 / 3.0)
    c = (0.5 * L, 0.5 * L, 0.5 * L)
    if shape == "cone":
        wall = wall_cone(c, 8.0, 3.0, 40)
    elif shape == "inkbottle":
        wall = wall_inkbottle(c, 3.0, 10, 8.0, 30)
    else:
        wall = wall_slit3d(c, 6.0, 40)
    return _finish("cfg3_%s_256k" % shape, seed, 3, (L, L, L), (BC_PERIODIC, BC_PERIODIC, BC_REFLECT), wall,
                   n_vapor, 0.3, 5000, "cells")


def config4(log2_n, seed=None, algo="cells"):
    """Scaling sweep: cylinder geometry, N_v = 2^log2_n at density 0.05."""
    k = (log2_n - 10) // 2
    seed = BASE_SEED + 4 + 1000 * k if seed is None else seed
    return cylinder_config(1 << log2_n, seed, "cfg4_cyl3d_2p%d" % log2_n, steps=1000, algo=algo)


def paper_size(dim, seed=BASE_SEED + 9):
    """Particle counts of the paper's own timing runs -- 2D: 420 + 1764 = 2184 molecules, 3D: 1000 +
    1800 = 2800 -- as a wall-free gas at the reduced density 0.05 of the other configurations (the
    paper's physical gas is ~1000x more dilute and uses no cut-off; this stands in for its SIZE only, to set a
    time per step beside Tables 1 and 4)."""
    n = 2184 if dim == 2 else 2800
    L = (n / 0.05) ** (1.0 / dim)
    bc = (BC_PERIODIC,) * dim
    return _finish("paper_size_%dd_%d" % (dim, n), seed + dim, dim, (L,) * dim, bc, np.zeros((0, dim)), n, 0.3, 2000,
                   "allpairs")


def paper_geometry(dim, seed=BASE_SEED + 20, n_pore=None):
    """The paper's own runs in reduced units (NEXT-3; readings A16 of DESIGN.md): a pore with GEOMETRIC reflecting walls
    (no wall particles), open at +x into an outer space with periodic boundaries, pore : outside density 5 : 1.
    2D: square pore 1 um x 1 um with 420 molecules, outer space 1764, 35 C.
    3D: prism 500 x 50 x 50 nm with 1000 molecules, outer space 1800 with 9x the volume, 25 C.
    dt = 0.016 ps = 0.00959 tau.  The gas is so dilute (4e-5 sigma^-2) that a cell grid would hold ~1e7 empty cells:
    the all-pairs kernel is the one to use, as in the paper.
    n_pore: molecules in the pore for the sweeps of Tables 2-3 (N = 100 ... 1500 "in the pore",
    pore : outside density ratio 5 : 1 kept): same geometry, 4.2 n_pore (2D) / 1.8 n_pore (3D) molecules outside, i.e.
    N_tot = 5.2 N / 2.8 N (reading A14)."""
    from . import units

    rng = SplitMix64(seed + dim)
    if dim == 2:
        l = units.length_reduced(1.0e-6)
        n_in, n_out, t_star = 420, 1764, units.temperature_reduced(35.0)
        if n_pore is not None:
            n_in, n_out = int(n_pore), int(round(4.2 * n_pore))
        box = (4.0 * l + 4.0, 7.0 * l)                              # pore + k = 3 pore widths of outer space, 2k + 1 tall
        lo, hi = np.array([2.0, 3.0 * l]), np.array([2.0 + l, 4.0 * l])
    else:
        lx, lw = units.length_reduced(500e-9), units.length_reduced(50e-9)
        n_in, n_out, t_star = 1000, 1800, units.temperature_reduced(25.0)
        if n_pore is not None:
            n_in, n_out = int(n_pore), int(round(1.8 * n_pore))
        box = (10.0 * lx + 4.0, lw + 4.0, lw + 4.0)                 # outer space: same cross-section, 9x the length
        lo, hi = np.array([2.0, 2.0, 2.0]), np.array([2.0 + lx, 2.0 + lw, 2.0 + lw])
    L = np.array(box)
    inside = lo + rng.uniform(n_in * dim).reshape(n_in, dim) * (hi - lo)
    outside = []
    while len(outside) < n_out:                                      # uniform in the box, outside the pore
        q = rng.uniform(dim) * L
        if not ((q > lo - 1.0) & (q < hi + 1.0)).all():
            outside.append(q)
    pos = np.ascontiguousarray(np.concatenate([inside, np.array(outside)]))
    vel = maxwell_boltzmann(rng, n_in + n_out, dim, t_star)
    Lp = [float(x) for x in box] + [1.0] * (3 - dim)
    return dict(name="paper_geometry_%dd_%d" % (dim, n_in + n_out), seed=seed, dim=dim, box_len=Lp,
                bc=[BC_PERIODIC] * 3, eps=1.0, sigma=1.0, eps_w=2.0, sigma_w=1.0, r_cut=2.5, shift_energy=1,
                dt=units.PAPER_DT, mass=1.0, pos=pos, vel=vel, wall=np.zeros((0, dim)), n_vapor=n_in + n_out, n_wall=0,
                steps=2000, algo="allpairs", t_star=t_star,
                pore=dict(kind="prism", axis=0, center=list(0.5 * (lo + hi)), length=float(hi[0] - lo[0]),
                          width=float(hi[1] - lo[1])))


def small_case(dim, n_vapor, box, bc, n_wall=0, seed=7, t_star=1.0, min_sep=0.9):
    """Small random dense-ish cases for tests: uniform positions with a minimum separation."""
    rng = SplitMix64(seed)
    L = [float(x) for x in box] + [1.0] * (3 - dim)
    pts = []
    tries = 0
    while len(pts) < n_vapor + n_wall:
        p = rng.uniform(dim) * np.array(L[:dim])
        tries += 1
        ok = True
        for q in pts:
            d = p - q
            for a in range(dim):
                if bc[a] == BC_PERIODIC:
                    d[a] -= L[a] * round(d[a] / L[a])
            if float(d @ d) < min_sep * min_sep:
                ok = False
                break
        if ok:
            pts.append(p)
        if tries > 200000:
            raise RuntimeError("small_case: cannot place particles")
    pts = np.array(pts).reshape(-1, dim)
    pos = np.ascontiguousarray(pts[:n_vapor])
    wall = np.ascontiguousarray(pts[n_vapor:])
    vel = maxwell_boltzmann(rng, n_vapor, dim, t_star)
    return dict(name="small", seed=seed, dim=dim, box_len=L, bc=list(bc) + [BC_PERIODIC] * (3 - dim), eps=1.0,
                sigma=1.0, eps_w=2.0, sigma_w=1.0, r_cut=2.5, shift_energy=1, dt=0.005, mass=1.0, pos=pos,
                vel=vel, wall=wall, n_vapor=n_vapor, n_wall=n_wall, steps=100, algo="allpairs")
