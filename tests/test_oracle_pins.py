"""Pins of the CPU oracle against what the mathematics fixes (no GPU, no CUDA path).

The paper prints no worked numerical example (PAPER.md has timings only), so every
pin is a closed form, an invariant, a special case or brute force.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import md_oracle as O
from paper_1812_07993_b200 import inputs as I

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "lj_closed_form.txt")


def base_cfg(dim=3, box=(20.0, 20.0, 20.0), bc=(0, 0, 0), **kw):
    L = list(box)[:dim] + [1.0] * (3 - dim)
    cfg = dict(dim=dim, box_len=L, bc=list(bc)[:dim] + [0] * (3 - dim), eps=1.0, sigma=1.0, eps_w=2.0, sigma_w=1.0,
               r_cut=2.5, shift_energy=0, dt=0.005, mass=1.0, pos=np.zeros((0, dim)), vel=np.zeros((0, dim)),
               wall=np.zeros((0, dim)))
    cfg.update(kw)
    return cfg


def pair(r, dim=3, wall=False, **kw):
    """Radial force on particle 0 (positive = repulsive) and total U for two sites r apart along x."""
    p0 = np.full(dim, 7.0)
    p1 = p0.copy()
    p0[0], p1[0] = r, 0.0          # exact separation r (no rounding in the subtraction)
    if wall:
        cfg = base_cfg(dim, pos=p0[None], wall=p1[None], **kw)
    else:
        cfg = base_cfg(dim, pos=np.stack([p0, p1]), **kw)
    out = O.forces(cfg)
    return out["f"][0, 0], out["U"], out


def golden_rows():
    rows = []
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            rows.append([float(x) for x in line.split()])
    return rows


def test_golden_rows_are_the_exact_rational_closed_form():
    for r, u, f in golden_rows():
        if abs(r - 2 ** (1 / 6)) < 1e-12:
            continue
        q = Fraction(r).limit_denominator(1000)
        ue = 4 * (q ** -12 - q ** -6)
        fe = 24 * (2 * q ** -12 - q ** -6) / q
        assert abs(float(ue) - u) <= 1e-14 * max(1.0, abs(u))
        assert abs(float(fe) - f) <= 1e-14 * max(1.0, abs(f))


@pytest.mark.parametrize("dim", [2, 3])
def test_two_particle_closed_form(dim):
    for r, u, f in golden_rows():
        if r >= 2.5:
            r = math.nextafter(2.5, 0.0)
        fo, uo, out = pair(r, dim)
        assert abs(uo - u) <= 2e-14 * max(1.0, abs(u)), (r, uo, u)
        assert abs(fo - f) <= 2e-13 * max(1.0, abs(f)), (r, fo, f)
        assert out["pairs_vv"] == 1 and out["pairs_vw"] == 0
        # Newton's third law on the pair, exactly antisymmetric
        assert out["f"][1, 0] == -out["f"][0, 0]
        # pe split half/half
        assert out["pe"][0] == out["pe"][1]


def test_force_is_minus_gradient_of_energy_sweep():
    # F = -dU/dr checked by Richardson-extrapolated central differences of the oracle's own U:
    # ties g to u (a wrong prefactor / exponent in either fails), u itself is tied by the rows above.
    rs = np.linspace(0.9, 2.49, 400)
    h = 1e-4
    for r in rs:
        f, _, _ = pair(r)
        d1 = (pair(r + h)[1] - pair(r - h)[1]) / (2 * h)
        d2 = (pair(r + 2 * h)[1] - pair(r - 2 * h)[1]) / (4 * h)
        dudr = (4 * d1 - d2) / 3
        assert abs(f + dudr) <= 1e-7 * max(1.0, abs(f)), (r, f, dudr)


def test_cutoff_strict_and_shift():
    f, u, out = pair(2.5)
    assert f == 0.0 and u == 0.0 and out["pairs_vv"] == 0
    f, u, out = pair(2.6)
    assert f == 0.0 and u == 0.0
    uc = golden_rows()[-1][1]
    _, u_sh, _ = pair(1.5, shift_energy=1)
    _, u_un, _ = pair(1.5, shift_energy=0)
    assert abs((u_un - u_sh) - uc) < 1e-15
    _, u_edge, _ = pair(math.nextafter(2.5, 0.0), shift_energy=1)
    assert abs(u_edge) < 1e-14  # continuous at r_c when shifted


def test_wall_closed_form():
    for r, u, f in golden_rows():
        if r >= 2.5:
            r = math.nextafter(2.5, 0.0)
        fo, uo, out = pair(r, wall=True)
        assert abs(uo - 2 * u) <= 4e-14 * max(1.0, abs(u))       # eps_w = 2: full share to the vapor particle
        assert abs(fo - 2 * f) <= 4e-13 * max(1.0, abs(f))
        assert out["pairs_vv"] == 0 and out["pairs_vw"] == 1
        assert out["pe_w"][0] == out["pe"][0]
    # sigma_w enters as sigma_w/r: sigma_w = 1.1 at r = 1.1 * 1.5 reproduces U(1.5) * eps_w
    _, u, _ = pair(1.65, wall=True, sigma_w=1.1, r_cut=3.0)
    assert abs(u - 2 * golden_rows()[2][1]) < 1e-13


def test_newton_third_law_and_momentum():
    cfg = I.small_case(3, 300, (9.0, 9.0, 9.0), (0, 0, 0), seed=11)
    out = O.forces(cfg)
    assert out["pairs_vv"] > 1000
    net = np.abs(out["f"].sum(axis=0)).max() / np.abs(out["f"]).sum()
    assert net <= 1e-12
    p0 = cfg["vel"].sum(axis=0)
    run = O.run(cfg, 200)
    assert np.abs(run["vel"].sum(axis=0) - p0).max() < 1e-11


def test_translation_invariance_and_minimum_image():
    cfg = I.small_case(3, 200, (8.0, 9.5, 11.0), (0, 0, 0), n_wall=30, seed=5)
    ref = O.forces(cfg)
    shift = np.array([3.3, -17.1, 5.55])
    L = np.array(cfg["box_len"])
    moved = dict(cfg)
    moved["pos"] = np.mod(cfg["pos"] + shift, L)
    moved["wall"] = np.mod(cfg["wall"] + shift, L)
    out = O.forces(moved)
    assert out["pairs_vv"] == ref["pairs_vv"] and out["pairs_vw"] == ref["pairs_vw"]
    scale = np.abs(ref["f"]).max()
    assert np.abs(out["f"] - ref["f"]).max() <= 1e-11 * scale
    assert abs(out["U"] - ref["U"]) <= 1e-11 * abs(ref["U"])


def test_pair_across_periodic_face_and_not_across_reflecting_face():
    rows = golden_rows()
    r, u, f = rows[2]  # r = 1.5
    for bc, hit in ((0, True), (1, False)):
        cfg = base_cfg(3, box=(20.0, 20.0, 20.0), bc=(bc, 0, 0),
                       pos=np.array([[0.5, 7.0, 7.0], [19.0, 7.0, 7.0]]))
        out = O.forces(cfg)
        if hit:
            assert abs(out["U"] - u) < 1e-13
            assert abs(out["f"][0, 0] - f) < 1e-12       # particle 0 is at +1.5 from the image of particle 1
            assert abs(out["f"][1, 0] + f) < 1e-12
        else:
            assert out["U"] == 0.0 and out["pairs_vv"] == 0


def test_free_flight_wrap_and_reflect():
    cfg = I.small_case(3, 50, (6.0, 7.0, 8.0), (0, 0, 1), n_wall=5, seed=3)
    cfg["eps"] = cfg["eps_w"] = 0.0
    cfg["dt"] = 0.01
    cfg["vel"] = cfg["vel"] * 4.0
    n = 700
    out = O.run(cfg, n)
    L = np.array(cfg["box_len"])
    t = n * cfg["dt"]
    free = cfg["pos"] + cfg["vel"] * t
    exp = free.copy()
    exp[:, :2] = np.mod(free[:, :2], L[:2])
    z = np.mod(free[:, 2], 2 * L[2])                      # triangular wave
    exp[:, 2] = np.where(z > L[2], 2 * L[2] - z, z)
    d = out["pos"] - exp
    d[:, :2] -= L[:2] * np.rint(d[:, :2] / L[:2])
    assert np.abs(d).max() < 1e-11
    assert np.allclose(np.abs(out["vel"]), np.abs(cfg["vel"]), rtol=0, atol=1e-13)
    assert (np.sign(out["vel"][:, 2]) != np.sign(cfg["vel"][:, 2])).any()   # some did bounce
    assert (out["pos"] >= 0).all() and (out["pos"][:, :2] < L[:2]).all() and (out["pos"][:, 2] <= L[2]).all()


def _period(x, dt):
    x = x - x.mean()
    up = [i for i in range(len(x) - 1) if x[i] < 0 <= x[i + 1]]
    t = [i + (-x[i]) / (x[i + 1] - x[i]) for i in up]
    return dt * (t[-1] - t[0]) / (len(t) - 1)


def test_bound_pair_harmonic_period():
    # U''(r_min) = 57.1464 eps/sigma^2 (= 72 * 2^(-1/3)); two free particles: mu = 1/2; vapor-wall: eps_w = 2, mu = 1
    kpp = 72.0 * 2.0 ** (-1.0 / 3.0)
    r0, delta, dt = 2.0 ** (1.0 / 6.0), 1e-3, 0.005
    for wall in (False, True):
        a = np.array([[5.0, 5.0, 5.0]])
        b = np.array([[5.0 + r0 + delta, 5.0, 5.0]])
        if wall:
            cfg = base_cfg(3, pos=b, vel=np.zeros((1, 3)), wall=a, dt=dt)
            omega = math.sqrt(2.0 * kpp / 1.0)
        else:
            cfg = base_cfg(3, pos=np.concatenate([a, b]), vel=np.zeros((2, 3)), dt=dt)
            omega = math.sqrt(kpp / 0.5)
        xs, pos, vel = [], cfg["pos"], cfg["vel"]
        for _ in range(600):
            o = O.run(cfg, 1, pos=pos, vel=vel)
            pos, vel = o["pos"], o["vel"]
            xs.append(pos[-1, 0] - (5.0 if wall else pos[0, 0]))
        xs = np.array(xs)
        T = _period(xs, dt)
        assert abs(T - 2 * math.pi / omega) / T < 2e-3          # O(delta) anharmonic + O(dt^2)
        amp = 0.5 * (xs.max() - xs.min())
        assert abs(amp - delta) / delta < 2e-2
        if not wall:
            assert abs(2 * math.pi / omega - 0.5877) < 1e-4      # = 117.5 steps of dt = 0.005


def _energy_error(cfg, t_end, dt):
    c = dict(cfg)
    c["dt"] = dt
    h = O.run(c, int(round(t_end / dt)), history=True)["hist"]
    e = h[:, 0] + h[:, 1] + h[:, 2]
    return e - e[0]


def test_energy_error_is_second_order_in_dt():
    # A cluster in the middle of a big box, r_cut beyond every pair: no cut-off crossing and no bounce,
    # so the smooth-Hamiltonian result holds: E(t; dt) - E(0) = dt^2 g(t) + O(dt^4)  => ratio 4.
    # (With the plainly truncated force of reading A2 every r_c crossing adds an O(dt) kink, and a
    # specular bounce likewise; both are measured, not pinned.)
    cfg = I.small_case(3, 64, (6.0, 6.0, 6.0), (1, 1, 1), n_wall=8, seed=21, min_sep=1.0)
    cfg["r_cut"], cfg["box_len"] = 100.0, [30.0, 30.0, 30.0]
    cfg["pos"], cfg["wall"] = cfg["pos"] + 12.0, cfg["wall"] + 12.0
    a, b = _energy_error(cfg, 0.4, 0.004), _energy_error(cfg, 0.4, 0.002)
    ratio = np.sqrt((a ** 2).mean() / (b[::2] ** 2).mean())
    assert abs(ratio - 4.0) < 0.1, ratio


def test_time_reversibility():
    cfg = I.small_case(3, 150, (8.0, 8.0, 8.0), (0, 0, 1), n_wall=10, seed=9)
    fwd = O.run(cfg, 100)
    back = O.run(cfg, 100, pos=fwd["pos"], vel=-fwd["vel"])
    d = back["pos"] - cfg["pos"]
    L = np.array(cfg["box_len"])
    d -= L * np.rint(d / L) * (np.array(cfg["bc"]) == 0)
    assert np.abs(d).max() < 1e-10
    assert np.abs(back["vel"] + cfg["vel"]).max() < 1e-10


@pytest.mark.parametrize("dim,box,bc,seed", [
    (3, (8.0, 9.3, 7.6), (0, 0, 0), 1), (3, (8.1, 7.5, 5.2), (0, 0, 1), 2), (3, (4.0, 8.0, 8.0), (1, 0, 0), 3),
    (2, (13.7, 9.9), (0, 1), 4), (2, (7.5, 7.5), (0, 0), 5), (2, (2.6, 30.0), (1, 0), 6)])
def test_cell_list_equals_brute_force(dim, box, bc, seed):
    vol = float(np.prod(box))
    n_wall = 40 if dim == 3 else 12
    n_vapor = min(300, int((0.5 if dim == 3 else 0.45) * vol) - n_wall)
    cfg = I.small_case(dim, n_vapor, box, bc, n_wall=n_wall, seed=seed, min_sep=0.9)
    L = cfg["box_len"]
    ra = O.run(cfg, 20)
    rb = O.run(cfg, 20, cells=True)
    assert np.abs(ra["pos"] - rb["pos"]).max() < 1e-9
    cfg["pos"] = cfg["pos"].copy()
    # put particles on cell faces, at 0 and (reflecting) at L
    cfg["pos"][0, 0] = 0.0
    cfg["pos"][1, 0] = L[0] / math.floor(L[0] / 2.5) if L[0] >= 5 else 0.0
    cfg["pos"][2, 1] = 2 * (L[1] / math.floor(L[1] / 2.5))
    if bc[0] == 1:
        cfg["pos"][3, 0] = L[0]
    a, b = O.forces(cfg), O.forces(cfg, cells=True)
    assert a["pairs_vv"] == b["pairs_vv"] and a["pairs_vw"] == b["pairs_vw"] and a["pairs_vv"] > 20
    scale = np.abs(a["f"]).max()
    assert np.abs(a["f"] - b["f"]).max() <= 1e-13 * scale
    assert np.abs(a["pe"] - b["pe"]).max() <= 1e-13 * np.abs(a["pe"]).max()
    assert np.abs(a["vir"] - b["vir"]).max() <= 1e-13 * np.abs(a["vir"]).max()


def test_cell_list_rejects_thin_periodic_box():
    cfg = I.small_case(2, 10, (6.0, 20.0), (0, 0), seed=2)
    with pytest.raises(ValueError):
        O.forces(cfg, cells=True)


def test_energy_matches_scipy_pdist_sum():
    from scipy.spatial.distance import pdist
    cfg = I.small_case(3, 60, (4.0, 4.0, 4.0), (1, 1, 1), seed=13, min_sep=0.95)   # no periodic images
    cfg["r_cut"], cfg["shift_energy"] = 100.0, 0
    out = O.forces(cfg)
    r = pdist(cfg["pos"])
    u = float((4.0 * (r ** -12 - r ** -6)).sum())
    assert abs(out["U"] - u) <= 1e-12 * abs(u)
    vir = float((24.0 * (2 * r ** -12 - r ** -6)).sum())   # sum_{i<j} r.F
    assert abs(out["vir"].sum() - vir) <= 1e-12 * abs(vir)


def test_uniform_gas_pair_count_poisson():
    rng = I.SplitMix64(99)
    n, L = 20000, 60.0
    cfg = base_cfg(3, box=(L, L, L), pos=rng.uniform(3 * n).reshape(n, 3) * L)
    cfg["eps"] = 0.0
    out = O.forces(cfg, cells=True)
    expect = 0.5 * n * (n / L ** 3) * (4 * math.pi / 3) * 2.5 ** 3
    assert abs(out["pairs_vv"] - expect) < 5 * math.sqrt(expect)


def test_energy_conservation_dilute_gas_10k_steps():
    # reading A8: drift := (<E>_last1000 - <E>_{1000..2000}) / K(0) on the dilute 3D gas, shifted energy.  The force is
    # plainly truncated (A2), so every r_c crossing leaves a small energy kink of either sign: the statistic is a
    # zero-mean random walk whose rms over realisations falls as 1/sqrt(N) -- measured over 16 seeds at N = 1728: mean
    # 5e-6, rms 1.5e-4 (rms sqrt(N) = 6.3e-3); 8 seeds at N = 4096: 1.1e-4.  north_star's "below 1e-4" is therefore a
    # statement about large N (rms 2.5e-5 at the 65,536 particles of the metric's workload, checked on the GPU); a single
    # realisation at N = 1728 (3.8e-5 for seed 4242) passing 1e-4 is luck, so the pin is on the distribution:
    # six seeds, rms within a factor 3 of the law, both signs present, and no run wanders beyond 1e-3 K(0) at any step.
    n, ds = 1728, []
    for seed in range(4242, 4248):
        cfg = I.cylinder_config(n, seed, "drift", box=(n / 0.05) ** (1 / 3), length=0)
        assert cfg["n_wall"] == 0
        h = O.run(cfg, 10000, cells=True, history=True)["hist"]
        e = h[:, 0] + h[:, 1] + h[:, 2]
        ds.append((e[-1000:].mean() - e[1000:2000].mean()) / h[0, 0])
        assert np.abs(e - e[0]).max() / h[0, 0] < 1e-3
    ds = np.array(ds)
    rms, law = np.sqrt((ds ** 2).mean()), 6.4e-3 / math.sqrt(n)
    assert law / 3 <= rms <= 3 * law, ds
    assert ds.min() < 0 < ds.max(), ds


def test_berendsen_thermostat_closed_forms():
    # F4.  Without forces K only changes through lambda, so T_{n+1} = T_n lambda^2 =
    # T_n + (dt/tau)(T_0 - T_n) exactly:  T_n = T_0 + (T_init - T_0)(1 - dt/tau)^n.
    cfg = I.small_case(3, 200, (12.0, 12.0, 12.0), (0, 0, 1), n_wall=6, seed=17, t_star=2.5)
    cfg["eps"] = cfg["eps_w"] = 0.0
    n, dim = cfg["n_vapor"], 3
    t_init = 2.0 * O.kinetic(cfg, cfg["vel"]) / (dim * n)
    cfg.update(tau_b=0.1, t_target=1.2, dt=0.005)
    h = O.run(cfg, 60, history=True)["hist"]
    t = 2.0 * h[:, 0] / (dim * n)
    expect = 1.2 + (t_init - 1.2) * (1.0 - 0.005 / 0.1) ** np.arange(61)
    assert np.abs(t - expect).max() < 1e-12 * t_init
    # tau_B = dt reaches T_0 in one step; T = T_0 leaves the dynamics untouched (lambda = 1)
    cfg.update(tau_b=0.005)
    h = O.run(cfg, 2, history=True)["hist"]
    assert abs(2.0 * h[1, 0] / (dim * n) - 1.2) < 1e-13
    lj = I.small_case(3, 150, (8.0, 8.0, 8.0), (0, 0, 1), n_wall=10, seed=9)
    nve = O.run(lj, 1)
    t1 = 2.0 * nve["K"] / (3 * 150)
    thermo = dict(lj, tau_b=0.3, t_target=t1)
    out = O.run(thermo, 1)
    assert np.abs(out["vel"] - nve["vel"]).max() < 1e-14
    # with forces on, a cold target pulls the system to T_0 within a few tau_B and holds it there
    cold = dict(lj, tau_b=0.05, t_target=0.3)
    hh = O.run(cold, 300, history=True)["hist"]
    tt = 2.0 * hh[:, 0] / (3 * 150)
    assert tt[0] > 0.9 and np.abs(tt[50:] - 0.3).max() < 0.06


def _prism_cfg(dim, pos, vel, axis=0, center=None, length=6.0, width=4.0, box=20.0, dt=0.01):
    cfg = base_cfg(dim, box=(box,) * dim, bc=(0,) * dim, pos=np.array(pos, dtype=float), vel=np.array(vel, dtype=float), dt=dt)
    cfg["eps"] = cfg["eps_w"] = 0.0
    cfg["pore"] = dict(kind="prism", axis=axis, center=center or [10.0] * dim, length=length, width=width)
    return cfg


def test_geometric_prism_pore_free_flight():
    # NEXT-3: the paper's pore: closed faces reflect from both sides, the +axis face is open.
    # 2D pore [7, 13] x [8, 12], open at x = 13.  Free flight => closed forms.
    # (a) bouncing between the side walls y = 8 and y = 12: triangular wave, |v| unchanged, x untouched
    cfg = _prism_cfg(2, [[9.0, 10.0]], [[0.0, 3.0]])
    out = O.run(cfg, 1000)
    t = 1000 * 0.01
    y = (10.0 - 8.0 + 3.0 * t) % 8.0
    y = 8.0 + (y if y <= 4.0 else 8.0 - y)
    assert abs(out["pos"][0, 1] - y) < 1e-10 and abs(out["pos"][0, 0] - 9.0) < 1e-12 and abs(abs(out["vel"][0, 1]) - 3.0) < 1e-14
    # (b) towards the closed end x = 7: comes back and leaves through the open mouth at x = 13, then keeps going
    cfg = _prism_cfg(2, [[9.0, 10.0]], [[-2.0, 0.0]])
    out = O.run(cfg, 250)                                   # 2.5 time units: 1 to the wall, 1.5 back => x = 7 + 3 = 10
    assert abs(out["pos"][0, 0] - 10.0) < 1e-10 and out["vel"][0, 0] == 2.0
    out = O.run(cfg, 500)
    assert abs(out["pos"][0, 0] - 15.0) < 1e-10            # x = 7 + 2 * 4: no wall at the mouth (x = 13)
    # (c) from outside: hits the side wall y = 12 from above and bounces back; beside the pore it flies on
    cfg = _prism_cfg(2, [[10.0, 14.0], [4.0, 14.0]], [[0.0, -1.0], [0.0, -1.0]])
    out = O.run(cfg, 400)
    assert abs(out["pos"][0, 1] - 14.0) < 1e-10 and out["vel"][0, 1] == 1.0     # 2 down, 2 back up
    assert abs(out["pos"][1, 1] - 10.0) < 1e-10 and out["vel"][1, 1] == -1.0    # x = 4 is outside [7, 13]
    # (d) enters through the mouth from the right and is turned round at the closed end
    cfg = _prism_cfg(2, [[16.0, 10.5]], [[-3.0, 0.0]])
    out = O.run(cfg, 500)                                   # 15 units of path: 9 to x = 7, 6 back => x = 13
    assert abs(out["pos"][0, 0] - 13.0) < 1e-10 and out["vel"][0, 0] == 3.0
    # (e) 3D prism along z, open at +z: corner bounce flips two components in one step
    cfg = _prism_cfg(3, [[11.9, 11.9, 10.0]], [[2.0, 2.0, 0.0]], axis=2, dt=0.1)
    out = O.run(cfg, 1)
    assert np.allclose(out["pos"][0], [11.9, 11.9, 10.0], atol=1e-12) and np.array_equal(out["vel"][0], [-2.0, -2.0, 0.0])
    # (f) with interactions on, the walls do no work: energy drift stays at the NVE level
    lj = I.small_case(2, 30, (20.0, 20.0), (0, 0), seed=5, min_sep=1.0)
    lj["pore"] = dict(kind="prism", axis=0, center=[10.0, 10.0], length=8.0, width=6.0)
    h = O.run(lj, 2000, history=True)["hist"]
    e = h[:, 0] + h[:, 1] + h[:, 2]
    assert np.abs(e - e[0]).max() < 2e-3 * h[0, 0]


# ---- parameters away from 1 (m_i, sigma and epsilon are parameters of the model) ---------------------
# Every pin above runs with mass = sigma = eps = 1, where a slip such as hk = dt*m/2, K = v^2/2 or a wrong power of
# sigma in g is invisible.  The pins below use m = 2.5, sigma = 1.3, eps = 0.7, sigma_w = 1.1, eps_w = 1.6.
M, SIG, EPS, SIGW, EPSW = 2.5, 1.3, 0.7, 1.1, 1.6


def test_scaled_parameters_pair_closed_form():
    # U(r; eps, sigma) = eps U_1(r / sigma), F(r; eps, sigma) = (eps / sigma) F_1(r / sigma), virial = F r:
    # golden rows (eps = sigma = 1) evaluated at r / sigma
    for x, u1, f1 in golden_rows():
        if x >= 2.5:
            continue
        for wall, eps, sig in ((False, EPS, SIG), (True, EPSW, SIGW)):
            r = x * sig
            fo, uo, out = pair(r, wall=wall, eps=EPS, sigma=SIG, eps_w=EPSW, sigma_w=SIGW, r_cut=4.0)
            assert abs(uo - eps * u1) <= 4e-14 * max(1.0, abs(u1)), (x, wall)
            assert abs(fo - eps / sig * f1) <= 4e-13 * max(1.0, abs(f1)), (x, wall)
            w = out["vir"].sum()
            assert abs(w - eps / sig * f1 * r) <= 1e-12 * max(1.0, abs(f1))
    # zero force at r = 2^(1/6) sigma, for both pair types
    for wall, sig in ((False, SIG), (True, SIGW)):
        fo, _, _ = pair(2.0 ** (1.0 / 6.0) * sig, wall=wall, eps=EPS, sigma=SIG, eps_w=EPSW, sigma_w=SIGW, r_cut=4.0)
        assert abs(fo) < 1e-13
    # the shift is u(r_cut) of the same (eps, sigma): 4 eps [(sigma / r_c)^12 - (sigma / r_c)^6], by rational arithmetic
    for wall, eps, sig in ((False, Fraction(7, 10), Fraction(13, 10)), (True, Fraction(8, 5), Fraction(11, 10))):
        q = sig / Fraction(3)
        uc = float(4 * eps * (q ** 12 - q ** 6))
        kw = dict(wall=wall, eps=EPS, sigma=SIG, eps_w=EPSW, sigma_w=SIGW, r_cut=3.0)
        _, u_un, _ = pair(2.0, shift_energy=0, **kw)
        _, u_sh, _ = pair(2.0, shift_energy=1, **kw)
        assert abs((u_un - u_sh) - uc) < 1e-15


def test_kinetic_energy_and_first_step_with_mass():
    # K = 1/2 m |v|^2 on hand-set velocities: 1/2 * 2.5 * (1 + 4 + 9) + 1/2 * 2.5 * 4 = 22.5
    cfg = base_cfg(3, mass=M, pos=np.array([[5.0, 5.0, 5.0], [12.0, 5.0, 5.0]]), vel=np.array([[1.0, 2.0, 3.0], [0.0, -2.0, 0.0]]))
    assert O.kinetic(cfg, cfg["vel"]) == 22.5
    # one step from rest: v(dt/2) = (dt / 2m) F, r(dt) = r + dt v(dt/2) = r + dt^2 F / (2 m): F2 of PAPER.md:79-80 with
    # a = F / m (Eq. (1)).  Two particles 1.5 sigma apart, eps = 0.7, sigma = 1.3.
    r = 1.5 * SIG
    f = EPS / SIG * golden_rows()[2][2]
    dt = 0.005
    cfg = base_cfg(3, mass=M, eps=EPS, sigma=SIG, r_cut=4.0, dt=dt, pos=np.array([[5.0 + r, 5.0, 5.0], [5.0, 5.0, 5.0]]),
                   vel=np.zeros((2, 3)))
    out = O.run(cfg, 1)
    assert abs((out["pos"][0, 0] - (5.0 + r)) - dt * dt * f / (2 * M)) < 1e-15
    assert abs((out["pos"][1, 0] - 5.0) + dt * dt * f / (2 * M)) < 1e-15
    # after the step v(dt) = (dt / 2m)(F(0) + F(dt)), F(dt) from the closed form at the new separation
    r1 = out["pos"][0, 0] - out["pos"][1, 0]
    x = r1 / SIG
    f_new = EPS / SIG * 24.0 * (2.0 * x ** -12 - x ** -6) / x
    assert abs(out["vel"][0, 0] - dt / (2 * M) * (f + f_new)) < 1e-15


def test_bound_pair_period_scales_with_mass_sigma_eps():
    # omega = sqrt(U''(r_min) / mu), U''(r_min) = 72 * 2^(-1/3) eps / sigma^2: period proportional to sqrt(m sigma^2 / eps)
    kpp = 72.0 * 2.0 ** (-1.0 / 3.0)
    dt, delta = 0.005, 1e-3
    for wall in (False, True):
        eps, sig = (EPSW, SIGW) if wall else (EPS, SIG)
        r0 = 2.0 ** (1.0 / 6.0) * sig
        a = np.array([[5.0, 5.0, 5.0]])
        b = np.array([[5.0 + r0 + delta, 5.0, 5.0]])
        kw = dict(mass=M, eps=EPS, sigma=SIG, eps_w=EPSW, sigma_w=SIGW, r_cut=4.0, dt=dt)
        if wall:
            cfg = base_cfg(3, pos=b, vel=np.zeros((1, 3)), wall=a, **kw)
            omega = math.sqrt(kpp * eps / sig ** 2 / M)
        else:
            cfg = base_cfg(3, pos=np.concatenate([a, b]), vel=np.zeros((2, 3)), **kw)
            omega = math.sqrt(kpp * eps / sig ** 2 / (0.5 * M))
        xs, pos, vel = [], cfg["pos"], cfg["vel"]
        for _ in range(1400):
            o = O.run(cfg, 1, pos=pos, vel=vel)
            pos, vel = o["pos"], o["vel"]
            xs.append(pos[-1, 0] - (5.0 if wall else pos[0, 0]))
        T = _period(np.array(xs), dt)
        assert abs(T - 2 * math.pi / omega) / T < 2e-3, (wall, T, 2 * math.pi / omega)


def test_dimensional_scaling_maps_onto_reduced_units():
    # Lengths x sigma, energies x eps, masses x m, times x sigma sqrt(m / eps): the run with (m, sigma, eps) on the
    # scaled input is the reduced-unit run (which the pins above fix) scaled back.  Exact in real arithmetic, so the
    # two differ by rounding only; any wrong power of m, sigma or eps in hk, K, g or u shows as an O(1) difference.
    cfg = I.small_case(3, 120, (8.0, 9.0, 7.6), (0, 0, 1), n_wall=20, seed=31, min_sep=0.95)
    cfg["eps_w"] = 1.6
    tau = SIG * math.sqrt(M / EPS)
    big = dict(cfg, pos=cfg["pos"] * SIG, wall=cfg["wall"] * SIG, vel=cfg["vel"] * SIG / tau,
               box_len=[x * SIG for x in cfg["box_len"]], r_cut=cfg["r_cut"] * SIG, dt=cfg["dt"] * tau, mass=M,
               eps=EPS, sigma=SIG, eps_w=1.6 * EPS, sigma_w=SIG)
    n = 60
    a, b = O.run(cfg, n, history=True), O.run(big, n, history=True)
    assert np.abs(b["pos"] / SIG - a["pos"]).max() < 1e-9
    assert np.abs(b["vel"] * tau / SIG - a["vel"]).max() < 1e-8
    assert np.abs(b["f"] * SIG / EPS - a["f"]).max() <= 1e-8 * np.abs(a["f"]).max()
    assert abs(b["K"] / EPS - a["K"]) < 1e-9 * a["K"] and abs(b["U"] / EPS - a["U"]) < 1e-9 * abs(a["U"])
    assert np.array_equal(a["hist"][:, 3:], b["hist"][:, 3:])          # pair counts step by step
    assert np.abs(b["vir"] / EPS - a["vir"]).max() < 1e-8 * np.abs(a["vir"]).max()
    # and the thermostat's temperature uses K with the mass in it: T = 2K / (d N), same lambda in both unit systems
    ta = O.run(dict(cfg, tau_b=0.05, t_target=0.5), n)
    tb = O.run(dict(big, tau_b=0.05 * tau, t_target=0.5 * EPS), n)
    assert np.abs(tb["vel"] * tau / SIG - ta["vel"]).max() < 1e-8


def test_free_flight_is_independent_of_mass():
    cfg = I.small_case(3, 40, (6.0, 7.0, 8.0), (0, 0, 1), n_wall=0, seed=3)
    cfg["eps"] = cfg["eps_w"] = 0.0
    a, b = O.run(cfg, 300), O.run(dict(cfg, mass=M), 300)
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["vel"], b["vel"])
    assert abs(b["K"] - M * a["K"]) < 1e-12 * b["K"]
