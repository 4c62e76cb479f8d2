"""GPU parity: CUDA path (through the C ABI) vs the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; metrics in tests/parity.py):
forces / per-particle energies <= 1e-10 relative in fp64 (<= 1e-4 in fp32), pair counts exact,
trajectories <= 1e-8 sigma after 100 steps.
"""
import numpy as np
import pytest
import torch

from oracle import md_oracle as O
from paper_1812_07993_b200 import inputs as I
from paper_1812_07993_b200 import md
from parity import force_error, scalar_error, traj_error

pytestmark = pytest.mark.gpu

FTOL, TRAJ_TOL = 1e-10, 1e-8


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    md.load_library()


def make_sim(cfg, algo, precision=64):
    try:
        return md.Simulation(cfg, precision=precision, algo=algo)
    except md.MDError as e:
        if e.code == md.MD_ERR_UNSUPPORTED and algo in ("verlet", "cells"):
            pytest.skip("%s needs >= 3 cells per periodic dimension in this box" % algo)
        raise


def _cutoff_bracket(cfg, cells):
    """fp32 mode takes the strict r^2 < r_c^2 decision in fp32 (the kernel's precision), the oracle in fp64: a pair whose
    r^2 lies within the fp32 rounding of r_c^2 (three roundings of 2^-24 in the fma chain; the differences themselves are
    exact) may fall on either side, and the force jumps by 0.039 eps/sigma there.  The oracle evaluated with
    r_c (1 -+ 2e-7) brackets every such decision: particles whose oracle force differs between the two are the
    ambiguous ones (about one pair in 2e6 at density 0.05)."""
    lo = O.forces(dict(cfg, r_cut=cfg["r_cut"] * (1 - 2e-7)), cells=cells)
    hi = O.forces(dict(cfg, r_cut=cfg["r_cut"] * (1 + 2e-7)), cells=cells)
    amb = (lo["f"] != hi["f"]).any(axis=1)
    return lo, hi, amb


def check_step0(cfg, algo, ref=None, precision=64, ftol=FTOL, bracket=None):
    sim = make_sim(cfg, algo, precision)
    ref = ref if ref is not None else O.forces(cfg, cells=cfg["n_vapor"] > 20000)
    st = sim.get_state()
    en = sim.energy()
    assert sim.info()["algo"] == algo
    assert np.array_equal(st["pos"], cfg["pos"]) or precision == 32
    k_ref = O.kinetic(cfg, cfg["vel"])
    scale = max(abs(ref["U"]), k_ref)
    if bracket is None:
        assert en["pairs_vv"] == ref["pairs_vv"] and en["pairs_vw"] == ref["pairs_vw"]
        assert force_error(st["f"], ref["f"]) <= ftol
        assert scalar_error(st["pe"], ref["pe"]) <= ftol
    else:
        # fp32 mode: counts inside the bracket; unambiguous particles against the oracle, ambiguous ones against
        # whichever side of the bracket the kernel's fp32 decision took
        lo, hi, amb = bracket
        assert lo["pairs_vv"] <= en["pairs_vv"] <= hi["pairs_vv"] and lo["pairs_vw"] <= en["pairs_vw"] <= hi["pairs_vw"]
        ok = ~amb
        assert force_error(st["f"][ok], ref["f"][ok]) <= ftol
        assert scalar_error(st["pe"][ok], ref["pe"][ok]) <= ftol
        for i in np.nonzero(amb)[0]:
            assert min(force_error(st["f"][i:i + 1], side["f"][i:i + 1]) for side in (lo, hi)) <= 10 * ftol
    assert abs(en["K"] - k_ref) <= 1e-12 * k_ref or precision == 32
    assert abs(en["U"] - ref["U"]) <= ftol * scale
    assert abs(en["U_vw"] - ref["U_vw"]) <= ftol * scale
    vir_amb = 0.0 if bracket is None else 0.1 * 2.5 * max(1, int(bracket[2].sum()))   # g r^2 = 0.039 * 2.5 per flipped pair
    assert abs(en["virial"] - ref["vir"].sum()) <= ftol * max(abs(ref["vir"].sum()), k_ref) + vir_amb
    sim.close()
    return ref


def check_traj(cfg, algo, n_steps=100, cells_oracle=False, chunks=(37, 63), ref=None):
    sim = make_sim(cfg, algo)
    ref = ref if ref is not None else O.run(cfg, n_steps, cells=cells_oracle)
    assert sum(chunks) == n_steps
    for c in chunks:                      # odd + odd chunk sizes exercise both graph parities
        sim.step(c)
    st = sim.get_state()
    en = sim.energy()
    assert st["step"] == n_steps and en["step"] == n_steps
    assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= TRAJ_TOL
    assert np.abs(st["vel"] - ref["vel"]).max() <= 1e-7
    assert force_error(st["f"], ref["f"]) <= 1e-5         # forces amplify the 1e-8 position tolerance
    scale = max(abs(ref["U"]), ref["K"])
    assert abs(en["K"] - ref["K"]) <= 1e-8 * scale and abs(en["U"] - ref["U"]) <= 1e-8 * scale
    sim.close()


ALGOS = ["allpairs", "cells", "verlet"]


@pytest.mark.parametrize("algo", ALGOS)
def test_config0_forces_and_trajectory(algo):
    cfg = I.config0()
    check_step0(cfg, algo)
    check_traj(cfg, algo, 100)
    check_traj(cfg, algo, 200, chunks=(200,))


@pytest.mark.parametrize("dim,box,bc,nw,seed", [
    (3, (8.0, 9.3, 7.6), (0, 0, 0), 40, 1), (3, (8.1, 7.5, 5.2), (0, 0, 1), 40, 2), (3, (4.0, 8.0, 8.0), (1, 0, 0), 0, 3),
    (2, (13.7, 9.9), (0, 1), 12, 4), (2, (7.5, 7.5), (0, 0), 12, 5), (2, (2.6, 30.0), (1, 0), 5, 6),
    (3, (3.0, 3.0, 3.0), (1, 1, 1), 2, 7), (3, (9.6, 10.5, 9.9), (0, 0, 0), 30, 8), (3, (9.5, 9.6, 5.2), (0, 0, 1), 30, 9),
    (2, (12.0, 9.6), (0, 0), 10, 10),
    # a periodic length in [2 r_c, 2.2 r_c): more than one image per dimension can sit within r_c + margin of a face,
    # so all-pairs runs the per-pair minimum-image kernel k_force_allpairs (cells / verlet: box too small, skipped)
    (3, (5.2, 9.0, 8.0), (0, 0, 0), 20, 13), (2, (5.3, 12.0), (0, 0), 8, 14), (3, (5.05, 5.4, 5.49), (0, 0, 0), 6, 15)])
@pytest.mark.parametrize("algo", ALGOS)
def test_small_ragged_cases(dim, box, bc, nw, seed, algo):
    vol = float(np.prod(box))
    nv = min(300, int((0.5 if dim == 3 else 0.45) * vol) - nw)
    cfg = I.small_case(dim, nv, box, bc, n_wall=nw, seed=seed, min_sep=0.9)
    cfg["pos"][0, 0] = 0.0
    if bc[0] == 1:
        cfg["pos"][1, 0] = box[0]
    check_step0(cfg, algo)
    cfg = I.small_case(dim, nv, box, bc, n_wall=nw, seed=seed, min_sep=0.9)
    check_traj(cfg, algo, 100)


@pytest.mark.parametrize("heavy_list", [1, 6, 41, 1000])
def test_verlet_heavy_lane_groups(heavy_list):
    """The persistent kernel gives particles whose list has md_opts.heavy_list entries or more (default 13) to 4-lane
    groups: every split between the two code paths -- all heavy, mixed, none -- must give the oracle's forces and
    100-step trajectory."""
    for dim, box, bc, nw, seed in [(3, (9.6, 10.5, 9.9), (0, 0, 1), 30, 11), (2, (13.7, 9.9), (0, 1), 12, 12)]:
        nv = min(300, int(0.3 * float(np.prod(box))) - nw)
        cfg = dict(I.small_case(dim, nv, box, bc, n_wall=nw, seed=seed, min_sep=0.9), heavy_list=heavy_list)
        check_step0(cfg, "verlet")
        check_traj(cfg, "verlet", 100)
    cfg = dict(I.config4(12), heavy_list=heavy_list)
    check_step0(cfg, "verlet")
    check_traj(cfg, "verlet", 100, cells_oracle=True, chunks=(1, 99))


def test_verlet_condensed_state_whole_warp_lists_on_every_block():
    """config 2 with 1,000 particles condensed into a droplet (inputs.config2_condensed): ~730 lists of 50-80 entries, more
    than the warps of the idle blocks (264-320 at this size), so the persistent kernel hands the rest to the warps of the
    particle blocks after their own particles; ~300 more go to 4-lane groups.  Step 0 and a 60-step trajectory (several
    prunes and a full rebuild in the droplet) against the oracle, then the profile path over another list event."""
    cfg = I.config2_condensed()
    assert cfg["n_droplet"] == 1000
    check_step0(cfg, "verlet")
    check_traj(cfg, "verlet", 60, cells_oracle=True, chunks=(1, 22, 37))
    sim = make_sim(cfg, "verlet")
    k = sim.profile_step(60)
    assert k["rebuilds"] + k["prunes"] >= 2
    ref = O.run(cfg, 60, cells=True)
    st = sim.get_state()
    assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= TRAJ_TOL
    sim.close()
    # the same lists in fp32 mode (the whole-warp walk folds per pair there), against the oracle on the float-rounded input
    c32 = _float_rounded(cfg)
    check_step0(c32, "verlet", ref=O.forces(c32, cells=True), precision=32, ftol=1e-4, bracket=_cutoff_bracket(c32, cells=True))


def test_verlet_condensed_state_three_blocks_per_sm_variant():
    """The same droplet in a 100,000-particle box: the 80-register build of the persistent kernel (several particles per
    thread, no idle blocks), where every whole-warp list is taken by a particle-block warp after its own particles and the
    lists of 13-48 entries stay with their own threads.  Step 0 and a 60-step trajectory against the oracle."""
    cfg = I.condense(I.cylinder_config(100000, 4321, "cyl3d_100k"))
    assert cfg["n_droplet"] == 1000 and cfg["n_vapor"] == 100000
    check_step0(cfg, "verlet")
    check_traj(cfg, "verlet", 60, cells_oracle=True, chunks=(1, 22, 37))


def test_allpairs_filter_in_a_huge_sparse_box():
    """The all-pairs filter compares t = |r_i|^2 - r^2 with |r_i|^2 - (r_c^2 + rounding bound) through the bits of positive
    numbers; the bound grows with the box (fp32: 1e-6 |r|^2), so in a box thousands of sigma wide the origin has to move out
    further than r_c + 1 or the threshold of a particle near x = 0 at the y, z centre turns negative.  Three dense clusters in a
    3000 sigma periodic box -- at that spot, in the far corner and in the middle -- against the oracle, fp64 and fp32."""
    L = 3000.0
    base = I.small_case(3, 240, (9.0, 9.0, 9.0), (1, 1, 1), n_wall=12, seed=31, min_sep=0.9)
    spots = np.array([[0.3, 0.5 * L - 4.0, 0.5 * L - 4.0], [L - 9.5, 0.4, 0.6], [0.5 * L, 0.5 * L, 0.5 * L]])
    pos = np.concatenate([base["pos"][k::3] + spots[k] for k in range(3)])
    vel = np.concatenate([base["vel"][k::3] for k in range(3)])
    cfg = dict(base, pos=np.ascontiguousarray(pos), vel=np.ascontiguousarray(vel), wall=base["wall"] + spots[0], box_len=[L, L, L], bc=[0, 0, 0])
    ref = O.forces(cfg)
    assert ref["pairs_vv"] > 400 and ref["pairs_vw"] > 20
    check_step0(cfg, "allpairs", ref=ref)
    c32 = _float_rounded(cfg)
    check_step0(c32, "allpairs", ref=O.forces(c32), precision=32, ftol=1e-4, bracket=_cutoff_bracket(c32, cells=False))


def test_single_particle_and_no_walls():
    cfg = I.small_case(3, 1, (10.0, 10.0, 10.0), (0, 1, 0), seed=3)
    for algo in ALGOS:
        sim = md.Simulation(cfg, algo=algo)
        sim.step(10)
        st = sim.get_state()
        assert (st["f"] == 0).all() and (st["pe"] == 0).all()
        ref = O.run(cfg, 10)
        assert np.abs(st["pos"] - ref["pos"]).max() < 1e-13
        assert sim.energy()["pairs_vv"] == 0
        sim.close()


def test_two_particle_closed_form_on_gpu():
    cfg = I.small_case(3, 2, (20.0, 20.0, 20.0), (0, 0, 0), seed=3)
    cfg["pos"] = np.array([[1.5, 7.0, 7.0], [0.0, 7.0, 7.0]])
    cfg["shift_energy"] = 0
    for algo in ALGOS:
        sim = md.Simulation(cfg, algo=algo)
        st, en = sim.get_state(), sim.energy()
        assert abs(en["U"] + 0.3203365942785745) < 1e-14
        assert abs(st["f"][0, 0] + 1.158028831046155) < 1e-13 and st["f"][1, 0] == -st["f"][0, 0]
        sim.close()


def test_reflecting_escape_is_reported():
    cfg = I.small_case(3, 4, (9.0, 9.0, 9.0), (1, 1, 1), seed=3)
    cfg["vel"][0, 0] = 9.0 * 3 / cfg["dt"]           # crosses the box three times in one step
    for algo in ALGOS:
        sim = md.Simulation(cfg, algo=algo)
        sim.step(1)
        with pytest.raises(md.MDError) as e:
            sim.get_state()
        assert e.value.code == md.MD_ERR_STATE


def test_config1_step0_and_100_steps():
    cfg = I.config1()
    ref = O.forces(cfg)                                   # brute-force oracle, 3.4e8 tests
    for algo in ("cells", "verlet"):
        check_step0(cfg, algo, ref=ref)
        check_traj(cfg, algo, 100, cells_oracle=True)


def test_config2_step0_brute_sample_and_cells():
    cfg = I.config2()
    ref = check_step0(cfg, "cells", ref=O.forces(cfg, cells=True))
    # brute-force definition on a sample of particles: oracle cells == oracle brute there (ties the big case to c.2)
    sub = dict(cfg)
    idx = np.arange(0, cfg["n_vapor"], 97)
    # forces on sampled particles from ALL others: evaluate brute force on the full set is 4.4e9 tests (~1 min);
    # instead compare energies/forces of the cell oracle with the GPU all-pairs kernel, an independent traversal
    sim = md.Simulation(cfg, algo="allpairs")
    st = sim.get_state(pos=False, vel=False, pe=False)
    assert force_error(st["f"][idx], ref["f"][idx]) <= FTOL
    assert sim.energy()["pairs_vv"] == ref["pairs_vv"]
    sim.close()
    check_step0(cfg, "verlet", ref=ref)
    check_traj(cfg, "cells", 100, cells_oracle=True)
    check_traj(cfg, "verlet", 100, cells_oracle=True)


def test_config2_bench_launch_configuration_2000_steps():
    """Full size, the launch bench.py times (MD_FORCE_VERLET, md_step(2000) = one persistent launch, then md_energy).
    Beyond 100 steps trajectories are no longer comparable point by point (north_star), so what holds at any size is
    checked: the step counter, energy conservation (|E(2000) - E(0)| <= 1e-4 K(0); measured 3.1e-5 -- a dropped or
    doubled pair term drifts far more) and the oracle's K, U and pair counts at the same step (measured agreement 5e-5,
    1e-4, < 1e-4 and 3e-4; bounds 2e-3, 2e-3, 5e-3 and 2e-2)."""
    cfg = I.config2()
    sim = md.Simulation(cfg, algo="verlet")
    e0 = sim.energy()
    sim.step(2000)
    e1 = sim.energy()
    assert e1["step"] == 2000
    assert abs((e1["K"] + e1["U"]) - (e0["K"] + e0["U"])) <= 1e-4 * e0["K"]
    ref = O.run(cfg, 2000, cells=True)
    assert abs(e1["K"] - ref["K"]) <= 2e-3 * ref["K"]
    assert abs(e1["U"] - ref["U"]) <= 2e-3 * abs(ref["U"])
    f = O.forces(dict(cfg, pos=ref["pos"]), cells=True)
    assert abs(e1["pairs_vv"] - f["pairs_vv"]) <= 5e-3 * f["pairs_vv"]
    assert abs(e1["pairs_vw"] - f["pairs_vw"]) <= 2e-2 * f["pairs_vw"] + 20
    sim.close()


@pytest.mark.parametrize("n_vapor", [100000, 262144])
def test_verlet_three_blocks_per_sm_variant_trajectory(n_vapor):
    """Beyond 2 x SMs x 256 particles md_step runs the 80-register, 3-blocks-per-SM build of the persistent kernel:
    with one thread per particle and idle blocks for the lane groups (100,000) and with several particles per
    thread (262,144).  Step 0 and the 100-step trajectory against the oracle's cell-list variant."""
    cfg = I.cylinder_config(n_vapor, 20261, "three_blocks_%d" % n_vapor)
    check_step0(cfg, "verlet", ref=O.forces(cfg, cells=True))
    check_traj(cfg, "verlet", 100, cells_oracle=True, chunks=(41, 59))


@pytest.mark.parametrize("shape", ["cone", "inkbottle", "slit"])
def test_config3_shapes_step0_and_100_steps(shape):
    # BASELINE.json configs[3]: 262,144 vapor particles, three pore shapes; oracle = its CPU cell-list variant
    cfg = I.config3(shape)
    ref = O.forces(cfg, cells=True)
    check_step0(cfg, "cells", ref=ref)
    check_step0(cfg, "verlet", ref=ref)
    traj = O.run(cfg, 100, cells=True)
    check_traj(cfg, "cells", 100, ref=traj)
    check_traj(cfg, "verlet", 100, ref=traj)


@pytest.mark.parametrize("log2n", [10, 12, 14])
def test_config4_sizes_both_kernels(log2n):
    cfg = I.config4(log2n)
    ref = O.forces(cfg)
    check_step0(cfg, "cells", ref=ref)
    check_step0(cfg, "allpairs", ref=ref)
    check_step0(cfg, "verlet", ref=ref)
    check_traj(cfg, "cells", 100, cells_oracle=True)
    check_traj(cfg, "verlet", 100, cells_oracle=True)


@pytest.mark.parametrize("log2n", [16, 18, 20])
def test_config4_large_sizes_all_paths(log2n):
    # BASELINE.json configs[4] with its own seeds: step 0 on all three paths (all-pairs at 2^20: 1.1e12 tests per
    # evaluation), 100-step trajectories on the two cell-based paths (and all-pairs at 2^16: 4.4e9 tests per step)
    cfg = I.config4(log2n)
    ref = O.forces(cfg, cells=True)
    for algo in ALGOS:
        check_step0(cfg, algo, ref=ref)
    traj = O.run(cfg, 100, cells=True)
    check_traj(cfg, "cells", 100, ref=traj)
    check_traj(cfg, "verlet", 100, ref=traj, chunks=(1, 42, 57))
    if log2n == 16:
        check_traj(cfg, "allpairs", 100, ref=traj)


def _float_rounded(cfg, keys=("pos", "wall")):
    c32 = dict(cfg)
    for k in keys:
        c32[k] = cfg[k].astype(np.float32).astype(np.float64)
    c32["box_len"] = [float(np.float32(x)) for x in cfg["box_len"]]
    return c32


@pytest.mark.parametrize("log2n", [12, 16, 20])
def test_fp32_mode_forces(log2n):
    # reading A12: fp32 state/arithmetic; compared with the oracle fed the same float-rounded inputs.  BASELINE.json
    # configs[4] runs every size in fp32 too: in the 276 sigma box of 2^20 one ulp of a coordinate is 3e-5 sigma, so the
    # <= 1e-4 bound only holds because differences are formed exactly (image shift on the particle at the top of the box)
    cfg = I.config4(log2n)
    c32 = _float_rounded(cfg)
    ref = O.forces(c32, cells=log2n > 14)
    bracket = _cutoff_bracket(c32, cells=log2n > 14)
    for algo in ("cells", "allpairs", "verlet"):
        check_step0(c32, algo, ref=ref, precision=32, ftol=1e-4, bracket=bracket)


@pytest.mark.parametrize("algo", ["cells", "verlet"])
def test_energy_drift_and_long_run_statistics_dilute_gas(algo):
    # long runs are chaotic: compare the drift statistic (reading A8: wall-free dilute 3D gas, shifted energy,
    # |<E>_{9000..10000} - <E>_{1000..2000}| / K(0)) and the temperature with the oracle's, not trajectories
    # The statistic is a random walk of r_c-crossing kinks whose relative size falls as 1/sqrt(N), and the GPU's
    # summation order (atomics) makes every run another realisation of it: measured over 12 runs 2e-6 .. 7e-5 at
    # N = 16384 (a tail beyond the 1e-4 bound) and 2e-7 .. 2e-5 at N = 65536, so the check runs at 65536
    cfg = I.cylinder_config(65536, 4242, "drift", box=(65536 / 0.05) ** (1 / 3), length=0)
    sim = md.Simulation(cfg, algo=algo)
    e0 = sim.energy()

    def window():
        out = []
        for _ in range(100):
            sim.step(10)
            e = sim.energy()
            out.append((e["K"], e["U"]))
        return np.array(out)

    sim.step(1000)
    wa = window()
    sim.step(7000)
    wb = window()
    assert sim.energy()["step"] == 10000
    drift = abs(wb.sum(axis=1).mean() - wa.sum(axis=1).mean()) / e0["K"]
    assert drift <= 1e-4, drift
    ref = O.run(cfg, 1500, cells=True, history=True)["hist"]
    t_ref = ref[1000:1500, 0].mean()
    assert abs(wa[:50, 0].mean() - t_ref) / t_ref < 0.02
    sim.close()


def _profiles(pos, cfg, r_max=10.0, n_r=10, n_z=11):
    """Radial (about the pore axis, inside the pore's z range) and axial vapor density profiles (host side)."""
    L = np.array(cfg["box_len"])
    c = 0.5 * L
    half = 0.5 * cfg["pore_length"]
    d = pos - c
    rho = np.hypot(d[:, 0], d[:, 1])
    inside = np.abs(d[:, 2]) <= half
    hr, edges = np.histogram(rho[inside], bins=n_r, range=(0.0, r_max))
    shell = np.pi * (edges[1:] ** 2 - edges[:-1] ** 2) * 2 * half
    hz, _ = np.histogram(pos[:, 2], bins=n_z, range=(0.0, L[2]))
    return hr / shell, hz / (L[0] * L[1] * L[2] / n_z)


@pytest.mark.parametrize("algo", ["cells", "verlet"])
def test_long_run_density_profiles_match_oracle_statistically(algo):
    # beyond 100 steps trajectories are chaotic: north_star compares the radial / axial density profile instead.
    # Same input, 3000 steps, profiles averaged over the last 1000 steps (every 50th); the two runs are different
    # realisations of the same ensemble, so bins must agree within counting noise (5 sigma + 5 %).
    cfg = I.config4(12)
    sim = md.Simulation(cfg, algo=algo)
    pos, vel = cfg["pos"], cfg["vel"]
    acc_g, acc_o, n_samples = None, None, 0
    sim.step(2000)
    o = O.run(cfg, 2000, cells=True)
    pos, vel = o["pos"], o["vel"]
    for _ in range(20):
        sim.step(50)
        o = O.run(cfg, 50, pos=pos, vel=vel, cells=True)
        pos, vel = o["pos"], o["vel"]
        pg = _profiles(sim.get_state(vel=False, force=False, pe=False)["pos"], cfg)
        po = _profiles(pos, cfg)
        acc_g = pg if acc_g is None else tuple(a + b for a, b in zip(acc_g, pg))
        acc_o = po if acc_o is None else tuple(a + b for a, b in zip(acc_o, po))
        n_samples += 1
    L = np.array(cfg["box_len"])
    half = 0.5 * cfg["pore_length"]
    vol_r = np.pi * (np.linspace(0, 10, 11)[1:] ** 2 - np.linspace(0, 10, 11)[:-1] ** 2) * 2 * half
    vol_z = np.full(11, L.prod() / 11)
    for g, o_, vol in ((acc_g[0], acc_o[0], vol_r), (acc_g[1], acc_o[1], vol_z)):
        g, o_ = g / n_samples, o_ / n_samples
        counts = np.maximum(o_ * vol, 1.0)                         # mean particles per bin per sample
        sigma = np.sqrt(counts) / vol                              # >= counting noise of one sample (correlated samples)
        assert (np.abs(g - o_) <= 5 * sigma + 0.05 * np.maximum(o_, g)).all(), (g, o_)
    sim.close()


def test_boundary_helpers_and_error_paths():
    cfg = I.config4(10)
    ref = O.forces(cfg)
    # pair-test counters: all-pairs is analytic (+ ghosts), cell walk >= list entries >= ordered hits
    hits = 2 * ref["pairs_vv"] + ref["pairs_vw"]
    counts = {}
    for algo in ALGOS:
        sim = md.Simulation(cfg, algo=algo)
        counts[algo] = sim.pair_tests()
        sim.step(0)                                            # no-op
        assert sim.get_state()["step"] == 0
        k = sim.profile_step(7)
        assert k["steps"] == 7 and k["total_ms"] > 0 and sim.energy()["step"] == 7
        sim.close()
    nv, nw = cfg["n_vapor"], cfg["n_wall"]
    assert counts["allpairs"] >= nv * (nv - 1 + nw) and counts["cells"] >= counts["verlet"] >= hits
    # profile_step and step advance the same dynamics
    a, b = md.Simulation(cfg, algo="verlet"), md.Simulation(cfg, algo="verlet")
    a.step(23)
    b.profile_step(23)
    assert np.abs(a.get_state()["pos"] - b.get_state()["pos"]).max() < 1e-12
    a.close(), b.close()
    # workspace too small
    import ctypes as C
    box, lj, opts = md._structs(cfg, 64, "verlet")
    ws = torch.empty(4096, dtype=torch.uint8, device="cuda")
    h = C.c_void_p()
    pos, vel, wall = (np.ascontiguousarray(cfg[k]) for k in ("pos", "vel", "wall"))
    rc = md.load_library().md_create(C.byref(h), C.byref(box), None, C.byref(lj), C.byref(opts), nv, md._dptr(pos),
                                     md._dptr(vel), nw, md._dptr(wall), ws.data_ptr(), ws.numel(), None)
    assert rc == md.MD_ERR_WORKSPACE and not h.value
    peaks = md.measure_peaks(scratch_mib=128)
    assert 10 < peaks["fp64_tflops"] < 60 and peaks["fp32_tflops"] > peaks["fp64_tflops"] and peaks["copy_gbs"] > 1000


def test_verlet_list_overflow_is_reported_not_dropped():
    # 160 particles inside a sphere of radius 1.2: every particle has > 128 neighbours within r_c + skin
    rng = I.SplitMix64(5)
    pts = []
    while len(pts) < 160:
        p = (rng.uniform(3) * 2 - 1) * 1.2
        if p @ p < 1.44:
            pts.append(p + 10.0)
    cfg = I.small_case(3, 160, (20.0, 20.0, 20.0), (0, 0, 0), seed=3, min_sep=0.5)
    cfg["pos"] = np.array(pts)
    cfg["eps"] = 0.0                                           # overlapping sites: keep the forces finite
    with pytest.raises(md.MDError) as e:
        md.Simulation(cfg, algo="verlet")
    assert e.value.code == md.MD_ERR_WORKSPACE
    sim = md.Simulation(cfg, algo="cells")                     # the per-step cell walk has no such limit
    assert sim.energy()["pairs_vv"] == 160 * 159 // 2
    sim.close()


@pytest.mark.parametrize("algo", ALGOS)
def test_fp32_trajectory_stays_close(algo):
    # fp32 mode over 100 steps against the fp64 oracle on the float-rounded input: rounding of the state
    # (ulp(L) ~ 4e-6 per step in position) bounds the agreement, not the force law
    cfg = I.config4(12)
    c32 = _float_rounded(cfg, ("pos", "wall", "vel"))
    ref = O.run(c32, 100, cells=True)
    sim = make_sim(c32, algo, precision=32)
    sim.step(100)
    st, en = sim.get_state(), sim.energy()
    assert traj_error(st["pos"], ref["pos"], c32["box_len"], c32["bc"]) < 2e-3
    assert abs(en["K"] - ref["K"]) < 1e-4 * ref["K"] and abs(en["U"] - ref["U"]) < 2e-3 * max(abs(ref["U"]), 1.0)
    sim.close()


@pytest.mark.parametrize("algo", ALGOS)
def test_berendsen_thermostat_matches_oracle(algo):
    # NEXT-1: the paper's kernel F4 after every step; same tolerances as the NVE trajectories
    cfg = dict(I.config4(12), tau_b=0.1, t_target=0.6)
    ref = O.run(cfg, 100, cells=True, history=True)
    sim = make_sim(cfg, algo)
    for chunk in (1, 36, 63):
        sim.step(chunk)
    st, en = sim.get_state(), sim.energy()
    assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= TRAJ_TOL
    assert np.abs(st["vel"] - ref["vel"]).max() <= 1e-7
    assert abs(en["K"] - ref["K"]) <= 1e-9 * ref["K"]
    t0 = 2 * ref["hist"][0, 0] / (3 * cfg["n_vapor"])
    t100 = 2 * en["K"] / (3 * cfg["n_vapor"])
    assert t0 > 0.95 and abs(t100 - 0.6) < 0.05                 # 5 rise times later the gas sits at T_0
    sim.close()
    # small 2D case, other parities of the step count
    c2 = dict(I.small_case(2, 40, (13.7, 9.9), (0, 1), n_wall=12, seed=4, min_sep=0.9), tau_b=0.02, t_target=1.5)
    r2 = O.run(c2, 33)
    s2 = make_sim(c2, algo)
    s2.step(33)
    assert traj_error(s2.get_state()["pos"], r2["pos"], c2["box_len"], c2["bc"]) <= TRAJ_TOL
    s2.close()


def _oracle_pressure(cfg, out):
    """(P_box, P_pore, n_pore) from the oracle's positions, velocities and per-particle virial."""
    dim = cfg["dim"]
    L = np.array(cfg["box_len"][:dim])
    k = 0.5 * cfg["mass"] * (out["vel"] ** 2).sum(axis=1)
    w = out["vir"]
    p_box = (2 * k.sum() + w.sum()) / (dim * L.prod())
    pd = cfg["pore"]
    d = out["pos"] - np.array(pd["center"][:dim])
    if pd["kind"] == "cylinder":
        ax = pd["axis"]
        a1, a2 = (ax + 1) % 3, (ax + 2) % 3
        inside = (np.abs(d[:, ax]) < 0.5 * pd["length"]) & (d[:, a1] ** 2 + d[:, a2] ** 2 < pd["r0"] ** 2)
        vol = np.pi * pd["r0"] ** 2 * pd["length"]
    else:
        ax = pd["axis"]
        inside = (np.abs(d[:, ax]) < 0.5 * pd["width"]) & (np.abs(d[:, 1 - ax]) < 0.5 * pd["length"])
        vol = pd["width"] * pd["length"]
    return p_box, (2 * k[inside].sum() + w[inside].sum()) / (dim * vol), int(inside.sum())


@pytest.mark.parametrize("algo", ALGOS)
def test_virial_pressure_box_and_pore(algo):
    # NEXT-2: P = (2K + W) / (d V) over the box and over the particles inside the pore volume
    for cfg, n in ((I.config4(12), 60), (I.config1(n_vapor=4096), 40)):
        ref = O.run(cfg, n, cells=True)
        p_box, p_pore, n_pore = _oracle_pressure(cfg, ref)
        sim = make_sim(cfg, algo)
        sim.step(n)
        pr = sim.pressure()
        assert pr["n_pore"] == n_pore and pr["step"] == n
        assert abs(pr["P_box"] - p_box) <= 1e-8 * abs(p_box)
        assert abs(pr["P_pore"] - p_pore) <= 1e-8 * max(abs(p_pore), abs(p_box))
        sim.close()
    # ideal gas limit: no forces -> P V = N T exactly (T = 2K / (d N))
    cfg = dict(I.config4(10), eps=0.0, eps_w=0.0)
    sim = make_sim(cfg, algo)
    pr, en = sim.pressure(), sim.energy()
    assert abs(pr["P_box"] * pr["V_box"] - 2 * en["K"] / 3) < 1e-9 * en["K"]
    sim.close()
    nopore = I.small_case(3, 50, (10.0, 10.0, 10.0), (0, 0, 1), seed=3)
    sim = make_sim(nopore, algo)
    with pytest.raises(md.MDError) as e:
        sim.pressure()
    assert e.value.code == md.MD_ERR_UNSUPPORTED
    sim.close()


@pytest.mark.parametrize("algo", ALGOS)
def test_device_density_profile_is_bit_exact(algo):
    # NEXT-4: integer work -> bit-exact against the same histogram taken on the host from md_get_state
    for cfg, n_ax, n_r, r_max in ((I.config4(12), 11, 10, 10.0), (I.config1(n_vapor=4096), 16, 8, 12.0)):
        sim = make_sim(cfg, algo)
        sim.step(37)
        pos = sim.get_state(vel=False, force=False, pe=False)["pos"]
        ax, ra = sim.density_profile(n_ax, n_r, r_max)
        pd, dim = cfg["pore"], cfg["dim"]
        L = np.array(cfg["box_len"][:dim])
        d = pos - np.array(pd["center"][:dim])
        if pd["kind"] == "cylinder":
            along, a1, a2 = pd["axis"], (pd["axis"] + 1) % 3, (pd["axis"] + 2) % 3
            rho = np.sqrt(d[:, a1] ** 2 + d[:, a2] ** 2)
        else:
            along = 1 - pd["axis"]
            rho = np.abs(d[:, pd["axis"]])
        inside = np.abs(d[:, along]) < 0.5 * pd["length"]
        ax_ref = np.bincount(np.clip(np.floor(pos[:, along] / L[along] * n_ax).astype(int), 0, n_ax - 1), minlength=n_ax)
        b = np.floor(rho / r_max * n_r).astype(int)
        ra_ref = np.bincount(b[inside & (b < n_r)], minlength=n_r)
        assert ax.sum() == cfg["n_vapor"] and np.array_equal(ax, ax_ref) and np.array_equal(ra, ra_ref)
        sim.close()


@pytest.mark.parametrize("algo", ALGOS)
def test_geometric_prism_pore_matches_oracle(algo):
    # NEXT-3: the paper's own pore geometry (closed faces reflect, +axis face open), gas inside and outside
    for dim, box, axis in ((3, (16.0, 15.0, 14.0), 2), (2, (24.0, 20.0), 0)):
        nv = 220 if dim == 3 else 90
        cfg = I.small_case(dim, nv, box, (0,) * dim, n_wall=0, seed=12 + dim, min_sep=1.0, t_star=2.0)
        cfg["pore"] = dict(kind="prism", axis=axis, center=[0.5 * b for b in box], length=7.0, width=5.0)
        cfg["dt"] = 0.01
        ref = O.run(cfg, 150, cells=False)
        assert not np.allclose(ref["pos"], O.run(dict(cfg, pore=None), 150)["pos"])      # the walls did act
        sim = make_sim(cfg, algo)
        sim.step(75)
        sim.step(75)
        st = sim.get_state()
        assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= TRAJ_TOL
        assert np.abs(st["vel"] - ref["vel"]).max() <= 1e-7
        sim.close()
    bad = dict(cfg)
    bad["pore"] = dict(kind="prism", axis=0, center=[2.0, 10.0], length=7.0, width=5.0)     # sticks out of the box
    with pytest.raises(md.MDError) as e:
        md.Simulation(bad, algo=algo)
    assert e.value.code == md.MD_ERR_INVALID_ARG


@pytest.mark.parametrize("n_pore", [None, 100, 1500])
@pytest.mark.parametrize("dim", [2, 3])
def test_paper_geometry_and_units_match_oracle(dim, n_pore):
    # NEXT-3: the paper's own runs in reduced units, geometric walls, all-pairs; and the end
    # points of its N sweeps (Tables 2-3: N = 100 and 1500 molecules in the pore)
    cfg = I.paper_geometry(dim, n_pore=n_pore)
    n_tot = {None: 2184 if dim == 2 else 2800, 100: 520 if dim == 2 else 280, 1500: 7800 if dim == 2 else 4200}[n_pore]
    assert cfg["n_vapor"] == n_tot and abs(cfg["dt"] - 0.00959) < 1e-5
    # 200 steps; 2000 for the 100-molecule pore, where 200 steps (3.8 sigma of flight in a 3155 sigma pore) see no bounce
    n_steps = 2000 if n_pore == 100 else 200
    ref = O.run(cfg, n_steps)
    assert not np.array_equal(np.sign(ref["vel"]), np.sign(cfg["vel"]))          # some molecules did bounce
    sim = md.Simulation(cfg, algo="allpairs")
    sim.step(n_steps)
    st = sim.get_state()
    assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= TRAJ_TOL
    assert np.abs(st["vel"] - ref["vel"]).max() <= 1e-7
    sim.close()


def _nonunit(cfg, sig=1.3, eps=0.7, sig_w=1.1, eps_w=1.6, mass=2.5, r_cut=3.0):
    """cfg with its geometry scaled by sig and every model parameter away from 1 (m_i, sigma, eps are
    parameters).  r_cut and sigma_w are NOT the scaled values, so this is not the reduced-unit system in disguise."""
    c = dict(cfg, pos=cfg["pos"] * sig, wall=cfg["wall"] * sig, box_len=[x * sig for x in cfg["box_len"]],
             sigma=sig, eps=eps, sigma_w=sig_w, eps_w=eps_w, mass=mass, r_cut=r_cut)
    if cfg.get("pore"):
        pd = dict(cfg["pore"])
        pd["center"] = [x * sig for x in pd["center"]]
        for k in ("length", "r0", "width"):
            if k in pd:
                pd[k] = pd[k] * sig
        c["pore"] = pd
    return c


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("thermostat", [False, True])
def test_parameters_away_from_one(algo, thermostat):
    """mass = 2.5, sigma = 1.3, eps = 0.7, sigma_w = 1.1, eps_w = 1.6, r_cut = 3: the first time the time loop's own
    coefficients (c12 = 48 eps sigma^12, c6 = 24 eps sigma^6), hk = dt / 2m, K = m v^2 / 2 and the thermostat's
    temperature see anything but 1 (the oracle's side is pinned by tests/test_oracle_pins.py::test_scaled_* and
    ::test_dimensional_scaling_*)."""
    extra = dict(tau_b=0.08, t_target=0.7) if thermostat else {}
    for base, cells in ((I.config4(12), True), (I.small_case(2, 90, (13.7, 9.9), (0, 1), n_wall=12, seed=4, min_sep=0.9), False),
                        (I.small_case(3, 200, (9.6, 10.5, 9.9), (0, 0, 1), n_wall=30, seed=8, min_sep=0.9), False)):
        cfg = dict(_nonunit(base), **extra)
        check_step0(cfg, algo, ref=O.forces(cfg, cells=cells))
        ref = O.run(cfg, 100, cells=cells)
        sim = make_sim(cfg, algo)
        for c in (1, 36, 63):
            sim.step(c)
        st, en = sim.get_state(), sim.energy()
        assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= TRAJ_TOL
        assert np.abs(st["vel"] - ref["vel"]).max() <= 1e-7
        scale = max(abs(ref["U"]), ref["K"])
        assert abs(en["K"] - ref["K"]) <= 1e-8 * scale and abs(en["U"] - ref["U"]) <= 1e-8 * scale
        if cfg.get("pore"):                                  # K with the mass in it also feeds the pressure monitor
            pr = sim.pressure()
            p_box, p_pore, n_pore = _oracle_pressure(cfg, ref)
            assert pr["n_pore"] == n_pore and abs(pr["P_box"] - p_box) <= 1e-7 * abs(p_box)
        sim.close()


def _drift_statistic(e, k0):
    """Reading A8: (<E> over the last 1000 steps - <E> over steps 1000..2000) / K(0), signed."""
    return (e[-1000:].mean() - e[1000:2000].mean()) / k0


def test_energy_drift_distribution_matches_oracle_over_seeds():
    """Reading A8 over several realisations instead of one pass/fail: the plainly truncated force makes every r_c
    crossing a small energy kink, so the statistic is a zero-mean random walk whose rms falls as 1/sqrt(N) (oracle, 8
    seeds each: rms 1.6e-4 at N = 1728, 1.1e-4 at N = 4096; A8).  GPU (Verlet path) and oracle are run on the
    same 8 seeded inputs at N = 4096; trajectories decorrelate (chaos), so the two sets of 8 values are compared as
    samples of one distribution: rms within a factor 3 of each other and of the 6.4e-3 / sqrt(N) law, no systematic
    sign."""
    n, seeds = 4096, range(4242, 4250)
    gpu, orc = [], []
    for seed in seeds:
        cfg = I.cylinder_config(n, seed, "drift", box=(n / 0.05) ** (1 / 3), length=0)
        h = O.run(cfg, 10000, cells=True, history=True)["hist"]
        orc.append(_drift_statistic(h[:, 0] + h[:, 1] + h[:, 2], h[0, 0]))
        sim = md.Simulation(cfg, algo="verlet")
        k0 = sim.energy()["K"]
        e = np.zeros(10001)                                  # E at steps 1000..1999 and 9001..10000, as the statistic reads
        sim.step(1000)
        for s in range(1000, 2000):
            en = sim.energy()
            e[s] = en["K"] + en["U"]
            sim.step(1)
        sim.step(7001)
        for s in range(9001, 10001):
            en = sim.energy()
            e[s] = en["K"] + en["U"]
            assert en["step"] == s
            if s < 10000:
                sim.step(1)
        assert sim.energy()["step"] == 10000
        gpu.append(_drift_statistic(e, k0))
        sim.close()
    gpu, orc = np.array(gpu), np.array(orc)
    rms_g, rms_o, law = np.sqrt((gpu ** 2).mean()), np.sqrt((orc ** 2).mean()), 6.4e-3 / np.sqrt(n)
    assert law / 3 <= rms_o <= 3 * law and law / 3 <= rms_g <= 3 * law and rms_o / 3 <= rms_g <= 3 * rms_o, (gpu, orc)
    assert gpu.min() < 0 < gpu.max() and orc.min() < 0 < orc.max()               # a zero-mean random walk, not a trend


@pytest.mark.parametrize("algo", ALGOS)
def test_fp32_mode_monitors(algo):
    # md_density_profile and md_pressure in fp32 mode: the histogram is integer work on the fp32 positions the handle
    # itself reports (bit-exact); the pressure is compared with the oracle on the float-rounded input (<= 1e-4)
    cfg = _float_rounded(I.config4(12), ("pos", "wall", "vel"))
    sim = make_sim(cfg, algo, precision=32)
    pr = sim.pressure()
    ref = O.forces(cfg)
    p_box, p_pore, n_pore = _oracle_pressure(cfg, dict(ref, pos=cfg["pos"], vel=cfg["vel"]))
    assert pr["n_pore"] == n_pore
    assert abs(pr["P_box"] - p_box) <= 1e-4 * abs(p_box) and abs(pr["P_pore"] - p_pore) <= 1e-4 * max(abs(p_pore), abs(p_box))
    sim.step(37)
    pos = sim.get_state(vel=False, force=False, pe=False)["pos"]
    ax, ra = sim.density_profile(11, 10, 10.0)
    pd = cfg["pore"]
    L = np.array(cfg["box_len"])
    d = pos - np.array(pd["center"])
    rho = np.sqrt(d[:, 0] ** 2 + d[:, 1] ** 2)
    inside = np.abs(d[:, 2]) < 0.5 * pd["length"]
    ax_ref = np.bincount(np.clip(np.floor(pos[:, 2] / L[2] * 11).astype(int), 0, 10), minlength=11)
    b = np.floor(rho / 10.0 * 10).astype(int)
    ra_ref = np.bincount(b[inside & (b < 10)], minlength=10)
    assert ax.sum() == cfg["n_vapor"] and np.array_equal(ax, ax_ref) and np.array_equal(ra, ra_ref)
    sim.close()


@pytest.mark.parametrize("list_prunes", [-1, 1, 2, 4])
def test_verlet_two_level_list_prunes(list_prunes):
    """md_opts.list_prunes: between two full rebuilds the r_c + skin list is pruned from an outer list.  Every setting --
    none (single-level list), the default two, and more than the box allows (reduced automatically) -- must give the
    oracle's forces and trajectory: 300 steps span several full rebuilds and prunes (checked through md_profile_step's
    counters), in chunks so that a launch starts with prunes pending from the previous one."""
    cfg = dict(I.config4(12), list_prunes=list_prunes)
    check_step0(cfg, "verlet")
    ref = O.run(cfg, 300, cells=True)
    sim = make_sim(cfg, "verlet")
    events = [sim.profile_step(n) for n in (7, 93, 1, 199)]
    st, en = sim.get_state(), sim.energy()
    rebuilds, prunes = sum(e["rebuilds"] for e in events), sum(e["prunes"] for e in events)
    assert rebuilds >= 3
    assert (prunes == 0) if list_prunes < 0 else (prunes >= rebuilds)
    # 300 steps: the 1e-8 sigma bound of 100 steps grows with the Lyapunov time (measured 3e-9); K, U to 1e-7
    assert traj_error(st["pos"], ref["pos"], cfg["box_len"], cfg["bc"]) <= 1e-6
    scale = max(abs(ref["U"]), ref["K"])
    assert abs(en["K"] - ref["K"]) <= 1e-7 * scale and abs(en["U"] - ref["U"]) <= 1e-7 * scale
    sim.close()
    # a box too small for any outer list (the setting is reduced to none), a dense 2D fluid, the thermostat's split phases
    for small, extra in ((I.small_case(3, 200, (9.6, 10.5, 9.9), (0, 0, 1), n_wall=30, seed=8, min_sep=0.9), {}),
                         (I.config0(), {}), (I.config4(10), dict(tau_b=0.1, t_target=0.7))):
        c = dict(small, list_prunes=list_prunes, **extra)
        check_traj(c, "verlet", 100, cells_oracle=c["n_vapor"] > 500)
