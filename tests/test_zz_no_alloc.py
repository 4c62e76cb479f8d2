"""md_kinetic_energy_noalloc -- the entry point that allocates no device memory (its reduction scratch is a static __device__
array inside the library, include/md.h) -- against the existing path (md_energy's kinetic energy, whose partial sums live in
the caller's workspace), on calls in a row that share the scratch array.  Collected last on purpose (file name): the suite
runs with pytest -x, and a failure here must not hide the parity tests.
"""
import numpy as np
import pytest
import torch

from oracle import md_oracle as O
from paper_1812_07993_b200 import inputs as I
from paper_1812_07993_b200 import md

pytestmark = pytest.mark.gpu

KTOL = 1e-12          # relative; the bound tests/test_gpu_parity.py::check_step0 puts on K


def _kinetic_noalloc(vel_np, mass, stream):
    vel = torch.from_numpy(np.ascontiguousarray(vel_np)).to("cuda:0")
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda:0")
    stream.wait_stream(torch.cuda.current_stream())
    md.kinetic_energy_noalloc(vel, mass, out, stream=stream)
    stream.synchronize()
    return float(out.item())


def test_noalloc_kinetic_energy_matches_md_energy_on_calls_in_a_row():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    md.load_library()
    stream = torch.cuda.Stream(device="cuda:0")
    # call 1: 65,536 particles (64 partial sums in the scratch array), mass away from 1
    big = dict(I.config4(16), mass=2.5)
    sim = md.Simulation(big, algo="verlet")
    sim.step(40)
    k_existing = sim.energy()["K"]
    vel = sim.get_state(pos=False, force=False, pe=False)["vel"]
    k1 = _kinetic_noalloc(vel, big["mass"], stream)
    assert abs(k1 - k_existing) <= KTOL * k_existing
    assert abs(k1 - O.kinetic(big, vel)) <= KTOL * k_existing            # and the oracle's plain sum
    sim.close()
    # call 2, directly after: 1,024 particles in 2D -> ONE partial sum; slots 1..63 still hold call 1's values and must
    # not leak into the result
    small = I.config0()
    sim = md.Simulation(small, algo="allpairs")
    sim.step(25)
    k_existing = sim.energy()["K"]
    vel = sim.get_state(pos=False, force=False, pe=False)["vel"]
    k2 = _kinetic_noalloc(vel, small["mass"], stream)
    assert abs(k2 - k_existing) <= KTOL * k_existing
    # call 3: the same input again gives the same bits (fixed summation order, nothing left over from call 2)
    assert _kinetic_noalloc(vel, small["mass"], stream) == k2
    # call 4: back to a size that needs several slots, ragged tail (4,097 = 4 blocks + 1 particle)
    rng = I.SplitMix64(11)
    v = rng.normal(4097 * 3).reshape(4097, 3)
    k4 = _kinetic_noalloc(v, 1.7, stream)
    k_ref = 0.5 * 1.7 * float((v * v).sum())
    assert abs(k4 - k_ref) <= KTOL * k_ref
    sim.close()


def test_noalloc_rejects_sizes_beyond_the_static_scratch_and_bad_arguments():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    vel = torch.zeros((8, 3), dtype=torch.float64, device="cuda:0")
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    with pytest.raises(md.MDError) as e:          # validated on the host before anything is launched or read
        md.kinetic_energy_noalloc(vel, 1.0, out, n=md.NOALLOC_MAX_PARTICLES + 1)
    assert e.value.code == md.MD_ERR_WORKSPACE and "MD_NOALLOC_MAX_PARTICLES" in str(e.value)
    for kw, mass in ((dict(n=0), 1.0), (dict(), 0.0)):
        with pytest.raises(md.MDError) as e:
            md.kinetic_energy_noalloc(vel, mass, out, **kw)
        assert e.value.code == md.MD_ERR_INVALID_ARG
    md.kinetic_energy_noalloc(vel, 1.0, out)                     # and a valid call still works afterwards
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
