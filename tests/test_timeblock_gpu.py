"""k-step temporal blocking inside one GPU (second half; the single-device analogue of the paper's enlarged
ghost, whose s = 8 loses to s = 4 because of redundant work): k time steps per pass over z
slabs, each slab recomputing 8 planes of ghost per remaining step on both sides.  The result must have the bits of k single
steps (and so of the oracle); the redundant compute is counted by the library."""
import math

import numpy as np
import pytest

from oracle import Oracle
from paper_2606_06910_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_06910_b200 import binding
    return binding


def _bits(a, b):
    return np.array_equal(np.ascontiguousarray(a).view(np.uint32), np.ascontiguousarray(b, np.float32).view(np.uint32))


@pytest.mark.parametrize("k,planes", [(2, 0), (2, 8), (2, 24), (3, 16), (4, 12), (4, 40)])
def test_time_blocked_steps_have_the_bits_of_single_steps(B, k, planes):
    """Heterogeneous c, CPML on all faces (unequal), three sources (one inside a z layer, one on a slab boundary), random
    initial state; 13 steps = whole blocks plus a remainder taken as single steps."""
    shape, cpml = (100, 40, 90), (12, 12, 8, 8, 10, 6)
    tot = tuple(shape[a] + cpml[2 * a] + cpml[2 * a + 1] for a in range(3))
    rng = np.random.default_rng(21)
    c = (1.0 + 0.3 * rng.random(tot[::-1])).astype(np.float32)
    kw = dict(dt=0.4 / 1.3, cpml_alpha_max=math.pi * inputs.F0, cpml_c_ref=1.3)
    steps = 13
    src = np.array([[60, 30, 4], [20, 10, 24], [100, 40, 70]], np.int32)
    wav = np.stack([inputs.ricker(steps, kw["dt"], t0=1.0), 0.1 * np.ones(steps, np.float32), np.linspace(-1, 1, steps).astype(np.float32)])
    o = Oracle(shape, cpml, **kw)
    o.set_model(c)
    o.set_sources(src, wav)
    sim = B.Fdtd(shape, cpml, kernel=B.FDTD_KERNEL_FUSED, time_block=k, time_block_planes=planes, **kw)
    sim.set_model(c)
    sim.set_sources(src, wav)
    for f in range(4):
        sim.fill_hash(f, 5, 0.5)
        o.fill_hash(f, 5, scale=0.5)
    sim.step(steps)
    o.step(steps)
    for f in range(4):
        assert _bits(sim.get_field(f), o.get(f)), (k, planes, f)
    for q in range(6):
        assert _bits(sim.get_psi(q), o.get(4 + q)), (k, planes, q)
    done, owned = sim.time_block_stats()
    assert owned == tot[2] * k * (steps // k)
    assert done > owned if 0 < planes < tot[2] else done >= owned       # ghost planes were recomputed, and counted
    sim.destroy()


def test_time_block_needs_the_single_pass_kernel(B):
    with pytest.raises(B.FdtdError):
        B.Fdtd((32,) * 3, dt=0.4, time_block=2)
    with pytest.raises(B.FdtdError):
        B.Fdtd((32,) * 3, dt=0.4, kernel=B.FDTD_KERNEL_FUSED, time_block=2, decomp=(1, 2, 1), ghost=8, substeps=2)


def test_time_block_config2_matches_single_steps_at_full_size(B):
    """BASELINE config 2 (288^3), 40 steps from zero fields with its source: k = 2 against k = 1, bit for bit."""
    w = inputs.config(2, steps=40)
    ref = B.from_workload(w, kernel=B.FDTD_KERNEL_FUSED)
    ref.step(40)
    sim = B.from_workload(w, kernel=B.FDTD_KERNEL_FUSED, time_block=2)
    sim.step(40)
    for f in range(4):
        a = ref.get_field(f)
        assert np.abs(a).max() > 0 and _bits(sim.get_field(f), a), f
    ref.destroy()
    sim.destroy()
