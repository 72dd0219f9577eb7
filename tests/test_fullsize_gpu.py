"""Parity at BASELINE's full sizes, in the launch configuration bench.py times (reading R26).

The oracle cannot run 552^3 or 1600^3, but the scheme's numerical reach is 8 cells per step (2 sub-updates x radius 4,
PAPER.md P:42), so a window cut out of the grid reproduces the full run wherever its cut faces are farther than
8 * steps cells (pinned on the oracle by test_window_equals_full_run_inside_domain_of_dependence).  Every field starts
from the counter-based random state (the same generator on both sides), so every window — centre, faces, edges,
corners, and the far end of a 4.1e9-point array — carries non-trivial data and live CPML memory variables."""
import numpy as np
import pytest

from oracle import Oracle
from paper_2606_06910_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-4
STEPS = 3
W = 72                      # window edge; 8 * STEPS = 24 cells are lost on every cut side
SEED = 2606


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_06910_b200 import binding
    return binding


def _windows(total):
    """Window origins: low corner, high corner, centre, the middle of the x-high face, a y-low / z-high edge, an odd
    (tile-straddling) spot on the y-high face.  A window either contains a face or stays clear of that face's layer."""
    n = total
    mid = [(t - W) // 2 for t in n]
    hi = [t - W for t in n]
    return [(0, 0, 0), tuple(hi), tuple(mid), (hi[0], mid[1], mid[2]), (mid[0], 0, hi[2]), (41, hi[1], mid[2] + 7)]


def _check(B, w, sim):
    total = w.total
    for f in range(4):
        sim.fill_hash(f, SEED, 0.5)
    sim.step(STEPS)
    worst = 0.0
    for off in _windows(total):
        size = tuple(min(W, total[a] - off[a]) for a in range(3))
        cp = [0] * 6
        cut_lo, cut_hi = [0] * 3, [0] * 3
        for a in range(3):
            if off[a] == 0:
                cp[2 * a] = w.cpml[2 * a]
            else:
                cut_lo[a] = 8 * STEPS
            if off[a] + size[a] == total[a]:
                cp[2 * a + 1] = w.cpml[2 * a + 1]
            else:
                cut_hi[a] = 8 * STEPS
        interior = tuple(size[a] - cp[2 * a] - cp[2 * a + 1] for a in range(3))
        o = Oracle(interior, cp, **w.cpml_kwargs())
        if w.c is not None:
            o.set_model(np.ascontiguousarray(w.c[off[2]:off[2] + size[2], off[1]:off[1] + size[1], off[0]:off[0] + size[0]]))
        inside = [k for k, s in enumerate(w.sources) if all(off[a] <= s[a] < off[a] + size[a] for a in range(3))]
        if inside:
            o.set_sources(w.sources[inside] - np.asarray(off, np.int32), w.wavelets[inside])
        for f in range(4):
            o.fill_hash(f, SEED, gdim=total, off=off, scale=0.5)
        o.step(STEPS)
        lo = [off[a] + cut_lo[a] for a in range(3)]
        sz = [size[a] - cut_lo[a] - cut_hi[a] for a in range(3)]
        for f in range(4):
            g = sim.get_field_box(f, lo, sz).astype(np.float64)
            r = o.get(f)[cut_lo[2]:size[2] - cut_hi[2], cut_lo[1]:size[1] - cut_hi[1], cut_lo[0]:size[0] - cut_hi[0]]
            err = float(np.abs(g - r).max() / np.abs(r).max())
            worst = max(worst, err)
            assert err <= TOL, (w.name, off, f, err)
    return worst


def test_config2_full_size_windows(B):
    w = inputs.config(2)
    sim = B.from_workload(w)
    _check(B, w, sim)
    sim.destroy()


@pytest.mark.parametrize("kernel", [0, 2])
def test_config3_full_size_windows_heterogeneous(B, kernel):
    w = inputs.config(3, steps=8)
    sim = B.from_workload(w, kernel=kernel)
    _check(B, w, sim)
    sim.destroy()


def test_config4_full_size_windows_fused_step(B):
    """The single-pass step at 1600^3: two copies of the state (131 GB of fields + psi) in one workspace, 64-bit offsets in
    both, odd number of buffer swaps."""
    w = inputs.config(4, steps=8)
    sim = B.from_workload(w, kernel=B.FDTD_KERNEL_FUSED)
    assert sim.workspace_bytes > 130e9
    _check(B, w, sim)
    sim.destroy()


def test_config4_full_size_windows_64bit_indexing(B):
    """1600^3: 4.096e9 points per field (> 2^31 elements, > 2^32 bytes); the high-corner window ends at the last element."""
    w = inputs.config(4, steps=8)
    sim = B.from_workload(w)
    assert sim.workspace_bytes > 65e9
    _check(B, w, sim)
    # nothing outside the numerical reach of a lone source after a few steps: a fresh run from zero fields
    sim.destroy()
    sim = B.from_workload(w)
    sim.step(4)
    c = w.sources[0]
    r = 8 * 4 + 1
    assert sim.field_absmax(B.FDTD_P, (0, 0, 0), (1600, 1600, int(c[2]) - r)) == 0.0
    assert sim.field_absmax(B.FDTD_P, (0, 0, int(c[2]) + r), (1600, 1600, 1600 - int(c[2]) - r)) == 0.0
    assert sim.field_absmax(B.FDTD_P) > 0.0
    sim.destroy()
