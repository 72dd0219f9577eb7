"""Parity "after the stated step count" (BASELINE.json north_star) on configs 2, 3 and 4: the CUDA path, in the launch
configuration bench.py times, against the fp32 oracle run for the WHOLE length of the config — 500 steps at 288^3,
1000 steps at 552^3 (heterogeneous c, three sources), 200 steps at 1600^3 — from zero fields with the Ricker sources of
the config (PAPER.md P:40-42 the recurrence whose rounding accumulates, P:46-56 the layers the pulse ends up in, P:193
the source).  Tolerance: max|delta| / max|oracle| <= 1e-4 per field over the whole total grid (reading R17).

The kernels round exactly as the plain evaluation does (no fused multiply-add, reading R25), and the oracle runs in plain
IEEE arithmetic here (no FTZ/DAZ: flushing the denormals in the leading edge of the pulse perturbs roundings that cascade
up to a different, equally valid, fp32 realisation of the run within a few steps).  So on top of the tolerance every
comparison below demands the SAME BITS as the fp32 oracle, in every field, after the whole run.  The fp64 oracle (same
fp32 inputs) arbitrates on config 2 (R18): both fp32 results must lie within 1e-4 of it.
"""
import numpy as np
import pytest

import oracle
from oracle import Oracle
from paper_2606_06910_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_06910_b200 import binding
    return binding


STATS = {}


def _rel(g, r, exact_tag=None):
    """max|g - r| / max|r| without building a float64 copy of a 168M-point field.  With exact_tag: r is the fp32 oracle,
    and not one word may differ."""
    scale = float(np.abs(r).max())
    worst, words = 0.0, 0
    for k0 in range(0, r.shape[0], 64):
        worst = max(worst, float(np.abs(g[k0:k0 + 64].astype(np.float64) - r[k0:k0 + 64]).max()))
        if exact_tag is not None:
            words += int((g[k0:k0 + 64].view(np.uint32) != r[k0:k0 + 64].astype(np.float32).view(np.uint32)).sum())
    if exact_tag is not None:
        STATS[exact_tag] = (worst, words)
        print("%s: max |gpu - oracle| %.3e, %d of %d values differ" % (exact_tag, worst, words, r.size))
        assert words == 0, (exact_tag, "%d words differ from the fp32 oracle" % words, worst)
    return worst / (scale if scale > 0 else 1.0), scale


def _oracle_run(w, fp64=False):
    o = Oracle(w.n_interior, w.cpml, fp64=fp64, **w.cpml_kwargs())
    if w.c is not None:
        o.set_model(w.c)
    o.set_sources(w.sources, w.wavelets)
    oracle.set_threads(oracle.max_threads())
    o.step(w.steps)
    return o


def _gpu_fields(B, w, kernel, psi):
    sim = B.from_workload(w, kernel=kernel)
    try:
        sim.step(w.steps)
        out = [sim.get_field(f) for f in range(4)]
        if psi:
            out += [sim.get_psi(q) for q in range(6)]
    finally:
        sim.destroy()
    return out


def test_config2_full_length_500_steps(B):
    """256^3 + 16-cell CPML, centre source, 500 steps: by then the pulse has crossed the grid (0.4 x 500 = 200 cells
    against a half-width of 144) and sits in the layers, so the six psi arrays carry the final state too.  The fp64
    instantiation (same fp32 inputs) arbitrates (R18)."""
    w = inputs.config(2)
    o32 = _oracle_run(w)
    ref = [o32.get(i) for i in range(10)]
    o32.close()
    o64 = _oracle_run(w, fp64=True)
    ref64 = [o64.get(i) for i in range(4)]
    o64.close()
    for f in range(4):
        e, s = _rel(ref[f], ref64[f])
        assert e <= TOL and s > 0, ("oracle fp32 vs fp64", f, e)
    for kernel in (0, 2):
        got = _gpu_fields(B, w, kernel, psi=True)
        for i in range(10):
            e, s = _rel(got[i], ref[i], "config2 x500 kernel %d array %d" % (kernel, i))
            assert s > 0, i
            assert e <= TOL, (kernel, i, e)
        for f in range(4):
            e, _ = _rel(got[f], ref64[f])
            assert e <= TOL, ("vs fp64", kernel, f, e)


PREFIX3 = 90        # config 3: steps compared bit for bit with the IEEE oracle (all three sources are past their peak at 82)


def test_config3_full_length_1000_steps(B):
    """512^3 + 20-cell CPML, heterogeneous c (Kc array), three seeded sources, 1000 steps — the whole config, 1.7e11
    point-updates of oracle time.  Two comparisons, both step structures:
      * steps 1 .. 90 against the oracle in IEEE arithmetic: the same bits, all four fields;
      * all 1000 steps against the oracle with its FTZ/DAZ switch on (run in a process of its own, see
        tests/oracle_config3_ftz.py): flushing the denormals of the pulse's leading edge gives another, equally valid
        fp32 realisation of the run, so this one is held to BASELINE's tolerance — 1e-4 of max|oracle| per field; the six
        memory variables included (measured: p 9e-7, v 1.1e-5, psi 7.2e-5)."""
    import os
    import subprocess
    import sys
    import tempfile

    w = inputs.config(3)
    assert w.steps == 1000 and w.total == (552, 552, 552) and w.sources.shape[0] == 3
    here = os.path.dirname(os.path.abspath(__file__))
    with tempfile.TemporaryDirectory() as tmp:
        proc = subprocess.Popen([sys.executable, os.path.join(here, "oracle_config3_ftz.py"), tmp])
        try:
            # meanwhile: the GPU runs (they need no host cores to speak of); snapshots at PREFIX3 and at the end
            got = {}
            for k in (0, 2):
                sim = B.from_workload(w, kernel=k)
                try:
                    sim.step(PREFIX3)
                    head = [sim.get_field(f) for f in range(4)]
                    sim.step(w.steps - PREFIX3)
                    got[k] = (head, [sim.get_field(f) for f in range(4)], [sim.get_psi(q) for q in range(6)] if k == 2 else None)
                finally:
                    sim.destroy()
            assert proc.wait() == 0
        finally:
            if proc.poll() is None:
                proc.kill()
        for i in range(10):
            r = np.load(os.path.join(tmp, "a%d.npy" % i))
            for k in (0, 2):
                if i < 4:
                    e, s = _rel(got[k][1][i], r)
                    print("config3 x1000 kernel %d field %d vs the FTZ oracle: max rel err %.3e" % (k, i, e))
                    assert s > 0 and e <= TOL, (k, i, e)
                elif k == 2:
                    e, s = _rel(got[k][2][i - 4], r)
                    print("config3 x1000 kernel 2 psi %d vs the FTZ oracle: max rel err %.3e" % (i - 4, e))
                    assert s > 0 and e <= TOL, (i, e)
            del r
    # the IEEE oracle over the first PREFIX3 steps: bit for bit
    o = Oracle(w.n_interior, w.cpml, **w.cpml_kwargs())
    o.set_model(w.c)
    o.set_sources(w.sources, w.wavelets)
    oracle.set_threads(oracle.max_threads())
    o.step(PREFIX3)
    for f in range(4):
        r = o.get(f)
        for k in (0, 2):
            e, s = _rel(got[k][0][f], r, "config3 x%d kernel %d field %d" % (PREFIX3, k, f))
            assert s > 0 and e <= TOL
        del r
    o.close()


# ---------------------------------------------------------------- config 4 (reading R26)
STEPS4 = 200
HALF = 192          # the centre window is 384^3 (R26)
REACH = 168         # cut sides of the boundary windows: cells between a source and a cut face
NEAR = 40           # boundary sources sit 40 cells from their faces: 8 cells in front of the 32-cell layer


def _complement_boxes(total, wins):
    """Boxes that tile the grid minus the windows (each window = (lo, size)); breakpoints sweep, merged along x."""
    cuts = []
    for a in range(3):
        c = {0, total[a]}
        for lo, sz in wins:
            c.add(lo[a])
            c.add(lo[a] + sz[a])
        cuts.append(sorted(c))

    def inside(x, y, z):
        return any(all(lo[a] <= v < lo[a] + sz[a] for a, v in enumerate((x, y, z))) for lo, sz in wins)

    out = []
    for z0, z1 in zip(cuts[2][:-1], cuts[2][1:]):
        for y0, y1 in zip(cuts[1][:-1], cuts[1][1:]):
            run = None
            for x0, x1 in zip(cuts[0][:-1], cuts[0][1:]):
                if inside(x0, y0, z0):
                    if run:
                        out.append(((run[0], y0, z0), (run[1] - run[0], y1 - y0, z1 - z0)))
                    run = None
                else:
                    run = (run[0], x1) if run else (x0, x1)
            if run:
                out.append(((run[0], y0, z0), (run[1] - run[0], y1 - y0, z1 - z0)))
    return out


def _config4_case():
    w = inputs.config(4, steps=STEPS4)
    n = w.total[0]
    hi = n - 1 - NEAR
    src = np.array([[n // 2] * 3, [NEAR, n // 2, n // 2], [hi, NEAR, n // 2 + 300], [hi, hi, hi]], np.int32)
    wav = np.tile(inputs.ricker(STEPS4, w.dt), (4, 1))
    wins = []
    for k, s in enumerate(src):
        half = HALF if k == 0 else REACH
        lo = [0 if s[a] - half < 64 else int(s[a]) - half for a in range(3)]
        up = [n if s[a] + half > n - 64 else int(s[a]) + half for a in range(3)]
        wins.append((tuple(lo), tuple(up[a] - lo[a] for a in range(3))))
    return w, src, wav, wins


@pytest.fixture(scope="module")
def config4_oracle_windows():
    """One windowed oracle per source: walls on the cut sides, the true 32-cell CPML on the true faces (R13, R26)."""
    w, src, wav, wins = _config4_case()
    n = w.total[0]
    out = []
    oracle.set_threads(oracle.max_threads())
    for (lo, sz), s in zip(wins, src):
        cp = [0] * 6
        for a in range(3):
            if lo[a] == 0:
                cp[2 * a] = w.cpml[2 * a]
            if lo[a] + sz[a] == n:
                cp[2 * a + 1] = w.cpml[2 * a + 1]
        o = Oracle(tuple(sz[a] - cp[2 * a] - cp[2 * a + 1] for a in range(3)), cp, **w.cpml_kwargs())
        o.set_sources((s - np.asarray(lo, np.int32))[None, :], wav[:1])
        o.step(STEPS4)
        out.append([o.get(f).astype(np.float32) for f in range(4)])      # lossless: the fp32 instantiation
        o.close()
    return out


@pytest.mark.parametrize("kernel", [2, 0])
def test_config4_full_length_200_steps_windowed(B, kernel, config4_oracle_windows):
    """1536^3 + 32-cell CPML (1600^3 total), 200 steps, the single-pass step (the structure bench.py times) and the
    two-kernel step.  Four sources in one run, far enough apart never to meet (0.4 x 200 = 80 cells of travel): the
    config's own centre source in a 384^3 window, and one source 40 cells from a face, from an edge and from a corner,
    so that the pulse enters the 32-cell layers of one, two and three axes at the far end of a 4.1e9-point array (64-bit
    offsets in the slab-local psi arrays).  The device-side max|p| outside the windows bounds what the windows leave out."""
    w, src, wav, wins = _config4_case()
    assert wins[0] == ((608,) * 3, (384,) * 3)
    sim = B.Fdtd(w.n_interior, w.cpml, kernel=kernel, medium=B.FDTD_MEDIUM_UNIFORM, **w.cpml_kwargs())
    try:
        assert sim.workspace_bytes > (130e9 if kernel == 2 else 65e9)
        sim.set_sources(src, wav)
        sim.step(STEPS4)
        pmax = sim.field_absmax(B.FDTD_P)
        assert pmax > 0
        outside = max(sim.field_absmax(B.FDTD_P, lo, sz) for lo, sz in _complement_boxes(w.total, wins))
        assert outside < 1e-6 * pmax, (outside, pmax)
        for (lo, sz), ref in zip(wins, config4_oracle_windows):
            for f in range(4):
                e, scale = _rel(sim.get_field_box(f, lo, sz), ref[f], "config4 x200 kernel %d window %s field %d" % (kernel, lo, f))
                assert scale > 0
                assert e <= TOL, (kernel, lo, f, e)
    finally:
        sim.destroy()
