"""The fp64 "verification precision" on the GPU ("double precision where stated", Tables 6-7 P:199-224;
SURVEY NEXT-3): fields, CPML memory variables and arithmetic in double, every coefficient the fp32 number of the fp32
path — the same contract as the oracle's fp64 instantiation, whose bits it must reproduce.  The convergence procedures of
Tables 6 and 7 are then run on the GPU: 8th order in space on the p-v operator (pin P3), 2.00 in time (pin P10)."""
import math

import numpy as np
import pytest

import oracle
from oracle import Oracle
from paper_2606_06910_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_06910_b200 import binding
    return binding


def _same(a, b):
    return np.array_equal(np.ascontiguousarray(a, np.float64).view(np.uint64), np.ascontiguousarray(b, np.float64).view(np.uint64))


def test_fp64_config1_has_the_bits_of_the_fp64_oracle(B):
    w = inputs.config(1)
    sim = B.from_workload(w, precision=B.FDTD_PRECISION_FP64)
    assert sim.kernel_in_use() == B.FDTD_KERNEL_REF
    o = Oracle(w.n_interior, w.cpml, fp64=True, **w.cpml_kwargs())
    o.set_sources(w.sources, w.wavelets)
    sim.step(w.steps)
    o.step(w.steps)
    for f in range(4):
        g = sim.get_field(f)
        assert g.dtype == np.float64 and np.abs(g).max() > 0
        assert _same(g, o.get(f)), f
    for q in range(6):
        assert _same(sim.get_psi(q), o.get(4 + q)), q
    # and it is a different thing from the fp32 run: the two differ at fp32 rounding level
    s32 = B.from_workload(w)
    s32.step(w.steps)
    d = np.abs(s32.get_field(0).astype(np.float64) - sim.get_field(0)).max() / np.abs(sim.get_field(0)).max()
    assert 1e-9 < d < 1e-4
    buf = np.empty(sim.shape, np.float32)
    with pytest.raises(B.FdtdError):                               # the fp32 entry points refuse an fp64 context
        B._check(B.lib.fdtd_get_field(sim._h, 0, buf.ctypes.data), "fdtd_get_field")
    s32.destroy()
    sim.destroy()


def test_fp64_heterogeneous_paper_cpml_set_random_state(B):
    """c(x) and rho(x) arrays, the paper's CPML set (kappa_max = 5), random fp64 state set through fdtd_set_field_f64."""
    shape, cpml = (44, 30, 37), (12, 9, 0, 7, 6, 10)
    tot = tuple(shape[a] + cpml[2 * a] + cpml[2 * a + 1] for a in range(3))
    rng = np.random.default_rng(8)
    c = (1.0 + 0.3 * rng.random(tot[::-1])).astype(np.float32)
    rho = (0.8 + 0.7 * rng.random(tot[::-1])).astype(np.float32)
    smax = -4 * math.log(1e-8) / (2 * 12)
    kw = dict(dt=0.4 / 1.3, cpml_order=3, cpml_R0=1e-8, cpml_kappa_max=5.0, cpml_alpha_max=0.05 * smax, cpml_c_ref=1.3)
    sim = B.Fdtd(shape, cpml, precision=B.FDTD_PRECISION_FP64, density=B.FDTD_DENSITY_ARRAY, **kw)
    o = Oracle(shape, cpml, fp64=True, **kw)
    sim.set_model(c, rho)
    o.set_model(c, rho)
    for f in range(4):
        a = rng.standard_normal(tot[::-1])
        sim.set_field(f, a)
        o.set(f, a)
    src = np.array([[tot[0] // 2, tot[1] // 3, tot[2] // 2]], np.int32)
    wav = inputs.ricker(12, kw["dt"], t0=1.0)[None, :]
    sim.set_sources(src, wav)
    o.set_sources(src, wav)
    sim.step(12)
    o.step(12)
    for f in range(4):
        assert _same(sim.get_field(f), o.get(f)), f
    for q in range(6):
        assert _same(sim.get_psi(q), o.get(4 + q)), q
    sim.destroy()


def test_fp64_refuses_what_it_does_not_run(B):
    for kw in (dict(kernel=B.FDTD_KERNEL_FUSED), dict(decomp=(1, 2, 2), ghost=8, substeps=2)):
        with pytest.raises(B.FdtdError):
            B.Fdtd((32,) * 3, dt=0.4, precision=B.FDTD_PRECISION_FP64, **kw)


def test_fp64_spatial_order_eight_on_the_gpu(B):
    """Method of Table 6 on the scheme's own operator: one step with B = Kc = 1 applies D- D+ to a sampled
    mode; the relative error against -k^2 is the closed form |1 - (D^/ik)^2| of the operator's symbol, evaluated with the
    fp32-rounded weights the kernels carry (pin P3: 5.04e-5 at N = 30 with the exact rationals), and falls at 8th order
    until the rounding of the weights themselves (relative 3e-8) shows."""
    c32 = B.fdtd_coeffs().astype(np.float64)
    errs, refs = [], []
    for N in (30, 60, 120):
        sim = B.Fdtd((N, 4, 4), dt=1.0, boundary=B.FDTD_PERIODIC, precision=B.FDTD_PRECISION_FP64)
        x = np.arange(N)
        p0 = np.broadcast_to(np.sin(2 * math.pi * 4 * x / N), (4, 4, N)).copy()
        sim.set_field(B.FDTD_P, p0)
        sim.step(1)
        lap = sim.get_field(B.FDTD_P) - p0
        th = 2 * math.pi * 4 / N
        errs.append(np.abs(lap + th * th * p0).max() / (th * th * np.abs(p0).max()))
        refs.append(abs(1 - (sum(c32[l] * 2 * math.sin((2 * l + 1) * th / 2) for l in range(4)) / th) ** 2))
        sim.destroy()
    for e, r in zip(errs, refs):
        assert abs(e - r) < 1e-12, (errs, refs)
    assert abs(errs[0] - 5.038e-5) < 3e-8                      # the exact-rational value of pin P3, to the weights' rounding
    r1 = math.log2(errs[0] / errs[1])
    assert 7.8 < r1 < 8.2, (errs, r1)


def test_fp64_temporal_order_two_on_the_gpu(B):
    """Standing wave of P:162 in a periodic box; the error against the exact solution falls at rate 2.00 when dt is
    halved (Table 7's rate).  Same procedure as pin P10, on the GPU."""
    N, m, T = 32, 1, 0.5
    h = 1.0 / N
    wf = 2 * math.pi * m * math.sqrt(3.0)
    xs = np.arange(N) * h
    z, y, x = np.meshgrid(xs, xs, xs, indexing="ij")
    k = 2 * math.pi * m
    errs = []
    for nsteps in (40, 80, 160):
        dt = T / nsteps
        sim = B.Fdtd((N,) * 3, dx=h, dt=dt, boundary=B.FDTD_PERIODIC, precision=B.FDTD_PRECISION_FP64)
        s = math.sin(wf * dt / 2) / wf
        sim.set_field(B.FDTD_P, np.sin(k * x) * np.sin(k * y) * np.sin(k * z))
        sim.set_field(B.FDTD_VX, k * np.cos(k * (x + h / 2)) * np.sin(k * y) * np.sin(k * z) * s)
        sim.set_field(B.FDTD_VY, k * np.sin(k * x) * np.cos(k * (y + h / 2)) * np.sin(k * z) * s)
        sim.set_field(B.FDTD_VZ, k * np.sin(k * x) * np.sin(k * y) * np.cos(k * (z + h / 2)) * s)
        sim.step(nsteps)
        exact = np.sin(k * x) * np.sin(k * y) * np.sin(k * z) * math.cos(wf * T)
        errs.append(np.abs(sim.get_field(B.FDTD_P) - exact).max())
        sim.destroy()
    r1, r2 = math.log2(errs[0] / errs[1]), math.log2(errs[1] / errs[2])
    assert abs(r1 - 2.0) < 0.05 and abs(r2 - 2.0) < 0.05, (errs, r1, r2)
