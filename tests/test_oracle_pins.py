"""Pins for the CPU oracle (no GPU): what the paper and the mathematics fix.

Each test is chosen so that a plausible mistake in oracle/fdtd_oracle.cpp (a dropped
term, a wrong sign or index, a transposed operand, a mis-staggered table) fails it.
Citations: P:NN = PAPER.md line NN; Rn / Pn = readings and pins listed in DESIGN.md.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from oracle import Oracle
from paper_2606_06910_b200 import inputs

from conftest import golden

NU = 0.4


def _coef_f32():
    g = golden("coefficients.txt")
    return np.array([int(b, 16) for b in g["bits"]], np.uint32).view(np.float32)


def _rationals():
    return [Fraction(s) for s in golden("coefficients.txt")["rational"]]


# ---------------------------------------------------------------- P1 coefficients
def test_p1_coefficient_bits_and_taylor_conditions():
    g = golden("coefficients.txt")
    c = oracle.coeffs()
    assert list(c.view(np.uint32)) == [int(b, 16) for b in g["bits"]]
    r = _rationals()
    # correct rounding of the exact rationals
    for v, q in zip(c, r):
        assert np.float32(float(q)) == v
    # staggered Taylor conditions (R1): sum c_l (2l-1) = 1 ; sum c_l (2l-1)^{3,5,7} = 0 — exact
    assert sum(q * (2 * l + 1) for l, q in enumerate(r)) == 1
    for pw in (3, 5, 7):
        assert sum(q * (2 * l + 1) ** pw for l, q in enumerate(r)) == 0
    assert abs(float(sum(abs(q) for q in r)) - float(g["sum_abs"][0])) < 1e-14
    assert abs(float(sum(q * q for q in r)) - float(g["sum_sq"][0])) < 1e-14


# ---------------------------------------------------------------- P2 dispersion
def _S(mode, N, nu, c):
    s = 0.0
    for m in mode:
        s += sum(float(c[l]) * math.sin((2 * l + 1) * math.pi * m / N) for l in range(4)) ** 2
    return nu * nu * s


@pytest.mark.parametrize("key", ["mode123", "mode100", "mode444", "mode888"])
def test_p2_dispersion_relation(key):
    g = golden("dispersion.txt")
    mode = [int(v) for v in g[key][:3]]
    S_paper = float(g[key][3])
    N = 16
    # golden value agrees with the closed form on the exact rationals
    assert abs(_S(mode, N, NU, [float(q) for q in _rationals()]) - S_paper) < 1e-13
    # the oracle's B and Kc are fp32(0.4) (R6: rounded once), so nu^2 = fp32(0.4)^2 in the closed form
    S32 = _S(mode, N, float(np.float32(NU)), _coef_f32().astype(np.float64))
    assert abs(S32 - S_paper) < 1e-7
    o = Oracle((N,) * 3, dt=NU, boundary=1, fp64=True)
    z, y, x = np.meshgrid(*(np.arange(N),) * 3, indexing="ij")
    ph = 2 * math.pi * (mode[0] * x + mode[1] * y + mode[2] * z) / N
    p0 = np.cos(ph + 0.3)
    o.set(oracle.P, p0)
    hist = [p0]
    for _ in range(6):
        o.step(1)
        hist.append(o.get(oracle.P))
    for n in range(1, 6):
        res = hist[n + 1] + hist[n - 1] - (2 - 4 * S32) * hist[n]
        assert np.abs(res).max() < 2e-13, (n, np.abs(res).max())
    # a mis-staggered operator changes S at the 1e-2 level: make sure the pin has teeth
    assert abs((2 - 4 * S32) - (2 - 4 * S32 * 1.01)) > 1e-4 or S32 < 1e-2


# ---------------------------------------------------------------- P3 spatial order
def test_p3_spatial_order_eight():
    g = golden("spatial_order.txt")
    c = [float(q) for q in _rationals()]
    errs = []
    for N in (30, 60, 120, 240):
        th = 2 * math.pi * 4 / N
        sym = sum(c[l] * 2 * math.sin((2 * l + 1) * th / 2) for l in range(4)) / th
        errs.append(abs(1 - sym * sym))
        assert abs(errs[-1] - float(g["N%d" % N][0])) < 2e-3 * float(g["N%d" % N][0]) + 2e-15
    # 2nd-order staggered operator applied twice reproduces the 2nd-order row of the paper's Table 6
    for N, ref in zip((30, 60, 120, 240, 480), g["table6_order2"]):
        th = 2 * math.pi * 4 / N
        e2 = abs(1 - (2 * math.sin(th / 2) / th) ** 2)
        assert abs(e2 - float(ref)) < 6e-4 * float(ref)
    # the oracle's own D+ on a sampled mode: relative error of (D- D+) p vs -k^2 p at N = 30, 60
    c32 = _coef_f32().astype(np.float64)            # the oracle carries the fp32-rounded weights
    for N in (30, 60):
        th = 2 * math.pi * 4 / N
        ref = abs(1 - (sum(c32[l] * 2 * math.sin((2 * l + 1) * th / 2) for l in range(4)) / th) ** 2)
        o = Oracle((N, 4, 4), dt=1.0, boundary=1, fp64=True)
        x = np.arange(N)
        p0 = np.broadcast_to(np.sin(2 * math.pi * 4 * x / N), (4, 4, N)).copy()
        o.set(oracle.P, p0)
        o.step(1)                                  # p1 = p0 + D-D+ p0 (B = Kc = 1)
        lap = o.get(oracle.P) - p0
        k2 = (2 * math.pi * 4 / N) ** 2
        got = np.abs(lap + k2 * p0).max() / (k2 * np.abs(p0).max())
        assert abs(got - ref) < 1e-12, (got, ref)


# ---------------------------------------------------------------- P4 impulse response
@pytest.mark.parametrize("fp64", [True, False])
def test_p4_one_step_impulse_response(fp64):
    g = golden("impulse.txt")
    L = [float(Fraction(s)) for s in g["L"]]
    N, s = 24, 11
    o = Oracle((N,) * 3, dt=NU, fp64=fp64)
    p0 = np.zeros((N,) * 3)
    p0[s, s, s] = 1.0
    o.set(oracle.P, p0)
    o.substep_v()
    c = _coef_f32().astype(np.float64)
    B = float(np.float32(NU))
    vx, vy, vz = o.get(oracle.VX), o.get(oracle.VY), o.get(oracle.VZ)
    exp_v = np.zeros(N)
    for l in range(1, 5):
        exp_v[s - l] = -B * c[l - 1]
        exp_v[s + l - 1] = +B * c[l - 1]
    tol = 1e-15 if fp64 else 1e-7
    assert np.abs(vx[s, s, :] - exp_v).max() < tol
    assert np.abs(vy[s, :, s] - exp_v).max() < tol
    assert np.abs(vz[:, s, s] - exp_v).max() < tol
    for v in (vx, vy, vz):                       # nothing off the three axis lines
        assert np.count_nonzero(v) == 8
    o.substep_p()
    p1 = o.get(oracle.P)
    tol = 2e-7                                   # fp32-rounded weights / nu vs the exact rationals
    assert abs(p1[s, s, s] - float(g["center"][0])) < tol
    for m in range(1, 8):
        for sgn in (-1, 1):
            e = NU * NU * L[m - 1]
            assert abs(p1[s, s, s + sgn * m] - e) < tol
            assert abs(p1[s, s + sgn * m, s] - e) < tol
            assert abs(p1[s + sgn * m, s, s] - e) < tol
    assert np.count_nonzero(p1) == 1 + 6 * 7
    # kernel of D-D+: L(0) = -2 sum c^2, sum over all offsets = 0, second moment = 2 (consistency with d^2/dx^2)
    sum_sq = float(golden("coefficients.txt")["sum_sq"][0])
    assert abs(sum(L) - sum_sq) < 1e-15 and abs(sum(m * m * L[m - 1] for m in range(1, 8)) - 1.0) < 1e-14


# ---------------------------------------------------------------- P5 / P6 symmetries
def _run_centre_source(N, L, steps, fp64, src=None):
    o = Oracle((N - 2 * L,) * 3, (L,) * 6, dt=NU, cpml_alpha_max=math.pi * inputs.F0, fp64=fp64)
    src = src if src is not None else (N // 2,) * 3
    o.set_sources([src], inputs.ricker(steps, NU)[None])
    o.step(steps)
    return o


@pytest.mark.parametrize("fp64", [False, True])
def test_p5_reflection_symmetry_bit_exact(fp64):
    N, L = 33, 6                                  # odd N: the grid mirrors about the centre node (R3)
    o = _run_centre_source(N, L, 60, fp64)
    p, vx, vy, vz = (o.get(w) for w in range(4))
    assert np.abs(p).max() > 0
    assert np.array_equal(p, p[:, :, ::-1]) and np.array_equal(p, p[:, ::-1, :]) and np.array_equal(p, p[::-1])
    # v_a(i) = -v_a(N-2-i) along its own axis; the pinned last half node stays 0
    assert np.array_equal(vx[:, :, :-1], -vx[:, :, -2::-1]) and not vx[:, :, -1].any()
    assert np.array_equal(vy[:, :-1, :], -vy[:, -2::-1, :]) and not vy[:, -1, :].any()
    assert np.array_equal(vz[:-1], -vz[-2::-1]) and not vz[-1].any()
    # CPML tables mirror: integer nodes b(i) = b(N-1-i); half nodes b(i) = b(N-2-i)
    a, b, ik, inn = o.cpml_table(0, 0)
    assert np.array_equal(b, b[::-1]) and np.array_equal(a, a[::-1]) and inn[:L].all() and not inn[L:N - L].any()
    a, b, ik, inn = o.cpml_table(0, 1)
    assert np.array_equal(b[:-1], b[-2::-1]) and np.array_equal(a[:-1], a[-2::-1])


def test_p6_axis_permutation_symmetry():
    N, L = 28, 6
    o = _run_centre_source(N, L, 50, True, src=(11, 11, 11))
    p, vx, vy, vz = (o.get(w) for w in range(4))
    sc = np.abs(p).max()
    for perm in ((0, 2, 1), (1, 0, 2), (2, 1, 0), (1, 2, 0)):
        assert np.abs(p - p.transpose(perm)).max() < 1e-12 * sc
    # arrays are (z,y,x): swapping x<->y maps vx -> vy
    assert np.abs(vx - vy.transpose(0, 2, 1)).max() < 1e-12 * np.abs(vx).max()
    assert np.abs(vx - vz.transpose(2, 1, 0)).max() < 1e-12 * np.abs(vx).max()


def test_r2_all_three_divergence_terms_present():
    """P:40 prints only the x and y terms; P:56 has all three (R2).  A z-only gradient must move p."""
    N = 20
    o = Oracle((N,) * 3, dt=NU, fp64=True)
    vz = np.zeros((N,) * 3)
    vz[9, 10, 10] = 1.0
    o.set(oracle.VZ, vz)
    o.substep_p()
    p = o.get(oracle.P)
    c = _coef_f32().astype(np.float64)
    assert abs(p[9, 10, 10] + NU * c[0]) < 1e-8 and abs(p[10, 10, 10] - NU * c[0]) < 1e-8


# ---------------------------------------------------------------- P7 CPML -> interior
@pytest.mark.parametrize("fp64", [False, True])
def test_p7_cpml_reduces_to_interior(fp64):
    """sigma = 0, alpha = 0, kappa = 1 => b = 1, a = 0 and the update is the interior one, bit for bit."""
    N, L, steps = 30, 7, 40
    w = inputs.ricker(steps, NU)[None]
    a = Oracle((N - 2 * L,) * 3, (L,) * 6, dt=NU, cpml_R0=1.0, cpml_alpha_max=0.0, fp64=fp64)   # ln(1) = 0 -> sigma_max = 0
    b = Oracle((N,) * 3, (0,) * 6, dt=NU, fp64=fp64)
    for o in (a, b):
        o.set_sources([(13, 14, 15)], w)
        o.step(steps)
    ta, tb, tik, tin = a.cpml_table(1, 1)
    assert tin[:L].all() and np.all(ta == 0) and np.all(tb[tin == 1] == 1) and np.all(tik == 1)
    for wch in range(4):
        assert np.array_equal(a.get(wch), b.get(wch))
    for wch in range(4, 10):
        assert not a.get(wch).any()


# ---------------------------------------------------------------- P8 energy
def test_p8_energy_conserved_without_cpml_heterogeneous():
    """D- = -(D+)^T with the wall / pinned-node rule (R3, R4) makes the leapfrog energy (R19) exact."""
    N = 18
    rng = np.random.default_rng(5)
    c = (1.0 + 0.2 * rng.random((N,) * 3)).astype(np.float32)
    rho = (1.0 + 0.5 * rng.random((N,) * 3)).astype(np.float32)
    o = Oracle((N,) * 3, dt=0.3, fp64=True)
    o.set_model(c, rho)
    o.set(oracle.P, rng.standard_normal((N,) * 3))
    o.track_energy(True)
    es = []
    for _ in range(40):
        o.step(1)
        es.append(o.energy())
    es = np.array(es)
    assert es[0] > 0 and np.abs(es / es[0] - 1).max() < 1e-6     # fp32-rounded B, Kc break exactness at 1e-7
    o2 = Oracle((N,) * 3, dt=0.3, fp64=True)
    o2.set(oracle.P, rng.standard_normal((N,) * 3))
    o2.track_energy(True)
    es = []
    for _ in range(40):
        o2.step(1)
        es.append(o2.energy())
    es = np.array(es)
    assert np.abs(es / es[0] - 1).max() < 1e-12                   # homogeneous: B, Kc exact -> round-off only


def test_p8_energy_decays_with_cpml_and_not_without():
    """Fig. 3: after the source ends the CPML run loses orders of magnitude, the wall run keeps its energy."""
    n, L, steps = 24, 10, 700
    w = inputs.ricker(steps, NU)[None]
    t_end = int((1 / inputs.F0 + 6 / (math.pi * inputs.F0)) / NU) + 1      # Ricker tail < 1e-14 of its peak
    out = {}
    for name, cp in (("cpml", (L,) * 6), ("wall", (0,) * 6)):
        tot = n + 2 * L
        o = Oracle((n,) * 3 if cp[0] else (tot,) * 3, cp, dt=NU, cpml_alpha_max=math.pi * inputs.F0, fp64=True)
        # energy is summed over the same n^3 box in both runs only for cpml; wall run sums the whole box
        o.set_sources([(tot // 2,) * 3], w)
        o.track_energy(True)
        es = []
        for s in range(steps):
            o.step(1)
            if s % 10 == 0:
                es.append(o.energy())
        out[name] = np.array(es)
    k0 = t_end // 10 + 1
    e = out["cpml"]
    peak = e.max()
    assert e[-1] < 1e-4 * peak, (peak, e[-1])                    # "several orders of magnitude"
    assert np.all(np.diff(e[k0:]) <= 1e-6 * peak)                # non-increasing once the source is silent
    ew = out["wall"]
    assert ew[-1] > 0.25 * ew.max() and e[-1] < 1e-4 * ew[-1]
    assert np.abs(ew[k0:] / ew[k0] - 1).max() < 1e-9             # retained: trapped by the reflecting walls


# ---------------------------------------------------------------- P9 stability edge
def test_p9_stability_edge():
    g = golden("dispersion.txt")
    lim = 1 / (math.sqrt(3) * float(sum(abs(q) for q in _rationals())))
    assert abs(lim - float(g["nu_max"][0])) < 1e-6
    N = 8
    z, y, x = np.meshgrid(*(np.arange(N),) * 3, indexing="ij")
    chk = (-1.0) ** (x + y + z)
    amp = {}
    for nu in (0.44, 0.46):
        o = Oracle((N,) * 3, dt=nu, boundary=1, fp64=True)
        o.set(oracle.P, chk)
        o.step(400)
        amp[nu] = np.abs(o.get(oracle.P)).max()
    assert amp[0.44] < 10.0          # bounded: |p^n| <= 1/cos(theta/2)-type factor from the inconsistent v start, no growth
    assert amp[0.46] > 1e3


# ---------------------------------------------------------------- P10 time order
def test_p10_second_order_in_time():
    """Standing wave of P:162 in periodic mode; error vs dt halves at rate 2.00 (Table 7's rate)."""
    N, m, T = 32, 1, 0.5
    h = 1.0 / N
    w = 2 * math.pi * m * math.sqrt(3.0)
    xs = (np.arange(N)) * h
    z, y, x = np.meshgrid(xs, xs, xs, indexing="ij")
    k = 2 * math.pi * m
    errs = []
    for nsteps in (40, 80, 160):
        dt = T / nsteps
        o = Oracle((N,) * 3, dx=h, dt=dt, boundary=1, fp64=True)
        o.set(oracle.P, np.sin(k * x) * np.sin(k * y) * np.sin(k * z))
        # v^{-1/2} = +grad(A) sin(w dt/2)/w at the half nodes (v_t = -grad p, rho = 1)
        s = math.sin(w * dt / 2) / w
        o.set(oracle.VX, k * np.cos(k * (x + h / 2)) * np.sin(k * y) * np.sin(k * z) * s)
        o.set(oracle.VY, k * np.sin(k * x) * np.cos(k * (y + h / 2)) * np.sin(k * z) * s)
        o.set(oracle.VZ, k * np.sin(k * x) * np.sin(k * y) * np.cos(k * (z + h / 2)) * s)
        o.step(nsteps)
        exact = np.sin(k * x) * np.sin(k * y) * np.sin(k * z) * math.cos(w * T)
        errs.append(np.abs(o.get(oracle.P) - exact).max())
    r1, r2 = math.log2(errs[0] / errs[1]), math.log2(errs[1] / errs[2])
    assert abs(r1 - 2.0) < 0.05 and abs(r2 - 2.0) < 0.05, (errs, r1, r2)


# ---------------------------------------------------------------- W2 CPML tables
def test_w2_worked_cpml_tables():
    g = golden("cpml_tables_config1.txt")
    w = inputs.config(1)
    o = Oracle(w.n_interior, w.cpml, **w.cpml_kwargs())
    smax = -(2 + 1) * 1.0 * math.log(1e-5) / (2 * 8 * 1.0)
    assert abs(smax - float(g["sigma_max"][0])) < 1e-12
    assert abs(w.cpml_alpha_max - float(g["alpha_max"][0])) < 1e-14
    assert abs(-4 * math.log(1e-8) / (2 * 20 * 1.0) - float(g["paper_sigma_max"][0])) < 1e-5
    for axis in range(3):
        a, b, ik, inn = o.cpml_table(axis, 0)
        assert np.allclose(b[:8], [float(v) for v in g["b_int"]], rtol=0, atol=6e-8)
        assert np.allclose(a[:8], [float(v) for v in g["a_int"]], rtol=0, atol=6e-8)
        assert list(inn[:9]) == [1] * 8 + [0] and list(inn[-9:]) == [0] + [1] * 8
        assert np.array_equal(b[:8], b[::-1][:8])
        a, b, ik, inn = o.cpml_table(axis, 1)
        assert np.allclose(b[:8], [float(v) for v in g["b_half"]], rtol=0, atol=6e-8)
        assert np.allclose(a[:8], [float(v) for v in g["a_half"]], rtol=0, atol=6e-8)
        assert np.all(ik == 1)
        # high-side half-node slab is [N-1-L, N-2] (R8)
        assert list(inn[-10:]) == [0] + [1] * 9
    # at rho = 1 alpha = 0 => a = b - 1 (R11: a < 0, psi opposes the derivative)
    a, b, _, _ = o.cpml_table(0, 0)
    assert abs(a[0] - (b[0] - 1)) < 1e-7 and a[0] < 0


def test_cpml_paper_parameter_set_kappa_profile():
    """The paper's own set: q = 3, R = 1e-8, kappa_max = 5, alpha_max = 0.05 sigma_max, L = 20."""
    L = 20
    smax = -4 * math.log(1e-8) / (2 * L)
    o = Oracle((24,) * 3, (L,) * 6, dt=0.05, cpml_order=3, cpml_R0=1e-8, cpml_kappa_max=5.0,
               cpml_alpha_max=0.05 * smax, cpml_c_ref=1.0)
    a, b, ik, inn = o.cpml_table(2, 0)
    assert abs(ik[0] - 1 / 5.0) < 1e-7                           # rho = 1 at the outermost node
    rho = (L - 3) / L
    sig, kap, al = smax * rho ** 3, 1 + 4 * rho ** 3, 0.05 * smax * (1 - rho)
    bb = math.exp(-(sig / kap + al) * 0.05)
    assert abs(b[3] - bb) < 1e-7 and abs(a[3] - sig * (bb - 1) / (kap * (sig + kap * al))) < 1e-7


# ---------------------------------------------------------------- infrastructure checks
def test_threads_bit_identical_and_hash_generator():
    w = inputs.config(1, scale=16, steps=12)
    res = []
    for nt in (1, 4):
        oracle.set_threads(nt)
        o = Oracle(w.n_interior, w.cpml, **w.cpml_kwargs())
        o.fill_hash(oracle.P, 77)
        o.set_sources(w.sources, w.wavelets)
        o.step(12)
        res.append([o.get(i) for i in range(10)])
    oracle.set_threads(oracle.max_threads())
    for a, b in zip(*res):
        assert np.array_equal(a, b)
    # oracle's own counter-based generator == the shared input generator, at a window of a larger grid
    o = Oracle((6, 5, 4))
    o.fill_hash(oracle.VY, 123, gdim=(1600, 1600, 1600), off=(1590, 7, 1500), scale=0.5)
    ref = inputs.hash_field(123, oracle.VY, (1600, 1600, 1600), off=(1590, 7, 1500), shape=(6, 5, 4), scale=0.5)
    assert np.array_equal(o.get(oracle.VY).astype(np.float32), ref)
    assert -1 <= ref.min() * 2 and ref.max() * 2 < 1


def test_window_equals_full_run_inside_domain_of_dependence():
    """R26: a window cut out of a larger grid reproduces the full run wherever the cut faces are
    farther than 8 cells per step (2 sub-updates x radius 4) — including across CPML faces."""
    full = (40, 36, 32)
    L = 6
    steps = 2
    kw = dict(dt=NU, cpml_alpha_max=math.pi * inputs.F0)
    o = Oracle(tuple(f - 2 * L for f in full), (L,) * 6, **kw)
    for wch in range(4):
        o.fill_hash(wch, 9)
    o.step(steps)
    # window at the low-x / high-y / low-z corner: 3 true faces, 3 cut faces
    wsz, off = (28, 26, 24), (0, 36 - 26, 0)
    cp = (L, 0, 0, L, L, 0)
    ow = Oracle((wsz[0] - L, wsz[1] - L, wsz[2] - L), cp, **kw)
    for wch in range(4):
        ow.fill_hash(wch, 9, gdim=full, off=off)
    ow.step(steps)
    m = 8 * steps
    for wch in range(4):
        a = o.get(wch)[0:wsz[2] - m, off[1] + m:36, 0:wsz[0] - m]
        b = ow.get(wch)[0:wsz[2] - m, m:, 0:wsz[0] - m]
        assert np.array_equal(a, b), wch
