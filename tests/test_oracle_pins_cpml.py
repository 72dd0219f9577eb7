"""More pins for the CPU oracle (no GPU): the terms round 1 left without a dynamic check.

  K1/K2  the coordinate-stretching factor (1/kappa) of PAPER.md P:46 with kappa != 1, through one sub-update, at both
         staggerings, on both faces, along every axis (exact values, in the manner of pin P4);
  K3     (1/kappa) d + psi with a live psi: kappa divides the derivative only, psi is refreshed first (R10);
  T1     the paper's own parameter set (Table 2) on an axis with unequal layers: tables on both faces and both
         staggerings against values worked by hand (tests/golden/cpml_tables_paper_set.txt);
  D1/D2  heterogeneous medium (reading R6): rho_bar = arithmetic mean of the two adjacent nodes, K = rho c^2.

A plausible slip in oracle/fdtd_oracle.cpp — `d / ik`, the integer-node table at a half node, kappa applied after psi is
added, a harmonic mean, rho indexed along the wrong axis — fails one of them.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from oracle import Oracle

from conftest import golden

NU = 0.4
N, LK = 24, 5            # K1/K2 grid: 24 nodes per axis, 5-cell layers on all six faces
MID = 12


def _c32():
    return np.array([int(b, 16) for b in golden("coefficients.txt")["bits"]], np.uint32).view(np.float32).astype(np.float64)


def _kappa_tables():
    g = golden("kappa_stretch.txt")
    ki = [float(v) for v in g["kappa_int"]]        # from the wall inwards
    kh = [float(v) for v in g["kappa_half"]]
    k_int = np.ones(N)
    k_half = np.ones(N)
    for d in range(LK):
        k_int[d] = ki[d]                           # low face: integer node d has depth rho = (L - d)/L
        k_int[N - 1 - d] = ki[d]                   # high face: integer node N-1-d has depth rho = (L - d)/L
        k_half[d] = kh[d]                          # low face: half node d+1/2
        k_half[N - 2 - d] = kh[d]                  # high face: half node N-2-d+1/2 mirrors d+1/2
    return k_int, k_half


def _stretch_oracle(fp64=True):
    # R = 1 => sigma_max = 0 => a = 0 and psi stays 0; only the division by kappa is left
    return Oracle((N - 2 * LK,) * 3, (LK,) * 6, dt=NU, cpml_order=2, cpml_R0=1.0, cpml_kappa_max=5.0, cpml_alpha_max=0.0, fp64=fp64)


def _unit(axis, idx):
    """Index (k, j, i) of the node / half node `idx` along `axis`, centred on the other two axes."""
    ijk = [MID, MID, MID]
    ijk[axis] = idx
    return ijk[2], ijk[1], ijk[0]


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("s", [4, 20])
def test_k1_velocity_subupdate_divides_by_kappa_at_half_nodes(axis, s):
    """Unit p impulse at node s inside a layer: v_a[s-l] = -B c_l / kappa(s-l+1/2), v_a[s+l-1] = +B c_l / kappa(s+l-1/2)
    (P:40), kappa from the HALF-node profile; the pinned last half node (R3) stays 0."""
    c = _c32()
    k_int, k_half = _kappa_tables()
    B = float(np.float32(NU))
    o = _stretch_oracle()
    p0 = np.zeros((N,) * 3)
    p0[_unit(axis, s)] = 1.0
    o.set(oracle.P, p0)
    o.substep_v()
    expect = np.zeros((N,) * 3)
    for l in range(1, 5):
        for idx, sign in ((s - l, -1.0), (s + l - 1, +1.0)):
            if 0 <= idx < N - 1:                                   # idx = N-1 is the pinned half node
                expect[_unit(axis, idx)] = sign * B * c[l - 1] * float(np.float32(1.0 / k_half[idx]))
    got = o.get(oracle.VX + axis)
    assert np.abs(got - expect).max() <= 1e-15, np.abs(got - expect).max()
    # teeth: the integer-node profile, or multiplying instead of dividing, is off by tens of percent
    near = s - 1 if s < MID else s
    assert abs(1.0 / k_half[near] - 1.0 / k_int[near]) > 0.05 and abs(k_half[near] - 1.0 / k_half[near]) > 0.05
    # the other two velocity components see an interior point of their own axes: plain -+B c_l
    for b in range(3):
        if b == axis:
            continue
        vb = o.get(oracle.VX + b)
        ijk = [MID, MID, MID]
        ijk[axis] = s
        for l in range(1, 5):
            lo, hi = list(ijk), list(ijk)
            lo[b] = MID - l
            hi[b] = MID + l - 1
            assert abs(vb[lo[2], lo[1], lo[0]] + B * c[l - 1]) <= 1e-15
            assert abs(vb[hi[2], hi[1], hi[0]] - B * c[l - 1]) <= 1e-15
    for w in (oracle.PSI_VX, oracle.PSI_VY, oracle.PSI_VZ):
        assert not o.get(w).any()


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("i0", [3, 20])
def test_k2_pressure_subupdate_divides_by_kappa_at_integer_nodes(axis, i0):
    """Unit v_a impulse at half node i0+1/2: p[i0-l+1] = -Kc c_l / kappa(i0-l+1), p[i0+l] = +Kc c_l / kappa(i0+l)
    (P:40), kappa from the INTEGER-node profile."""
    c = _c32()
    k_int, k_half = _kappa_tables()
    Kc = float(np.float32(NU))
    o = _stretch_oracle()
    v0 = np.zeros((N,) * 3)
    v0[_unit(axis, i0)] = 1.0
    o.set(oracle.VX + axis, v0)
    o.substep_p()
    expect = np.zeros((N,) * 3)
    for l in range(1, 5):
        for idx, sign in ((i0 - l + 1, -1.0), (i0 + l, +1.0)):
            if 0 <= idx < N:
                expect[_unit(axis, idx)] = sign * Kc * c[l - 1] * float(np.float32(1.0 / k_int[idx]))
    got = o.get(oracle.P)
    assert np.abs(got - expect).max() <= 1e-15, np.abs(got - expect).max()
    assert abs(1.0 / k_half[i0] - 1.0 / k_int[i0]) > 0.05
    for w in (oracle.PSI_PX, oracle.PSI_PY, oracle.PSI_PZ):
        assert not o.get(w).any()


def test_k1_k2_fp32_instantiation_matches():
    """The fp32 instantiation (the parity reference, R18) gives the same values to fp32 rounding."""
    c = _c32()
    _, k_half = _kappa_tables()
    o = _stretch_oracle(fp64=False)
    p0 = np.zeros((N,) * 3)
    p0[_unit(0, 4)] = 1.0
    o.set(oracle.P, p0)
    o.substep_v()
    vx = o.get(oracle.VX)
    for l in range(1, 5):
        want = -float(np.float32(NU)) * c[l - 1] / k_half[4 - l]
        assert abs(vx[_unit(0, 4 - l)] - want) <= 3e-7 * abs(want)


# ---------------------------------------------------------------- T1 / K3: the paper's own parameter set
NP, L_LO, L_HI, DT_P = 64, 20, 12, 0.3


def _paper_oracle(fp64=True, axis=0):
    smax20 = -4.0 * math.log(1e-8) / (2 * 20)
    cp = [0] * 6
    cp[2 * axis], cp[2 * axis + 1] = L_LO, L_HI
    n_int = [16, 16, 16]
    n_int[axis] = NP - L_LO - L_HI
    return Oracle(tuple(n_int), tuple(cp), dt=DT_P, cpml_order=3, cpml_R0=1e-8, cpml_kappa_max=5.0,
                  cpml_alpha_max=0.05 * smax20, cpml_c_ref=1.0, fp64=fp64)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_t1_paper_set_tables_both_faces_both_staggerings(axis):
    g = golden("cpml_tables_paper_set.txt")
    o = _paper_oracle(axis=axis)
    tabs = {0: o.cpml_table(axis, 0), 1: o.cpml_table(axis, 1)}
    for key, row in g.items():
        if key.endswith("_layer"):
            continue
        idx, rho_txt, a_ref, b_ref, ik_ref = int(row[0]), row[1], float(row[2]), float(row[3]), float(row[4])
        half = 1 if "_half_" in key else 0
        a, b, ik, inn = tabs[half]
        assert inn[idx] == 1, key
        assert abs(a[idx] - a_ref) <= 2e-7 * max(abs(a_ref), 1e-3), (key, a[idx], a_ref)
        assert abs(b[idx] - b_ref) <= 1e-7, (key, b[idx], b_ref)
        assert abs(ik[idx] - ik_ref) <= 1e-7, (key, ik[idx], ik_ref)
        # the hand-written depth reproduces 1/kappa: kappa = 1 + 4 rho^3
        num, den = rho_txt.split("/")
        rho = float(Fraction(num)) / float(den)
        assert abs(1.0 / (1.0 + 4.0 * rho ** 3) - ik_ref) < 1e-11, key
    for half, key in ((0, "int_layer"), (1, "half_layer")):
        lo0, lo1, hi0, hi1 = (int(v) for v in g[key])
        inn = tabs[half][3]
        want = np.zeros(NP, np.uint8)
        want[lo0:lo1 + 1] = 1
        want[hi0:hi1 + 1] = 1
        assert np.array_equal(inn, want), key
        a, b, ik, _ = tabs[half]
        assert np.all(a[want == 0] == 0) and np.all(b[want == 0] == 1) and np.all(ik[want == 0] == 1)
    # the other two axes carry no layer at all
    for other in range(3):
        if other != axis:
            assert not o.cpml_table(other, 0)[3].any() and not o.cpml_table(other, 1)[3].any()


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_k3_stretch_and_memory_variable_combine_as_in_p46(axis):
    """One velocity sub-update from a unit p impulse with psi = 0 (paper set: sigma != 0 and kappa != 1):
    psi <- a d, then d/kappa + psi (update-then-use, R10), so v[s-1] = -B c_1 (1/kappa + a) with the half-node
    values of index 7 / 58 from the hand-worked table.  (d + psi)/kappa, or psi used before its refresh, differs at the
    1e-2 level."""
    g = golden("cpml_tables_paper_set.txt")
    c = _c32()
    B = float(np.float32(DT_P))
    for key, s in (("low_half_7", 8), ("high_half_58", 59)):
        a_ref, ik_ref = float(g[key][2]), float(g[key][4])
        o = _paper_oracle(axis=axis)
        shape = o.shape
        p0 = np.zeros(shape)
        ijk = [8, 8, 8]
        ijk[axis] = s
        p0[ijk[2], ijk[1], ijk[0]] = 1.0
        o.set(oracle.P, p0)
        o.substep_v()
        ijk[axis] = s - 1
        got = o.get(oracle.VX + axis)[ijk[2], ijk[1], ijk[0]]
        psi = o.get(oracle.PSI_VX + axis)[ijk[2], ijk[1], ijk[0]]
        d = c[0] * (1.0 - 0.0)
        assert abs(psi - a_ref * d) <= 3e-7 * abs(a_ref)
        want = -B * d * (ik_ref + a_ref)
        assert abs(got - want) <= 3e-7 * abs(want), (key, got, want)
        wrong_order = -B * d * (1.0 + a_ref) * ik_ref          # (d + psi)/kappa
        stale_psi = -B * d * ik_ref                            # psi used before its refresh
        assert abs(want - wrong_order) > 1e-2 * abs(want) and abs(want - stale_psi) > 1e-2 * abs(want)
        # second sub-update family: unit v impulse, p at the node next to it, integer-node values
    for key, i0 in (("low_int_7", 7), ("high_int_58", 58)):
        a_ref, ik_ref = float(g[key][2]), float(g[key][4])
        o = _paper_oracle(axis=axis)
        v0 = np.zeros(o.shape)
        ijk = [8, 8, 8]
        ijk[axis] = i0                                         # half node i0+1/2; node i0 gets -Kc c_1 (...)
        v0[ijk[2], ijk[1], ijk[0]] = 1.0
        o.set(oracle.VX + axis, v0)
        o.substep_p()
        got = o.get(oracle.P)[ijk[2], ijk[1], ijk[0]]
        want = -B * c[0] * (ik_ref + a_ref)
        assert abs(got - want) <= 3e-7 * abs(want), (key, got, want)


# ---------------------------------------------------------------- D1 / D2: heterogeneous medium (R6)
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_d1_rho_bar_is_the_arithmetic_mean_of_the_two_adjacent_nodes(axis):
    """rho = 1 on nodes <= 9 and 3 on nodes >= 10 along `axis`; unit p impulse at node 10.  The half node 9+1/2 lies
    between the two media: v[9] = -dt / (1/2 (1 + 3) dx) c_1 (P:36 'coefficients are absorbed', reading R6).  A harmonic
    (1.5) or geometric (1.73) mean, or rho taken from one node, is off by >= 13 %."""
    M = 20
    c = _c32()
    o = Oracle((M,) * 3, dt=NU, fp64=True)
    idx = np.arange(M)
    shape = [1, 1, 1]
    shape[2 - axis] = M
    rho = np.broadcast_to(np.where(idx >= 10, 3.0, 1.0).reshape(shape), (M,) * 3).astype(np.float32)
    o.set_model(None, rho)
    p0 = np.zeros((M,) * 3)
    ijk = [10, 10, 10]
    p0[10, 10, 10] = 1.0
    o.set(oracle.P, p0)
    o.substep_v()

    def at(field, a, i):
        q = [10, 10, 10]
        q[a] = i
        return o.get(field)[q[2], q[1], q[0]]

    f32 = lambda x: float(np.float32(x))
    assert abs(at(oracle.VX + axis, axis, 9) + f32(NU / 2.0) * c[0]) <= 1e-15          # between rho = 1 and rho = 3
    assert abs(at(oracle.VX + axis, axis, 10) - f32(NU / 3.0) * c[0]) <= 1e-15         # both nodes rho = 3
    assert abs(at(oracle.VX + axis, axis, 8) + f32(NU / 1.0) * c[1]) <= 1e-15          # both nodes rho = 1
    assert abs(at(oracle.VX + axis, axis, 11) - f32(NU / 3.0) * c[1]) <= 1e-15
    for b in range(3):                                                                  # transverse: node 10 has rho = 3
        if b != axis:
            assert abs(at(oracle.VX + b, b, 9) + f32(NU / 3.0) * c[0]) <= 1e-15
            assert abs(at(oracle.VX + b, b, 10) - f32(NU / 3.0) * c[0]) <= 1e-15
    assert abs(NU / 2.0 - NU / 1.5) > 0.13 * NU / 2.0


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_d2_pressure_coefficient_is_rho_c_squared_at_the_node(axis):
    """Unit v impulse at half node 9+1/2: p[9] = -K(9) dt/dx c_1, p[10] = +K(10) dt/dx c_1 with K = rho c^2 at the node."""
    M = 20
    c = _c32()
    o = Oracle((M,) * 3, dt=0.1, fp64=True)
    idx = np.arange(M)
    shape = [1, 1, 1]
    shape[2 - axis] = M
    rho = np.broadcast_to(np.where(idx >= 10, 3.0, 1.0).reshape(shape), (M,) * 3).astype(np.float32)
    spd = np.broadcast_to(np.where(idx >= 10, 2.0, 1.5).reshape(shape), (M,) * 3).astype(np.float32)
    o.set_model(spd, rho)
    v0 = np.zeros((M,) * 3)
    q = [10, 10, 10]
    q[axis] = 9
    v0[q[2], q[1], q[0]] = 1.0
    o.set(oracle.VX + axis, v0)
    o.substep_p()
    p = o.get(oracle.P)
    f32 = lambda x: float(np.float32(x))
    assert abs(p[q[2], q[1], q[0]] + f32(1.0 * 1.5 * 1.5 * 0.1) * c[0]) <= 1e-15
    q[axis] = 10
    assert abs(p[q[2], q[1], q[0]] - f32(3.0 * 2.0 * 2.0 * 0.1) * c[0]) <= 1e-15
