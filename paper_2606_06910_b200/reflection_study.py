"""CPML reflection against layer thickness with the paper's own parameter set (Table 8).

  python -m paper_2606_06910_b200.reflection_study [--interior 96] [--steps 320] [--baseline-set] [--kappa-max 5]
                                                   [--f0 0.04] [--courant 0.4]

The paper prints reflected-to-incident ratios 9.4e-1, 8.0e-2, 6.7e-3, 5.6e-4, 3.3e-5 for 0 / 8 / 12 / 16 / 24 cells but
not the procedure, so only the trend is comparable.  Procedure used here:
  * test run: interior^3 cells + an L-cell CPML on all six faces, Ricker source (f0 = 0.04, 25 cells per wavelength) at
    the centre, Courant 0.4, paper set q = 3, R = 1e-8, kappa_max = 5, alpha_max = 0.05 sigma_max (Table 2);
  * reference run: the same source in a wall-bounded box so large that nothing returns to the compared region within
    the run (reach 8 cells per step is the numerical bound, the wave itself travels 0.4 cells per step);
  * ratio = max over the sampled steps of max |p_test - p_ref| over the test run's interior, divided by the largest
    |p_ref| any interior cell within 4 cells of a face sees during the run (the incident amplitude at the layer).
Prints one JSON object per thickness.  Every field value comes from the CUDA path (fdtd_step through the C ABI)."""
import argparse
import json
import math

import numpy as np

from . import binding, inputs


def run(interior, L, steps, sample_from, every, pad, cpml_kw, kernel, dt=inputs.COURANT, f0=inputs.F0):
    """-> list of interior snapshots (numpy, interior^3) at the sampled steps; pad = extra wall-bounded cells per side."""
    n = interior + 2 * pad
    sim = binding.Fdtd((n,) * 3, (L,) * 6, dt=dt, kernel=kernel, **cpml_kw)
    c = n // 2 + L
    sim.set_sources([(c, c, c)], inputs.ricker(steps, dt, f0=f0)[None, :])
    lo = (L + pad,) * 3
    out, done = [], 0
    for s in range(sample_from, steps + 1, every):
        sim.step(s - done)
        done = s
        out.append(sim.get_field_box(binding.FDTD_P, lo, (interior,) * 3))
    sim.destroy()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--interior", type=int, default=96)
    ap.add_argument("--steps", type=int, default=320)
    ap.add_argument("--baseline-set", action="store_true", help="BASELINE.json's set (q = 2, R0 = 1e-5, kappa = 1, alpha = pi f0) instead of the paper's")
    ap.add_argument("--kappa-max", type=float, default=5.0, help="kappa_max of the paper set (P:124 uses 5)")
    ap.add_argument("--kernel", type=int, default=binding.FDTD_KERNEL_AUTO)
    ap.add_argument("--f0", type=float, default=inputs.F0, help="Ricker peak frequency: cells per wavelength = 1 / f0 at c = dx = 1")
    ap.add_argument("--courant", type=float, default=inputs.COURANT, help="c dt / dx (P:112 names a scaling parameter 0.05; R15)")
    a = ap.parse_args()
    every = max(20, a.steps // 16)
    first = every
    # reference: walls far enough that their echo cannot reach the compared region: it would have to travel 2 * pad cells
    pad = int(math.ceil(a.steps * a.courant * 1.3 / 2.0 / 4.0)) * 4 + 16
    ref = run(a.interior, 0, a.steps, first, every, pad, dict(), a.kernel, a.courant, a.f0)
    m = a.interior
    shell = np.ones((m, m, m), bool)
    shell[4:-4, 4:-4, 4:-4] = False
    incident = max(float(np.abs(r[shell]).max()) for r in ref)
    for L in (0, 8, 12, 16, 20, 24):
        if a.baseline_set:
            kw = dict(cpml_order=2, cpml_R0=1e-5, cpml_kappa_max=1.0, cpml_alpha_max=math.pi * a.f0)
            name = "BASELINE set (q=2, R0=1e-5, kappa_max=1, alpha_max=pi f0)"
        else:
            smax = -4.0 * math.log(1e-8) / (2.0 * max(L, 1) * 1.0)
            kw = dict(cpml_order=3, cpml_R0=1e-8, cpml_kappa_max=a.kappa_max, cpml_alpha_max=0.05 * smax)
            name = "paper set (q=3, R=1e-8, kappa_max=%g, alpha_max=0.05 sigma_max)" % a.kappa_max
        test = run(a.interior, L, a.steps, first, every, 0, kw if L else dict(), a.kernel, a.courant, a.f0)
        err = max(float(np.abs(t - r).max()) for t, r in zip(test, ref))
        print(json.dumps({"cpml_cells": L, "parameters": name, "reflected_over_incident": err / incident, "incident_amplitude": incident,
                          "interior": a.interior, "steps": a.steps, "reference_box": a.interior + 2 * pad, "f0": a.f0, "courant": a.courant}))


if __name__ == "__main__":
    main()
