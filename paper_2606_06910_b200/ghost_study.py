"""Ghost-width cost on one device (BASELINE config 5; the single-GPU analogue of the paper's Table 12).

  python -m paper_2606_06910_b200.ghost_study [--steps 100] [--scale 512] [--layouts] [--fused]

Splits the 512^3 + 20-cell-CPML grid into 1x2x2 in-HBM subdomains with ghost width g and m sub-updates between halo
exchanges (g >= 4 m; (8,2) is the paper's s = 1, (16,4) its s = 2, (32,8) its s = 4), times it against the monolithic
kernel and reports the redundant ghost compute (points updated / points owned) and the exchange share.  Prints one
JSON object per line.  --layouts runs the three four-subdomain layouts of the paper's Table 5 at
(g, m) = (8, 2) — slab-z 1x1x4, block-xy 2x2x1 (its halo cuts the contiguous x axis: g-wide column blocks), pencil-yz
1x2x2 — plus slab-y 1x4x1 and 1x4x2, with the halo-exchange time split out, so that the ordering of Table 5 can be
compared by halo cost.  --fused runs the subdomains with the single-pass step (two sub-updates per launch, so m is even)."""
import argparse
import json

import torch

from . import binding, inputs


def run(w, steps, **kw):
    sim = binding.from_workload(w, **kw)
    sim.step(10)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sim.step(steps)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    prof = sim.step_profiled(steps)
    sim.destroy()
    return ms, {k: v / steps for k, v in prof.items()}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--scale", type=int, default=512)
    ap.add_argument("--layouts", action="store_true")
    ap.add_argument("--fused", action="store_true")
    a = ap.parse_args()
    kern = binding.FDTD_KERNEL_FUSED if a.fused else binding.FDTD_KERNEL_AUTO
    w = inputs.config(5, scale=a.scale, steps=2 * a.steps + 10)
    pts = w.points
    ms0, prof0 = run(w, a.steps, decomp=(1, 1, 1), ghost=0, substeps=0, kernel=kern)
    print(json.dumps({"layout": "monolithic", "kernel": "fused" if a.fused else "two-pass", "ms_per_step": ms0, "Mpts_s": pts / ms0 / 1e3,
                      "kernels_ms": prof0}))
    own = w.total[1] // 2
    if a.layouts:
        for name, dec in (("slab-z 1x1x4", (1, 1, 4)), ("block-xy 2x2x1", (2, 2, 1)), ("pencil-yz 1x2x2", (1, 2, 2)), ("slab-y 1x4x1", (1, 4, 1)),
                          ("1x4x2", (1, 4, 2))):
            g, m = 8, 2
            ms, prof = run(w, a.steps, decomp=dec, ghost=g, substeps=m, kernel=kern)
            upd = 1.0                       # points updated / points owned: edge subdomains carry one ghost side, inner ones two
            for ax in (0, 1, 2):
                d, o = dec[ax], w.total[ax] // dec[ax]
                if d > 1:
                    upd *= (2 * (o + g) + (d - 2) * (o + 2 * g)) / (o * d)
            print(json.dumps({"layout": name, "ghost": g, "substeps_per_exchange": m, "ms_per_step": ms, "Mpts_s": pts / ms / 1e3,
                              "vs_monolithic": ms0 / ms, "points_updated_per_owned": upd, "exchange_ms": prof["exchange"],
                              "exchange_share": prof["exchange"] / sum(prof.values()), "kernels_ms": prof}))
        return
    for g, m in ((4, 1), (8, 2), (16, 4), (32, 8), (16, 2), (32, 4)):
        if a.fused and m % 2:
            continue
        ms, prof = run(w, a.steps, decomp=(1, 2, 2), ghost=g, substeps=m, kernel=kern)
        print(json.dumps({"layout": "pencil-yz 1x2x2", "ghost": g, "substeps_per_exchange": m, "ms_per_step": ms,
                          "Mpts_s": pts / ms / 1e3, "vs_monolithic": ms0 / ms, "points_updated_per_owned": ((own + g) / own) ** 2,
                          "kernels_ms": prof}))


if __name__ == "__main__":
    main()
