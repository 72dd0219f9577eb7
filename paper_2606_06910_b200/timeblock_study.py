"""k-step temporal blocking inside one GPU: the sweep of k (the single-device analogue of the paper's
sweep of the enlarged ghost s in Table 12, where s = 8 loses to s = 4 because of redundant work).

  python -m paper_2606_06910_b200.timeblock_study [--workload 2] [--steps 48]

For k in {1, 2, 4} (and several slab thicknesses) times the single-pass step in its time-blocked mode — k steps per pass
over z slabs, 8 planes of ghost recomputed per remaining step on both sides of a slab — and prints ms per time step,
Mpoints/s, and the redundant compute (plane-steps computed / plane-steps owned) as counted by the library.  One JSON
object per line.  Every result has the bits of the k = 1 run (tests/test_timeblock_gpu.py)."""
import argparse
import json

import torch

from . import binding, inputs


def run(w, steps, **kw):
    sim = binding.from_workload(w, kernel=binding.FDTD_KERNEL_FUSED, **kw)
    for f in range(4):
        sim.fill_hash(f, 99, 1e-3)
    sim.step(8)
    torch.cuda.synchronize()
    l0 = sim.launch_count()
    c0 = sim.time_block_stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sim.step(steps)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    c1 = sim.time_block_stats()
    launches = sim.launch_count() - l0
    sim.destroy()
    red = (c1[0] - c0[0]) / (c1[1] - c0[1]) if c1[1] > c0[1] else 1.0
    return ms, red, launches / steps


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", type=int, default=2, choices=[2, 3])
    ap.add_argument("--steps", type=int, default=48)
    a = ap.parse_args()
    w = inputs.config(a.workload, steps=a.steps + 16)
    pts = w.points
    ms1, _, l1 = run(w, a.steps)
    print(json.dumps({"workload": w.name, "k": 1, "ms_per_step": ms1, "Mpts_s": pts / ms1 / 1e3, "planes_computed_per_owned": 1.0,
                      "launches_per_step": l1}))
    for k in (2, 4):
        for planes in (0, 16, 32, 64, 128):
            if planes > w.total[2]:
                continue
            ms, red, lps = run(w, a.steps, time_block=k, time_block_planes=planes)
            print(json.dumps({"workload": w.name, "k": k, "slab_planes": planes or "auto (L2-sized)", "ms_per_step": ms, "Mpts_s": pts / ms / 1e3,
                              "vs_k1": ms1 / ms, "planes_computed_per_owned": red, "launches_per_step": lps}))


if __name__ == "__main__":
    main()
