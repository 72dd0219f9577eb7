"""Power, clocks and sustained rate of the time step against plain copies on the same GPU.

  python -m paper_2606_06910_b200.power_study [--seconds 5] [--workloads 4,3]

The bench loop of `bench.py` runs for seconds, long enough for the board's power cap to set the SM clock.  This prints,
for a device-to-device copy, an in-place add, a fill, and for both step structures of each workload (from the
counter-based random state that `bench.py` times and from all-zero fields), the sustained rate together with the median
power draw and SM clock that `nvidia-smi` reports while the loop runs.  One JSON object per line."""
import argparse
import json
import subprocess
import tempfile
import time

import numpy as np
import torch

from . import binding, inputs


def sample(fn, label, secs, sync_every=4):
    f = tempfile.NamedTemporaryFile("w+", suffix=".csv")
    p = subprocess.Popen(["nvidia-smi", "-i", str(torch.cuda.current_device()), "--query-gpu=power.draw,clocks.sm,clocks.mem,temperature.gpu",
                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=f)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0, n = time.time(), 0
    e0.record()
    while time.time() - t0 < secs:
        fn()
        n += 1
        if n % sync_every == 0:
            torch.cuda.synchronize()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n
    p.terminate()
    p.wait()
    f.flush()
    f.seek(0)
    rows = [[float(x) for x in line.split(",")] for line in f if line.count(",") == 3]
    a = np.array(rows[len(rows) // 3:])            # the first third is the ramp to the cap
    out = {"what": label, "ms_per_call": ms, "calls": n}
    if a.size:
        out.update({"power_W": float(np.median(a[:, 0])), "sm_mhz": float(np.median(a[:, 1])), "mem_mhz": float(np.median(a[:, 2])),
                    "temp_C": float(np.median(a[:, 3]))})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--seconds", type=float, default=5.0)
    ap.add_argument("--workloads", default="4,3")
    a = ap.parse_args()
    x = torch.empty(2 * 1024 ** 3, dtype=torch.float32, device="cuda")
    y = torch.empty_like(x)
    nbytes = x.numel() * 4
    for label, fn, moved in (("copy 8 GiB", lambda: y.copy_(x), 2 * nbytes), ("in-place add 8 GiB", lambda: x.add_(1.0), 2 * nbytes),
                             ("fill 8 GiB", lambda: x.zero_(), nbytes)):
        r = sample(fn, label, a.seconds)
        r["GB_s"] = moved / r["ms_per_call"] / 1e6
        print(json.dumps(r), flush=True)
    del x, y
    torch.cuda.empty_cache()
    for c in [int(t) for t in a.workloads.split(",")]:
        w = inputs.config(c, steps=100000)
        k = max(1, int(100.0 / (w.points / 1.3e8)))      # about 100 ms of steps per call
        for kern, kname in ((binding.FDTD_KERNEL_FUSED, "single-pass step"), (binding.FDTD_KERNEL_AUTO, "two-kernel step")):
            sim = binding.from_workload(w, kernel=kern)
            for scale, sname in ((1e-3, "counter-based random state"), (0.0, "zero fields")):
                for f in range(4):
                    sim.fill_hash(f, 99, scale)
                r = sample(lambda: sim.step(k), "%s, %s, %s" % (w.name, kname, sname), a.seconds)
                r["ms_per_step"] = r.pop("ms_per_call") / k
                r["Mpts_s"] = w.points / r["ms_per_step"] / 1e3
                print(json.dumps(r), flush=True)
            sim.destroy()
            del sim
            torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
