#!/usr/bin/env python
"""bench.py — throughput of the FDTD + CPML time step on B200, and the oracle beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3|config2|config4|config1]
  python bench.py --impl reference ...        # the CPU oracle, as it stands, on a bounded sample of the same workload

A "step" is one time step of the whole hot path (velocity sub-update, pressure sub-update, source; SURVEY 8a rows
a1-a5) over the whole grid.  metric = Mpoints/s = Nx Ny Nz steps / (1e6 T) counting interior + CPML cells
(PAPER.md P:228).  One process per GPU; N > 1 runs N independent replicas (the path does not shard: DESIGN.md
"Multi-GPU"), value = points of all ranks / max-over-ranks time.  Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Mpoints/s per time step (interior+CPML)"
UNIT = "Mpts/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3", choices=["config1", "config2", "config3", "config4"])
    ap.add_argument("--kernel", default="fused", choices=["fused", "two-pass"],
                    help="fused: one single-pass launch per step (FDTD_KERNEL_FUSED, 32 B/pt, twice the field memory; the default); "
                         "two-pass: update_v + update_p (48 B/pt)")
    ap.add_argument("--no-alt", action="store_true", help="do not also time the other kernel for the 'alt_kernel' entry")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpml-off", action="store_true", help="same total grid with plain walls (CPML overhead run, P:228)")
    return ap.parse_args()


def workload(name, steps):
    from paper_2606_06910_b200 import inputs

    w = inputs.config(int(name[-1]), steps=steps)
    return w


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def slab_points(w):
    """Points that carry a psi variable, per family: sum over axes of (cells in the two layers) x cross-section."""
    nx, ny, nz = w.total
    cp = w.cpml
    return (cp[0] + cp[1]) * ny * nz + (cp[2] + cp[3]) * nx * nz + (cp[4] + cp[5]) * nx * ny


def algorithmic_bytes(w):
    """bytes one launch of each kernel must move (fp32): (update_v, update_p, step_fused)."""
    n = w.points
    psi = 8 * slab_points(w)                              # read + write one psi per slab point per family
    kc = 4 if w.c is not None else 0
    bv = 28 * n + psi                                     # read p; read+write vx, vy, vz
    bp = (20 + kc) * n + psi                              # read vx, vy, vz (+Kc); read+write p
    bf = (32 + kc) * n + 2 * psi                          # read p, vx, vy, vz (+Kc); write p, vx, vy, vz; both psi families
    return bv, bp, bf


def ncu_traffic(wname):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture (profiles/*.csv)."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return {}
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, wl, b = line.strip().split(",")[:3]
            if wl == wname:
                out[k] = float(b)
    return out


def max_over_ranks(x, world, device):
    """Max of a per-rank scalar over all ranks (torch.distributed all_reduce MAX; nccl on cuda, gloo on cpu)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def throughput_mpts(points_per_rank, steps, world, seconds):
    """Whole-job Mpoints/s: points of all ranks x steps / (1e6 x max-over-ranks time)."""
    return points_per_rank * steps * world / seconds / 1e6


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return None
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return None
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(w, steps, window=256):
    """The oracle, as it stands, on a bounded sample: the low-corner window^3 sub-grid of the workload (CPML on its
    three outer faces, the heterogeneous c of that window), random state, `steps` time steps, all host cores, FTZ on."""
    import oracle
    from oracle import Oracle

    win = tuple(min(window, t) for t in w.total)
    cp = list(w.cpml)
    for a in range(3):
        if win[a] < w.total[a]:
            cp[2 * a + 1] = 0                     # cut face
    interior = tuple(win[a] - cp[2 * a] - cp[2 * a + 1] for a in range(3))
    o = Oracle(interior, cp, **w.cpml_kwargs())
    if w.c is not None:
        o.set_model(np.ascontiguousarray(w.c[:win[2], :win[1], :win[0]]))
    o.set_ftz(True)
    for f in range(4):
        o.fill_hash(f, 1234, gdim=w.total, scale=0.5)
    threads = oracle.max_threads()
    oracle.set_threads(threads)
    o.step(1)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    pts = win[0] * win[1] * win[2]
    return {"value": pts * steps / dt / 1e6, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": "%dx%dx%d low-corner window of %s (CPML on its 3 outer faces), %d steps, fp32, FTZ/DAZ on, OpenMP over z planes"
                      % (win[0], win[1], win[2], w.name, steps), "seconds": dt, "points_per_step": pts}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = workload(args.workload, max(args.steps, 1))
    # one step = one oracle time step on the bounded sample; sized so K + W steps end within minutes
    window = 160 if args.steps + args.warmup > 60 else 256
    import oracle
    from oracle import Oracle

    win = tuple(min(window, t) for t in w.total)
    cp = list(w.cpml)
    for a in range(3):
        if win[a] < w.total[a]:
            cp[2 * a + 1] = 0
    interior = tuple(win[a] - cp[2 * a] - cp[2 * a + 1] for a in range(3))
    o = Oracle(interior, cp, **w.cpml_kwargs())
    if w.c is not None:
        o.set_model(np.ascontiguousarray(w.c[:win[2], :win[1], :win[0]]))
    o.set_ftz(True)
    for f in range(4):
        o.fill_hash(f, 1234, gdim=w.total, scale=0.5)
    threads = oracle.max_threads()
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    pts = win[0] * win[1] * win[2]
    val = pts * args.steps / dt / 1e6
    sample = "%dx%dx%d low-corner window of %s per step, fp32 oracle, FTZ/DAZ on, %d OpenMP threads" % (win[0], win[1], win[2], w.name, threads)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "total_grid": list(w.total), "cpml": list(w.cpml), "sample_grid": list(win)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2606_06910_b200 import binding

    K, W = args.steps, max(args.warmup, 3)
    w = workload(args.workload, 2 * K + W)
    if args.cpml_off:
        w.n_interior, w.cpml = w.total, (0,) * 6

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fused = args.kernel == "fused"
    kern = binding.FDTD_KERNEL_FUSED if fused else binding.FDTD_KERNEL_AUTO

    def timed_run(kernel, sample_clocks):
        """W warm-up steps, then K steps between two CUDA events (barrier + synchronize on both sides), then the same
        K steps again with an event after every launch group for the per-kernel split."""
        sim = binding.from_workload(w, device=local, kernel=kernel)
        for f in range(1, 4):                   # non-trivial state everywhere (values do not change the traffic)
            sim.fill_hash(f, 99, 1e-3)
        sim.step(W)
        barrier()
        sampler = ClockSampler(local) if (rank == 0 and sample_clocks) else None
        l0 = sim.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        sim.step(K)
        e1.record()
        barrier()
        t = e0.elapsed_time(e1)
        n_launch = sim.launch_count() - l0
        split = sim.step_profiled(K)
        clk = sampler.stop() if sampler else None
        t = max_over_ranks(t, world, "cuda")
        sim.destroy()
        del sim
        torch.cuda.empty_cache()
        return t, n_launch, split, clk

    ms, launches, prof, clocks = timed_run(kern, True)
    alt = None
    if not args.no_alt and w.total[0] % 4 == 0:
        other = binding.FDTD_KERNEL_AUTO if fused else binding.FDTD_KERNEL_FUSED
        a_ms, _, a_prof, _ = timed_run(other, False)
        alt = {"kernel": "two-pass" if fused else "fused", "value": throughput_mpts(w.points, K, world, a_ms * 1e-3), "unit": UNIT,
               "ms_per_step": a_ms / K, "kernels_ms_per_step": {("step_fused" if (k == "update_v" and not fused) else k): v / K for k, v in a_prof.items() if v > 0}}

    # ---- end to end through the C ABI with host buffers: model up, K steps, pressure field down
    e2e = None
    if not args.no_e2e:
        n = w.points
        c_host = None
        if w.c is not None:
            c_host = torch.from_numpy(w.c).pin_memory()
        out_host = torch.empty(n, dtype=torch.float32).pin_memory()
        sim = binding.Fdtd(w.n_interior, w.cpml, device=local, kernel=kern, **w.cpml_kwargs())
        barrier()
        t0 = time.perf_counter()
        if c_host is not None:
            sim.set_model_from(c_host.data_ptr())
        sim.set_sources(w.sources, w.wavelets)
        sim.step(K)
        sim.get_field_into(binding.FDTD_P, out_host.data_ptr())
        torch.cuda.synchronize()
        dt_e = time.perf_counter() - t0
        dt_e = max_over_ranks(dt_e, world, "cuda")
        h2d = (n * 4 if c_host is not None else 0) + w.sources.nbytes + w.wavelets.nbytes
        e2e = {"value": throughput_mpts(n, K, world, dt_e), "unit": UNIT, "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": n * 4 / K,
               "seconds": dt_e, "what": "fdtd_set_model + fdtd_set_sources + fdtd_step(K) + fdtd_get_field(p), pinned host buffers"}
        sim.destroy()
        del sim

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    value = throughput_mpts(w.points, K, world, ms * 1e-3)
    bv, bp, bf = algorithmic_bytes(w)
    peak, peak_src = peaks()
    if fused:
        dom, dur, byt, step_bytes = "step_fused", prof["update_v"] / K * 1e-3, bf, bf
        prof = {"step_fused": prof["update_v"], "inject": prof["inject"], "exchange": prof["exchange"]}
    else:
        dom = "update_v_tiled" if prof["update_v"] >= prof["update_p"] else "update_p_tiled"
        dur = (prof["update_v"] if dom == "update_v_tiled" else prof["update_p"]) / K * 1e-3
        byt, step_bytes = (bv if dom == "update_v_tiled" else bp), bv + bp
    traffic = ncu_traffic(w.name)
    step_gbps = step_bytes / (ms * 1e-3 / K) / 1e9
    roof = {"bound": "hbm", "kernel": dom, "achieved": byt / dur / 1e9, "peak": peak, "unit": "GB/s",
            "frac": byt / dur / 1e9 / peak, "peak_source": peak_src, "traffic": traffic.get(dom),
            "algorithmic_bytes_per_launch": byt, "avg_launch_ms": dur * 1e3,
            "step": {"bytes": step_bytes, "model": "single pass, 32 B/pt + Kc + psi" if fused else "two passes, 48 B/pt + Kc + psi",
                     "GBps": step_gbps, "frac": step_gbps / peak, "frac_of_8000": step_gbps / 8000.0,
                     "two_pass_equivalent_GBps": (bv + bp) / (ms * 1e-3 / K) / 1e9},
            "kernels_ms_per_step": {k: v / K for k, v in prof.items()}}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name + ("-cpml-off" if args.cpml_off else ""), "total_grid": list(w.total), "cpml": list(w.cpml),
                   "medium": "heterogeneous c (Kc array)" if w.c is not None else "homogeneous", "sources": int(w.sources.shape[0]),
                   "kernel": args.kernel, "parallelism": "replicas x%d" % world, "l2": "inputs larger than L2 (fields %.1f GB)" % (w.points * 16 / 1e9)},
        "roofline": roof, "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e, "alt_kernel": alt,
    }
    if alt is not None:
        ab = (bv + bp) if fused else bf                # algorithmic bytes of the other kernel structure
        alt["step_frac_of_peak"] = ab / (alt["ms_per_step"] * 1e-3) / 1e9 / peak
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = oracle_sample(w, 24)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
