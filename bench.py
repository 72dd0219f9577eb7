#!/usr/bin/env python
"""bench.py — throughput of the FDTD + CPML time step on B200, and the oracle beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config4|config3|config2|config1]
  python bench.py --impl reference ...        # the CPU oracle, as it stands, on a bounded sample of the same workload

A "step" is one time step of the whole hot path (velocity sub-update, pressure sub-update, source; SURVEY 8a rows
a1-a5) over the whole grid.  metric = Mpoints/s = Nx Ny Nz steps / (1e6 T) counting interior + CPML cells
(PAPER.md P:228).  The default workload is BASELINE config 4 (1600^3 total), the largest single-GPU configuration;
configs 3 and 2 are timed in the same run and carried under "other_workloads".  The timed region of K steps is repeated
5 times (CUDA events, barrier + synchronize on both sides); value / ms_per_step are the median repeat (the paper
reports medians), min and max are printed beside it.  One process per GPU; N > 1 runs N independent
replicas (the path does not shard: DESIGN.md "Multi-GPU"), value = points of all ranks / max-over-ranks time.
Every workload is timed from a counter-based random state (random mantissas draw the most power, and the loop runs at the
board's power cap); the config's own initial state (zero fields + its sources) is timed beside it as "state_zero_fields".
Prints ONE JSON line on rank 0.
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
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--repeats", type=int, default=5, help="timed regions of K steps; the median is reported")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4", choices=["config1", "config2", "config3", "config4"])
    ap.add_argument("--no-others", action="store_true", help="do not also time the other BASELINE workloads and the CPML-off runs")
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
    """dram__bytes_read.sum + dram__bytes_write.sum per launch as recorded by a committed `ncu --set full` capture
    (profiles/dram_traffic.csv: kernel, workload, bytes, source file).  Not measured by this run: -> {kernel: (bytes, source)}."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return {}
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, wl, b, src = (line.strip().split(",") + [""])[:4]
            if wl == wname:
                out[k] = (float(b), src)
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
                                       "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
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

    K, W, R = args.steps, max(args.warmup, 3), max(args.repeats, 1)
    total_steps = W + (R + 1) * K + 8
    peak, peak_src = peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fused = args.kernel == "fused"
    kern = binding.FDTD_KERNEL_FUSED if fused else binding.FDTD_KERNEL_AUTO
    kname = {binding.FDTD_KERNEL_FUSED: "fused", binding.FDTD_KERNEL_AUTO: "two-pass"}

    def timed_run(w, kernel, sample_clocks=False, scale=1e-3):
        """W warm-up steps, then R regions of K steps, each between two CUDA events with barrier + synchronize on both sides;
        then K more steps with an event after every launch group (the per-kernel split; it carries event overhead)."""
        sim = binding.from_workload(w, device=local, kernel=kernel)
        for f in range(4):                      # non-trivial state everywhere: the values decide the power drawn, not the traffic
            sim.fill_hash(f, 99, scale)         # (scale 0: the config's own initial state, zero fields + its sources)
        sampler = ClockSampler(local) if (rank == 0 and sample_clocks) else None      # started before the warm-up
        sim.step(W)
        times, n_launch = [], 0
        for _ in range(R):
            barrier()
            l0 = sim.launch_count()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sim.step(K)
            e1.record()
            barrier()
            times.append(max_over_ranks(e0.elapsed_time(e1), world, "cuda"))
            n_launch = sim.launch_count() - l0
        clk = sampler.stop() if sampler else None
        split = sim.step_profiled(K)
        sim.destroy()
        del sim
        torch.cuda.empty_cache()
        ms = float(np.median(times))
        return {"ms": ms, "times": times, "launches": n_launch, "split": split, "clocks": clk}

    def summarise(w, run, kernel):
        """value, ms/step and the roofline of the step structure that ran, from the median back-to-back region."""
        bv, bp, bf = algorithmic_bytes(w)
        is_f = kernel == binding.FDTD_KERNEL_FUSED
        step_bytes = bf if is_f else bv + bp
        ms_step = run["ms"] / K
        gbps = step_bytes / (ms_step * 1e-3) / 1e9
        return {"kernel": kname[kernel], "value": throughput_mpts(w.points, K, world, run["ms"] * 1e-3), "unit": UNIT, "ms_per_step": ms_step,
                "ms_per_step_min": min(run["times"]) / K, "ms_per_step_max": max(run["times"]) / K,
                "step_bytes": step_bytes, "step_GBps": gbps, "step_frac_of_peak": gbps / peak, "step_frac_of_8000": gbps / 8000.0}

    def cpml_off(w):
        import copy
        o = copy.copy(w)
        o.n_interior, o.cpml = w.total, (0,) * 6
        return o

    w = workload(args.workload, total_steps)
    if args.cpml_off:
        w = cpml_off(w)
    main_run = timed_run(w, kern, sample_clocks=True)
    ms, launches, prof, clocks = main_run["ms"], main_run["launches"], main_run["split"], main_run["clocks"]

    # the same workload from the state BASELINE gives it (fields initialised to zero, the Ricker source running): the board sits
    # at its power cap in both runs, and all-zero buses draw less than random mantissas, so the clock is higher
    zero_state = None
    if not args.no_others and world == 1:
        z_run = timed_run(w, kern, sample_clocks=True, scale=0.0)
        zero_state = {"value": throughput_mpts(w.points, K, world, z_run["ms"] * 1e-3), "unit": UNIT, "ms_per_step": z_run["ms"] / K,
                      "clocks": z_run["clocks"], "state": "zero fields + the config's sources (BASELINE's initial state)"}

    alt = None
    if not args.no_alt and w.total[0] % 4 == 0:
        other = binding.FDTD_KERNEL_AUTO if fused else binding.FDTD_KERNEL_FUSED
        a_run = timed_run(w, other)
        alt = summarise(w, a_run, other)
        alt["kernels_ms_per_step_profiled"] = {("step_fused" if (k == "update_v" and not fused) else k): v / K for k, v in a_run["split"].items() if v > 0}

    # CPML overhead of the headline workload (R23: same total grid, plain walls), same kernel
    overhead = None
    if not args.no_others and not args.cpml_off and world == 1:
        o_run = timed_run(cpml_off(w), kern)
        overhead = {"cpml_off_ms_per_step": o_run["ms"] / K, "cpml_off_value": throughput_mpts(w.points, K, world, o_run["ms"] * 1e-3),
                    "overhead": ms / o_run["ms"] - 1.0, "psi_byte_floor": 16.0 * slab_points(w) / ((32 if fused else 48) * w.points + (4 * w.points if w.c is not None else 0))}

    # ---- end to end through the C ABI with host buffers: the same state as the timed leg (counter-based fill, set up
    # before the clock starts), then inside the timed region: model up from pinned host memory, sources up, K steps,
    # pressure field down into pinned host memory.
    e2e = None
    if not args.no_e2e:
        n = w.points
        c_host = torch.tensor(w.c).pin_memory() if w.c is not None else None
        out_host = torch.empty(n, dtype=torch.float32).pin_memory()
        sim = binding.Fdtd(w.n_interior, w.cpml, device=local, kernel=kern,
                           medium=binding.FDTD_MEDIUM_ARRAY if w.c is not None else binding.FDTD_MEDIUM_UNIFORM, **w.cpml_kwargs())
        for f in range(4):
            sim.fill_hash(f, 99, 1e-3)
        sim.step(W)                              # warm: the same clocks and power state as the timed leg
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        if c_host is not None:
            sim.set_model_from(c_host.data_ptr())
        sim.set_sources(w.sources, w.wavelets)
        e0.record()
        sim.step(K)
        e1.record()
        sim.get_field_into(binding.FDTD_P, out_host.data_ptr())
        torch.cuda.synchronize()
        dt_e = time.perf_counter() - t0
        step_s = e0.elapsed_time(e1) * 1e-3
        dt_e = max_over_ranks(dt_e, world, "cuda")
        h2d = (n * 4 if c_host is not None else 0) + w.sources.nbytes + w.wavelets.nbytes
        e2e = {"value": throughput_mpts(n, K, world, dt_e), "unit": UNIT, "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": n * 4 / K,
               "seconds": dt_e, "step_seconds": step_s, "copy_seconds": dt_e - step_s,
               "d2h_GBps": n * 4 / max(dt_e - step_s, 1e-9) / 1e9 if c_host is None else None,
               "what": "fdtd_set_model + fdtd_set_sources + fdtd_step(K) + fdtd_get_field(p) on the warmed, hash-filled state of the timed leg; "
                       "pinned host buffers; copy_seconds = seconds - step_seconds (CUDA events around the K steps)"}
        sim.destroy()
        del sim, out_host, c_host
        torch.cuda.empty_cache()

    # ---- the other BASELINE workloads in the same run (parity-test configurations, reported for context): both step
    # structures, and the CPML-off run of R23 for the overhead BASELINE config 2 asks for
    others = None
    if not args.no_others and not args.cpml_off and world == 1:
        others = {}
        for name in ("config3", "config2"):
            if name == args.workload:
                continue
            ow = workload(name, total_steps)
            r_on = timed_run(ow, kern)
            r_off = timed_run(cpml_off(ow), kern)
            r_alt = timed_run(ow, binding.FDTD_KERNEL_AUTO if fused else binding.FDTD_KERNEL_FUSED)
            ent = summarise(ow, r_on, kern)
            ent["total_grid"] = list(ow.total)
            ent["cpml_off_ms_per_step"] = r_off["ms"] / K
            ent["cpml_overhead"] = r_on["ms"] / r_off["ms"] - 1.0
            ent["psi_byte_floor"] = 16.0 * slab_points(ow) / ((32 if fused else 48) * ow.points + (4 * ow.points if ow.c is not None else 0))
            ent["alt_kernel"] = summarise(ow, r_alt, binding.FDTD_KERNEL_AUTO if fused else binding.FDTD_KERNEL_FUSED)
            others[name] = ent

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    head = summarise(w, main_run, kern)
    bv, bp, bf = algorithmic_bytes(w)
    tot_prof = sum(prof.values())
    if fused:
        dom, byt, share = "step_fused", bf, prof["update_v"] / tot_prof
        prof = {"step_fused": prof["update_v"], "inject": prof["inject"], "exchange": prof["exchange"]}
    else:
        dom = "update_v_tiled" if prof["update_v"] >= prof["update_p"] else "update_p_tiled"
        share = (prof["update_v"] if dom == "update_v_tiled" else prof["update_p"]) / tot_prof
        byt = bv if dom == "update_v_tiled" else bp
    dur = head["ms_per_step"] * 1e-3 * share             # the kernel's share of the back-to-back step time
    traffic = ncu_traffic(w.name).get(dom)
    roof = {"bound": "hbm", "kernel": dom, "achieved": byt / dur / 1e9, "peak": peak, "unit": "GB/s",
            "frac": byt / dur / 1e9 / peak, "frac_of_8000": byt / dur / 1e9 / 8000.0, "peak_source": peak_src,
            "traffic": traffic[0] if traffic else None,
            "traffic_source": ("committed ncu --set full capture, not this run: profiles/" + traffic[1]) if traffic else None,
            "algorithmic_bytes_per_launch": byt, "avg_launch_ms": dur * 1e3,
            "avg_launch_ms_source": "median back-to-back ms_per_step x the kernel's share of the event-profiled split",
            "kernel_share_of_step": share,
            "step": {"bytes": head["step_bytes"], "model": "single pass, 32 B/pt + Kc + psi" if fused else "two passes, 48 B/pt + Kc + psi",
                     "GBps": head["step_GBps"], "frac": head["step_frac_of_peak"], "frac_of_8000": head["step_frac_of_8000"],
                     "two_pass_equivalent_GBps": (bv + bp) / (head["ms_per_step"] * 1e-3) / 1e9},
            "kernels_ms_per_step_profiled": {k: v / K for k, v in prof.items()},
            "profiled_note": "one CUDA event after every launch: about 2 % slower than back to back"}
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": head["ms_per_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name + ("-cpml-off" if args.cpml_off else ""), "total_grid": list(w.total), "cpml": list(w.cpml),
                   "medium": "heterogeneous c (Kc array)" if w.c is not None else "homogeneous", "sources": int(w.sources.shape[0]),
                   "kernel": args.kernel, "parallelism": "replicas x%d" % world, "l2": "inputs larger than L2 (fields %.1f GB)" % (w.points * 16 / 1e9),
                   "state": "counter-based random fields (scale 1e-3) + the config's sources"},
        "repeats": {"n": R, "statistic": "median", "ms_per_step": [t / K for t in main_run["times"]],
                    "min": head["ms_per_step_min"], "max": head["ms_per_step_max"]},
        "roofline": roof, "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e, "alt_kernel": alt, "state_zero_fields": zero_state, "cpml": overhead,
        "other_workloads": others,
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = oracle_sample(w, 300)        # about 12 s on 16 cores
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
