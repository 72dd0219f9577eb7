"""Host logic of bench.py (no GPU): byte models, the N > 1 aggregation over world_size-2 gloo, the reference arm."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from conftest import ROOT

sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_2606_06910_b200 import inputs  # noqa: E402


def test_byte_models_match_survey_8d():
    # two-pass model 48 B/pt + psi 16 B per slab point per axis (+4 for a Kc array): SURVEY 8d / BASELINE.md table
    for idx, expect in ((2, 53.33), (4, 49.92)):
        w = inputs.config(idx, steps=1)
        bv, bp, bf = bench.algorithmic_bytes(w)
        assert abs((bv + bp) / w.points - expect) < 0.01
        assert abs(bf / w.points - (expect - 16.0)) < 0.01        # single pass: 32 instead of 48 B/pt, same psi bytes
    w = inputs.config(1, steps=1)
    bv, bp, bf = bench.algorithmic_bytes(w)
    assert bv == 28 * 80 ** 3 + 8 * 3 * 16 * 80 * 80 and bp == 20 * 80 ** 3 + 8 * 3 * 16 * 80 * 80
    assert bf == 32 * 80 ** 3 + 16 * 3 * 16 * 80 * 80
    w.c = 1                                  # a Kc array adds 4 B/pt to update_p and to the fused step
    assert bench.algorithmic_bytes(w)[1] == bp + 4 * 80 ** 3 and bench.algorithmic_bytes(w)[2] == bf + 4 * 80 ** 3
    assert bench.throughput_mpts(1000, 10, 2, 0.5) == pytest.approx(1000 * 10 * 2 / 0.5 / 1e6)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank                    # rank 1 is the slow one
    dist.barrier()
    got = bench.max_over_ranks(ms, world, "cpu")
    out[rank] = (got, bench.throughput_mpts(1000, 4, world, got * 1e-3))
    dist.destroy_process_group()


def test_max_over_ranks_world_size_2_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0] == out[1]
    assert out[0][0] == 15.0                                   # the max over ranks, on every rank
    assert out[0][1] == pytest.approx(1000 * 4 * 2 / 15e-3 / 1e6)   # whole-job value: both replicas' points


def test_reference_arm_prints_one_json_line_and_other_ranks_stay_silent():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "config1", "--steps", "2", "--warmup", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, env=dict(os.environ, RANK="0"), timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "Mpts/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["config"]["workload"] == "config1"
    r = subprocess.run(cmd, capture_output=True, text=True, env=dict(os.environ, RANK="1", WORLD_SIZE="2"), timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
