"""Host logic of bench.py (no GPU): the N > 1 aggregation over ranks on gloo (world size 2), the
roofline byte model, the bounded oracle sample and the `--impl reference` JSON line."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms, upd = bench.aggregate_over_ranks(100.0 + 50.0 * rank, 1000 * (rank + 1), dist)
    dist.barrier()
    q.put((rank, ms, upd))
    dist.destroy_process_group()


def test_aggregate_over_ranks_gloo_world2():
    """Replicas only: time = max over ranks, updates = sum over ranks."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, upd in got:
        assert ms == 150.0 and upd == 3000


def test_aggregate_single_rank_is_identity():
    import bench
    assert bench.aggregate_over_ranks(12.5, 77, None) == (12.5, 77)


def test_algorithmic_bytes_model():
    import bench
    # Q read + phi read-modify-write + sigma_t shared by the batch
    assert bench.algorithmic_bytes_per_cell_octant(16, 4) == 64 + 128 + 1
    assert bench.algorithmic_bytes_per_cell_octant(1, 1) == 4 + 8 + 4
    peak, src = bench.measured_peak()
    assert 3000 < peak < 9000 and ("measured" in src or "fallback" in src)


def test_oracle_sample_is_bounded():
    import bench
    for idx in (2, 3, 4):
        wl, what = bench.oracle_sample(idx)
        assert wl.G == 1 and len(wl.sources) == 1 and wl.fixed_iters >= 1
        assert wl.cells * wl.n_dir * wl.fixed_iters <= 1.4e9          # ~10-30 s of oracle work
        assert "group 0" in what


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["steps"] == 2 and line["warmup"] == 1 and line["higher_is_better"] is True
    # config 0: 10 sweeps x 512 cells x 8 directions per step.  `value` is the oracle's SWEEP rate (sweeps timed apart from the
    # ray trace and the fixed-source assembly); the whole step is e2e.value and ms_per_step
    upd = 10 * 512 * 8
    assert abs(line["e2e"]["value"] * line["ms_per_step"] * 1e-3 - upd) < 1e-6 * upd
    split = line["ms_per_step_split"]
    assert abs(line["value"] * split["sweep"] * 1e-3 - upd) < 1e-6 * upd
    assert split["sweep"] + split["raytrace"] + split["fixed_source"] <= line["ms_per_step"] and line["value"] >= line["e2e"]["value"]
    assert line["config"]["workload"] == "cfg0_8c_S2P0" and "sample" in line["config"]
