"""Host-side logic of the N-GPU path on CPU: frequency sharding + one image all-reduce (gloo, world 2).

The per-rank migration itself is stood in for by the FP64 oracle (this is a test of the sharding
and the exchange step); the identity being checked is the oracle's own pin P8:
image(S1 u S2) = image(S1) + image(S2) for disjoint frequency sets.
"""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
import pdm_inputs
from paper_1912_05529_b200.shard import shard_lines, shard_workload

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_lines_partition_every_line_exactly_once():
    for nw in (1, 2, 7, 92, 803):
        for world in (1, 2, 3, 8):
            if world > nw:
                with pytest.raises(ValueError):
                    shard_workload({"nw": nw, "omega": np.zeros(nw, np.float32),
                                    "P0": np.zeros((nw, 1), np.complex64)}, world - 1, world)
                continue
            got = np.concatenate([shard_lines(nw, r, world) for r in range(world)])
            assert sorted(got.tolist()) == list(range(nw))
            sizes = [shard_lines(nw, r, world).size for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_lines(5, 2, 2)


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch
    import torch.distributed as dist
    from paper_1912_05529_b200.shard import allreduce_image
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    cfg = pdm_inputs.random_problem(77, 96, 10, 7, 15, model="field")
    mine = shard_workload(cfg, rank, world)
    part = oracle.migrate(mine)                            # stands in for the rank's pdm_migrate
    img = torch.from_numpy(part.astype(np.float32))
    allreduce_image(img)
    np.save(os.path.join(out_dir, f"rank{rank}.npy"), img.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_allreduce_reproduces_the_unsharded_image(tmp_path):
    import torch.multiprocessing as mp
    port = 29500 + (os.getpid() % 2000)
    mp.start_processes(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True, start_method="spawn")
    cfg = pdm_inputs.random_problem(77, 96, 10, 7, 15, model="field")
    full = oracle.migrate(cfg)
    a = np.load(tmp_path / "rank0.npy")
    b = np.load(tmp_path / "rank1.npy")
    assert np.array_equal(a, b)                            # every rank holds the same reduced image
    rel = np.linalg.norm(a - full) / np.linalg.norm(full)
    assert rel < 1e-6


def test_bench_reference_arm_prints_the_contract_line():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--config", "0", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "samples/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0 and line["higher_is_better"] is True
