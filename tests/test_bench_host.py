"""Host logic of bench.py that needs no GPU: the N > 1 plumbing (replicas only) under a
world_size-2 gloo group, the byte accounting, and the reference arm's rank handling."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r reports (time, spikes, events) = (10 + 5 r, 100 (r + 1), 1000 (r + 1))
    ms, spikes, events = bench.reduce_over_ranks(dist, torch.device("cpu"), 10.0 + 5.0 * rank, 100 * (rank + 1), 1000 * (rank + 1))
    seed = bench.rank_seed(4, rank)
    dist.barrier()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "spikes": spikes, "events": events, "seed": seed}, f)
    dist.destroy_process_group()


def test_two_rank_reduction_and_seeding(tmp_path):
    import torch.multiprocessing as mp
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(2)]
    for x in r:                                   # every rank sees the whole-job figures
        assert x["ms"] == 15.0                    # MAX over ranks
        assert x["spikes"] == 300.0 and x["events"] == 3000.0   # SUM over ranks
    assert r[0]["seed"] != r[1]["seed"]           # independent replicas of the same recipe


def test_single_process_passthrough():
    import bench
    assert bench.reduce_over_ranks(None, None, 7.5, 3, 9) == (7.5, 3, 9)
    from gn_inputs import MASTER_SEED
    assert bench.rank_seed(4, 0) == MASTER_SEED + 4


def test_reference_arm_other_ranks_exit_without_work():
    """Under torchrun only rank 0 runs the oracle; the other ranks print nothing and exit 0."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_reference_arm_prints_the_contract_line_on_a_small_config():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "2",
                        "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-500:]
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "vertex-steps/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0


def test_byte_constants_match_design():
    import bench
    assert bench.UPDATE_BYTES_PER_VERTEX == pytest.approx(24 + 8 + 2 + 1 + 0.125)
    assert bench.EVENT_BYTES == 9 + 8 and bench.SOURCE_BYTES == 12
