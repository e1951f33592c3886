"""N > 1 path on CPU: world_size-2 `gloo` processes exercise the only cross-rank logic the
bench has ("replicas only"): per-rank seeds, MAX over ranks of the times,
SUM over ranks of the units, and the reference arm's "rank 0 alone prints" rule."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1603_09255_b200 import replicas, workloads
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert replicas.env_rank() == (rank, rank, world)
    cfg = replicas.replica_config(workloads.config(3, scale=0.001), rank)
    rows = workloads.initial_rows(cfg, 0)
    # each rank "measured" a different time and processed a different number of units
    times, units = replicas.reduce_over_ranks(dist, [10.0 + rank, 3.0 - rank], [1000 * (rank + 1), 7])
    with open(os.path.join(out_dir, "r%d.json" % rank), "w") as f:
        json.dump({"seed": cfg["seed"], "crc": int(rows.astype(np.uint64).sum() % (1 << 61)), "times": times,
                   "units": units}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_replica_reduction_world2(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / ("r%d.json" % k))) for k in range(world)]
    assert r[0]["seed"] != r[1]["seed"] and r[0]["crc"] != r[1]["crc"]      # independent replicas
    for k in range(world):
        assert r[k]["times"] == [11.0, 3.0]                                    # max over ranks
        assert r[k]["units"] == [3000.0, 14.0]                                 # sum over ranks
    from paper_1603_09255_b200 import replicas
    assert replicas.throughput(3000.0, 11.0) == 3000.0 / 11.0e-3


def test_single_process_reduction_is_identity():
    from paper_1603_09255_b200 import replicas, workloads
    assert replicas.reduce_over_ranks(None, [1.5], [2, 3]) == ([1.5], [2.0, 3.0])
    cfg = workloads.config(3, scale=0.001)
    assert replicas.replica_config(cfg, 0)["seed"] == cfg["seed"]


def test_reference_arm_torchrun_world2():
    """`bench.py --impl reference` under torchrun: rank 0 alone times the oracle and prints ONE
    JSON line with impl=reference; rank 1 exits 0 without work."""
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "3", "--ref-budget-s", "4"]
    p = subprocess.run(cmd, capture_output=True, text=True, env=env, cwd=ROOT, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
