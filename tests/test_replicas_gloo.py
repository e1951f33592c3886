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


# ---- the sweep of unlinked patches (S6) shards by patch: no data-path collective either

def _sweep_worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1603_09255_b200 import replicas
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = replicas.sweep_shard(7, rank, world, scale=0.002)
    sp = cfg["species"][0]
    # gather every rank's block of per-patch parameters (padded to the larger block)
    pad = 4
    mine = torch.full((2, pad), float("nan"), dtype=torch.float64)
    mine[0, :cfg["grid"][0]] = torch.from_numpy(np.asarray(sp["K_patch"], dtype=np.float64))
    mine[1, :cfg["grid"][0]] = torch.from_numpy(np.asarray(sp["gaussian"]["theta_patch"], dtype=np.float64))
    got = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(got, mine)
    _, units = replicas.reduce_over_ranks(dist, [0.0], [cfg["n0"][0]])
    with open(os.path.join(out_dir, "s%d.json" % rank), "w") as f:
        json.dump({"first": cfg["first_patch"], "P": cfg["grid"][0], "seed": cfg["seed"], "units": units,
                   "K": [[x for x in g[0].tolist() if x == x] for g in got],
                   "theta": [[x for x in g[1].tolist() if x == x] for g in got]}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_sweep_shards_by_patch_world2(tmp_path):
    from paper_1603_09255_b200 import replicas, workloads
    world, port = 2, _free_port()
    mp.spawn(_sweep_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / ("s%d.json" % k))) for k in range(world)]
    whole = workloads.sweep_config(n_patches=7, scale=0.002)
    sp = whole["species"][0]
    assert (r[0]["first"], r[0]["P"], r[1]["first"], r[1]["P"]) == (0, 4, 4, 3)
    assert r[0]["seed"] != r[1]["seed"]
    for k in range(world):
        # the blocks, in rank order, are exactly the whole sweep's parameter arrays
        assert np.array_equal(np.concatenate(r[k]["K"]), np.asarray(sp["K_patch"], dtype=np.float64))
        assert np.array_equal(np.concatenate(r[k]["theta"]).astype(np.float32), sp["gaussian"]["theta_patch"])
        assert r[k]["units"] == [float(whole["n0"][0])]


def test_patch_block_partitions():
    from paper_1603_09255_b200 import replicas
    for P in (1, 7, 8, 100):
        for W in (1, 2, 3, 8):
            blocks = [replicas.patch_block(P, r, W) for r in range(W)]
            assert blocks[0][0] == 0 and sum(c for _, c in blocks) == P
            assert all(blocks[i][0] + blocks[i][1] == blocks[i + 1][0] for i in range(W - 1))
            assert max(c for _, c in blocks) - min(c for _, c in blocks) <= 1
