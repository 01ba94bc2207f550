"""Multi-process host logic (N > 1 path of bench.py) on CPU: world_size-2 `gloo` process groups on
127.0.0.1.  The data path has no collective (replicas / member sharding);
what is exercised here is the rendezvous, the barrier, the max-over-ranks of the timed region,
the member partition and the reference arm's rank-0-only contract."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_1611_05293_b200 import dist
    r, lr, w = dist.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    dist.barrier()
    res = {
        "max": dist.reduce_max(10.0 + rank),          # timed region: max over ranks
        "sum": dist.reduce_sum(1.0 + rank),
        "shard": dist.shard_members(7, rank, world),
        "seeds": list(dist.replica_seeds((1, 2), rank)),
    }
    dist.barrier()
    dist.shutdown()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump(res, f)


def test_gloo_world2_barrier_reductions_and_sharding(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    res = [json.load(open(tmp_path / f"r{r}.json")) for r in range(2)]
    assert res[0]["max"] == res[1]["max"] == 11.0
    assert res[0]["sum"] == res[1]["sum"] == 3.0
    assert res[0]["shard"] + res[1]["shard"] == list(range(7))          # disjoint, complete, ordered
    assert len(res[0]["shard"]) - len(res[1]["shard"]) in (0, 1)
    assert res[0]["seeds"] == [1, 2] and res[1]["seeds"] == [1 + 7919, 2 + 7919]


def test_shard_members_edge_cases():
    sys.path.insert(0, ROOT)
    from paper_1611_05293_b200 import dist
    for members in (0, 1, 5, 256):
        for world in (1, 2, 3, 8):
            parts = [dist.shard_members(members, r, world) for r in range(world)]
            assert sum(parts, []) == list(range(members))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        dist.shard_members(4, 2, 2)


def test_reference_arm_two_ranks_prints_once():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 runs the oracle and prints ONE JSON
    line, rank 1 exits 0 without work (no process group is needed for that arm)."""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--workload", "C0", "--steps", "2", "--warmup", "1", "--inner", "5"],
                           capture_output=True, text=True, env=env, timeout=300)
        assert p.returncode == 0, p.stderr[-2000:]
        outs.append([l for l in p.stdout.splitlines() if l.startswith("{")])
    assert len(outs[0]) == 1 and outs[1] == []
    line = json.loads(outs[0][0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
