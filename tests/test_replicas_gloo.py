"""N > 1 path of bench.py on CPU: world_size-2 gloo processes (replicas only).  The
path has no data-path collective; what the ranks exchange is the timing (MAX) and the work count (SUM), and
only rank 0 of the reference arm does any work."""
import json
import os
import socket
import subprocess
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (10 + 5 r) ms on 1000 (r + 1) points
    ms, n_all = bench.aggregate_replicas(10.0 + 5.0 * rank, 1000 * (rank + 1))
    dist.barrier()
    dist.destroy_process_group()
    with open(os.path.join(out, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "n_all": n_all, "value": bench.stage_updates_per_s(n_all, 3, ms)}, f)


def test_aggregate_replicas_world2(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    res = [json.load(open(tmp_path / f"r{r}.json")) for r in range(2)]
    for r in res:
        assert r["ms"] == 15.0            # slowest rank
        assert r["n_all"] == 3000.0       # all ranks' points
        assert r["value"] == 3000.0 * 4 * 3 / 15e-3


def test_aggregate_replicas_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_replicas(7.5, 123) == (7.5, 123.0)


def test_reference_arm_under_torchrun_only_rank0_prints():
    """`--impl reference` launched with 2 ranks: rank 0 runs the oracle and prints one JSON line, rank 1
    exits 0 without work."""
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()), WORLD_SIZE="2")
    outs = []
    for rank in (0, 1):
        e = dict(env, RANK=str(rank), LOCAL_RANK=str(rank))
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "0", "--workload", "small"], env=e, capture_output=True,
                           text=True, timeout=600)
        assert p.returncode == 0, p.stderr
        outs.append(p.stdout.strip())
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert outs[1] == ""
