"""-m "not gpu": bench.py's reference arm (the oracle timed on host cores) and its N > 1 launch contract
(under torchrun only rank 0 works and prints; the other ranks exit 0 silently)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _json_lines(out: str):
    return [json.loads(l) for l in out.splitlines() if l.startswith("{")]


def test_reference_arm_single_process():
    r = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--ctx", "2048", "--steps", "2", "--warmup", "1"],
                       cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["unit"] == "GB/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0


def test_reference_arm_under_torchrun_world2():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29631", "bench.py", "--impl", "reference", "--gpus", "2", "--ctx", "1024", "--steps", "1", "--warmup", "1"]
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["impl"] == "reference"


def _gloo_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        ms_local = [3.0, 5.0][rank]                          # the second replica is the slow one
        dist.barrier()
        ms = bench.max_over_ranks(ms_local, world, torch.device("cpu"))
        q.put((rank, ms, bench.replica_value(1.0e9, ms, 10, world), bench.replica_seed_shift(rank)))
    finally:
        dist.destroy_process_group()


def test_replica_aggregation_world2_gloo():
    """bench.py --gpus N (N > 1) runs independent replicas: per-rank seeds, barrier, max-over-ranks time, whole-job value =
    N x per-rank bytes / slowest rank's time.  The host logic, exercised with two gloo processes on CPU."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, 29647, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[0] for g in got] == [0, 1]
    assert all(g[1] == 5.0 for g in got)                    # both ranks see the slowest rank's time
    assert all(abs(g[2] - 2 * 1.0e9 / (0.5e-3) / 1e9) < 1e-9 for g in got)     # 2 replicas x 1 GB per step / 0.5 ms per step
    assert [g[3] for g in got] == [0, 1]                    # distinct workloads per replica
    import bench
    assert bench.max_over_ranks(7.0, 1, None) == 7.0 and bench.replica_value(2.0e9, 4.0, 2, 1) == 1000.0
