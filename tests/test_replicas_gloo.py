"""The N > 1 path of bench.py on CPU: two processes over gloo.  The method does not shard ("replicas only",
DESIGN.md "Multi-GPU"), so the only cross-rank logic is the barrier around the timed region, the
max-over-ranks time, the sum of the work and `--impl reference` running on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_1004_1932_b200.replicas import Ranks
    r = Ranks(backend="gloo")
    try:
        assert (r.rank, r.world) == (rank, world)
        r.barrier()
        seconds = 1.0 + rank          # rank 1 is the slow replica
        units = 100.0 * (rank + 1)
        res = dict(max=r.max(seconds), sum=r.sum(units), thr=r.throughput(units, seconds))
        r.barrier()
        out.put((rank, res))
    finally:
        r.close()


def test_two_replicas_over_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(k, 2, port, out)) for k in range(2)]
    for p in procs:
        p.start()
    got = dict(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank in (0, 1):
        assert got[rank]["max"] == 2.0                    # the job is as slow as its slowest replica
        assert got[rank]["sum"] == 300.0                  # all replicas' units
        assert got[rank]["thr"] == 150.0                  # whole-job throughput, identical on every rank


def test_world_size_one_needs_no_process_group():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    code = ("import sys; sys.path.insert(0, %r); from paper_1004_1932_b200.replicas import Ranks; r = Ranks(); "
            "r.barrier(); assert r.max(3.5) == 3.5 and r.sum(2.0) == 2.0; r.close(); print('ok')" % ROOT)
    assert subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True).stdout.strip() == "ok"


def test_reference_arm_runs_on_rank0_only_under_torchrun_env():
    """bench.py --impl reference with WORLD_SIZE=2: rank 1 exits 0 without output; rank 0 prints one JSON line
    whose keys follow the contract (the oracle on the host cores; tiny run)."""
    base = {k: v for k, v in os.environ.items()}
    base.update(WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0"]
    r1 = subprocess.run(cmd, env=dict(base, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=600)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(base, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=600)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["unit"] == "pairs/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["value"] > 0 and line["vs_baseline"] is None
