"""The N>1 plumbing of bench.py (barrier, max-over-ranks of the device time, sum of the processed
bytes) on CPU with the gloo backend, world_size 2.  The hot path itself has no collective: ranks are
independent replicas."""
import os
import socket
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    assert bench.dist_env() == (rank, rank, world)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    ms, units = bench.aggregate(1.0 + rank, 100.0 * (rank + 1), world, device="cpu")
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms, units))


def test_aggregate_world_size_2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # every rank sees max time (2.0 ms) and the summed units (300): value = units / time is whole-job
    assert res == [(0, 2.0, 300.0), (1, 2.0, 300.0)]


def test_aggregate_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 7.0, 1) == (3.5, 7.0)


def test_gpus_flag_spawns_the_ranks_itself():
    """`bench.py --gpus 2` started bare (no torchrun): two rank processes are spawned, rendezvous over gloo, and
    rank 0 prints the aggregate (max of the times, sum of the units) for a world of 2."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--plumbing-only"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    rec = json.loads(lines[0])
    assert rec == {"plumbing_only": True, "n_gpus": 2, "ms_per_step": 2.0, "units": 300.0}


def test_gpus_flag_must_match_the_world():
    import subprocess
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--plumbing-only"], env=env,
                         capture_output=True, text=True, timeout=120)
    assert out.returncode != 0 and "WORLD_SIZE" in out.stderr


def test_watchdog_prints_the_line_and_leaves_when_a_launch_never_returns():
    """bench.guarded: the zero-copy e2e leg runs under it.  A call that never comes back (stood in for by a long
    sleep) makes the watchdog thread print what is known and end the process with status 0; a call that returns in
    time returns its value and the watchdog stays silent."""
    import subprocess
    import time
    code = ("import sys, os, time; sys.path.insert(0, %r); import bench\n"
            "def give_up():\n    print('LINE', flush=True); os._exit(0)\n"
            "print(bench.guarded(lambda: 41 + 1, 5.0, give_up), flush=True)\n"
            "bench.guarded(lambda: time.sleep(60), 0.5, give_up)\n"
            "print('NOT REACHED', flush=True)\n") % ROOT
    t0 = time.time()
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=50)
    assert r.returncode == 0 and r.stdout.split() == ["42", "LINE"], (r.stdout, r.stderr)
    assert time.time() - t0 < 40
