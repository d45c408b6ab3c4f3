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


def test_compact_bench_line_is_small_single_line_and_complete(capsys, tmp_path, monkeypatch):
    """The line the driver keeps: bench.compact_line on a canned verbose record (tests/golden/bench_verbose_record.json
    = the 21.6 KB line of round 2, which the driver could not keep) must be one line of JSON under 4 KB that round-trips
    and still carries the contract's keys, `roofline`, `cpu_baseline`, `e2e`, `clocks` and the per-configuration summary;
    emit() prints the verbose record first, behind a non-JSON prefix, and the compact line LAST."""
    import json
    sys.path.insert(0, ROOT)
    import bench
    rec = json.load(open(os.path.join(ROOT, "tests", "golden", "bench_verbose_record.json")))
    assert len(json.dumps(rec)) > 20000
    rec["e2e"]["zero_copy_hung"] = False
    for v in rec["per_config"].values():
        v["traffic_ratio"] = 1.00369
    rec["compact_topk"]["roofline"] = {"bound": "hbm", "achieved": 5771.123, "peak": 6533.2, "unit": "GB/s",
                                       "frac": 0.88335, "traffic": 1601234567}
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))          # emit() writes gpurun_out/bench_detail.json under ROOT
    bench.emit(rec)
    lines = capsys.readouterr().out.strip("\n").split("\n")
    assert len(lines) == 2 and lines[0].startswith("BENCH_DETAIL {")
    assert json.loads(lines[0][len("BENCH_DETAIL "):]) == rec
    assert json.loads(open(tmp_path / "gpurun_out" / "bench_detail.json").read()) == rec
    last = lines[-1]
    assert len(last.encode()) < 4096 and "\n" not in last
    c = json.loads(last)
    assert c == bench.compact_line(rec)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert k in c, k
    assert c["value"] > 0 and c["metric"] == rec["metric"] and c["config"]["workload"] == "8b"
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in c["roofline"], k
    assert abs(c["roofline"]["frac"] - rec["roofline"]["frac"]) < 1e-3
    for k in ("value", "unit", "cores", "kind", "sample"):
        assert k in c["cpu_baseline"], k
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "zero_copy_hung"):
        assert k in c["e2e"], k
    summ = c["config"]["per_config_summary"]
    for name in ("tiny", "8b", "32b", "skew", "uniform"):                  # the five configurations of BASELINE.json
        assert len(summ[name]) == len(summ["columns"])
    assert abs(summ["32b"][summ["columns"].index("pct_of_8tbs")] - rec["per_config"]["32b"]["pct_of_8tbs"]) < 0.1
    assert summ["skew"][summ["columns"].index("cta_spread")] == bench.sig(rec["per_config"]["skew"]["cta_spread"], 2)
    # a record with every optional block missing (multi-rank run) still gives a valid line
    small = {k: rec[k] for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                                 "scaling", "vs_baseline", "dtype", "data", "roofline", "e2e", "clocks", "gpu_launches")}
    small["config"] = {"workload": "8b"}
    assert len(json.dumps(bench.compact_line(small))) < 2048
