#!/usr/bin/env python
"""bench.py -- decode-attention layer-step benchmark of the Tangram hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 8b] [--impl ours|reference]

One "step" = one pass of the whole hot path's device side over one batch: one
tangram_decode_attention call (split-KV decode kernel with the LSE merge inside its persistent grid:
one cooperative launch) on the uploaded AoT plan.
The host planners (a1-a3) run once before the timed region (zero runtime planning) and
are reported separately in ms.  Prints ONE JSON line (rank 0).  See DESIGN.md §Measurement.

Multi-GPU: the path shards by request with no exchange step, so --gpus N runs N independent
replicas of the workload (one process per GPU, weak scaling); torch.distributed is used only for the
barrier and the max-over-ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "decode-attention µs per layer-step and achieved HBM TB/s (% of ~8 TB/s)"
NOMINAL_TBS = 8.0
FALLBACK_PEAK_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback


def csrc_hash(files=("tangram_decode.cu", "tangram_internal.h")) -> str:
    """sha256 (first 16 hex digits) over a kernel's sources (by default the decode kernel's: tangram_decode.cu +
    tangram_internal.h): ties a committed ncu capture of that kernel to the code it measured."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_06302_b200", "csrc")
    for fn in files:
        h.update(fn.encode())
        h.update(open(os.path.join(d, fn), "rb").read())
    return h.hexdigest()[:16]


KERNEL_SOURCES = {"tangram_decode_kernel": ("tangram_decode.cu", "tangram_internal.h"),
                  "tangram_compact_topk": ("tangram_compact.cu", "tangram_internal.h")}


def profiled_traffic(workload: str, kernel: str = "tangram_decode_kernel"):
    """dram__bytes_read.sum + dram__bytes_write.sum of a kernel (for tangram_compact_topk: of the call's three kernels
    together), per launch, from the committed `ncu --set full` capture of this workload (profiles/*_traffic.csv) --
    only from a row whose `csrc_hash` column equals the hash of the current sources of that kernel (a capture of
    older code says nothing about this build); else None."""
    best = None
    try:
        import csv
        import glob
        cur = csrc_hash(KERNEL_SOURCES[kernel])
        for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
            for row in csv.DictReader(open(path)):
                if row["workload"] == workload and row["kernel"] == kernel and row.get("csrc_hash", "") == cur:
                    best = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    except Exception:
        return None
    return best


def sig(x, n=4):
    """x rounded to n significant digits (None, bools, ints and strings pass through)."""
    if isinstance(x, bool) or not isinstance(x, float):
        return x
    if x == 0 or not math.isfinite(x):
        return x
    return round(x, n - 1 - int(math.floor(math.log10(abs(x)))))


COMPACT_LINE_LIMIT = 4096      # bytes; the driver's record kept round 1's 10.6 KB line and lost round 2's 21.6 KB one


def compact_line(line: dict) -> dict:
    """The ONE JSON line the driver keeps, built from the verbose record: the contract's keys, `roofline`,
    `cpu_baseline`, `e2e`, `clocks`, `gpu_launches` and a `config` that names the workload, the plan and one summary row
    per configuration -- numbers to 3-4 significant digits, no prose, nothing twice.  Everything else stays in the
    verbose record (the BENCH_DETAIL line printed before it, gpurun_out/bench_detail.json)."""
    cfg = line.get("config", {})
    out = {k: sig(line[k], 6) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
                                        "higher_is_better", "scaling", "vs_baseline", "dtype", "data") if k in line}
    if "impl" in line:
        out["impl"] = line["impl"]
    out["us_per_layer_step"] = sig(line.get("us_per_layer_step"))
    out["pct_of_8tbs_nominal"] = sig(line.get("pct_of_8tbs_nominal"))
    c = {k: cfg[k] for k in ("workload", "R", "Hq", "H", "d", "page_size", "clusters", "plan", "W", "dyn_permille",
                             "dyn_rounds", "granule", "c0", "items", "kv_bytes", "algorithmic_bytes") if k in cfg}
    c["l2"] = "inputs > L2 and an L2 flush before every timed step"
    c["multi_gpu"] = "replicas only"
    if "cta_spread" in line:
        c["cta_spread"] = sig(line["cta_spread"], 3)
    per = line.get("per_config")
    if per:
        cols = ["us", "tbs", "pct_of_8tbs", "kernel_gbs", "cta_spread", "static_even_x", "traffic_ratio"]
        rows = {}
        for k, v in per.items():
            rows[k] = [sig(v.get("us_per_layer_step"), 4), sig(v.get("tbs"), 3), sig(v.get("pct_of_8tbs"), 3),
                       sig(v.get("decode_kernel_gbs"), 4), sig(v.get("cta_spread"), 2),
                       sig(v.get("static_even", {}).get("slowdown_vs_balanced"), 3), sig(v.get("traffic_ratio"), 4)]
        c["per_config_summary"] = {"columns": cols, **rows}
    dl = line.get("decode_loop")
    if dl:
        c["decode_loop"] = {"us_per_layer_step": sig(dl.get("us_per_layer_step")), "layers": dl.get("layers"),
                            "launches_per_layer_step": dl.get("launches_per_layer_step"), "overflow": dl.get("overflow")}
    ct = line.get("compact_topk")
    if ct:
        c["compact_topk"] = {"us": sig(ct.get("us")), "pct_of_measured_copy": sig(ct.get("pct_of_measured_copy"), 3),
                             "roofline": {k: sig(v) for k, v in ct.get("roofline", {}).items()}}
    out["config"] = c
    r = line.get("roofline", {})
    out["roofline"] = {k: sig(r[k], 5) for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic",
                                                 "kernel_us", "algorithmic_bytes_per_launch", "read_peak_gbs",
                                                 "frac_of_read_peak") if k in r}
    if "peak_source" in r:
        out["roofline"]["peak_source"] = "measured" if str(r["peak_source"]).startswith("measured") else "fallback"
    cb = line.get("cpu_baseline")
    if cb:
        out["cpu_baseline"] = {k: sig(cb[k]) for k in ("value", "unit", "cores", "kind") if k in cb}
        out["cpu_baseline"]["sample"] = str(cb.get("sample", ""))[:160]
        if "us_per_layer_step_extrapolated" in cb:
            out["cpu_baseline"]["us_per_layer_step_extrapolated"] = sig(cb["us_per_layer_step_extrapolated"])
    e = line.get("e2e")
    if e:
        out["e2e"] = {k: sig(e[k]) for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "us_per_layer_step",
                                             "us_per_layer_step_staged_copies", "zero_copy", "zero_copy_hung") if k in e}
    if "clocks" in line:
        out["clocks"] = line["clocks"]
    if "gpu_launches" in line:
        out["gpu_launches"] = line["gpu_launches"]
    out["detail"] = "BENCH_DETAIL line above; gpurun_out/bench_detail.json"
    return out


def emit(line: dict):
    """Prints the verbose record on a line of its own behind a non-JSON prefix (and writes it to
    gpurun_out/bench_detail.json when that folder can be written), then -- LAST -- the compact JSON line."""
    detail = json.dumps(line)
    print("BENCH_DETAIL " + detail, flush=True)
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "bench_detail.json"), "w") as f:
            f.write(detail + "\n")
    except OSError:
        pass
    text = json.dumps(compact_line(line), separators=(",", ":"))
    assert "\n" not in text and len(text.encode()) <= COMPACT_LINE_LIMIT, f"compact bench line is {len(text.encode())} bytes"
    print(text, flush=True)


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_PEAK_GBS, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------
# distributed plumbing (also exercised on CPU with gloo by tests/test_bench_dist.py)
# ------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def aggregate(ms_local: float, units_local: float, world: int, device=None):
    """max over ranks of the device time, sum over ranks of the processed units."""
    if world == 1:
        return ms_local, units_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def spawn_ranks(n: int, argv) -> int:
    """`bench.py --gpus N` started bare (no torchrun, WORLD_SIZE unset): start the N ranks ourselves, one process per
    GPU, rendezvous on 127.0.0.1, and wait for them.  Rank 0 prints the JSON line."""
    import socket
    import subprocess
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    procs = []
    for r in range(n):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(n), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + list(argv), env=env))
    rcs = [p.wait() for p in procs]
    return next((rc for rc in rcs if rc != 0), 0)


def plumbing_only(args):
    """The multi-rank plumbing without the GPU work (tests/test_bench_dist.py, gloo on CPU): rendezvous, barrier,
    max-over-ranks / sum-over-ranks aggregation, rank 0 prints one JSON line."""
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1:
        dist.init_process_group("gloo", rank=rank, world_size=world)
        dist.barrier()
    ms, units = aggregate(1.0 + rank, 100.0 * (rank + 1), world, device="cpu")
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"plumbing_only": True, "n_gpus": world, "ms_per_step": ms, "units": units}))


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.004):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
            self._period = period_s
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else 0x8,
                 "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4,
                 "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self._period)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": int(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------
# workload setup through the product's own API
# ------------------------------------------------------------------------------------------------
def algorithmic_bytes(wl, kv, plan, t):
    """sum kv_len*4d (K+V bf16) + q in / out + partials out+in + page ids."""
    d, G = wl.d, wl.G
    kv_bytes = int(kv.astype(np.int64).sum()) * 4 * d
    qo = 2 * wl.R * wl.Hq * d * 2
    multi = plan.items[plan.items[:, 7] > 1]
    partials = int(multi.shape[0]) * G * (d + 1) * 4 * 2
    page_ids = 4 * int(np.sum(-(-kv.astype(np.int64) // wl.P)))
    return {"kv": kv_bytes, "q_out": qo, "partials": partials, "page_ids": page_ids,
            "total": kv_bytes + qo + partials + page_ids}


def setup_workload(T, I, name, device, W=None, mode=None, c0=1, dyn=None, layer=0, plan_capacity=False, R=None,
                   headroom=0, page_size=None):
    """Budgets, tables and plan of workload `name` through the product's API.  headroom > 0: growable tables (that
    many empty page slots per row, and a pool / free list large enough to fill them) for the decode loop."""
    import torch
    wl = I.make_workload(name, layer=layer, R=R, page_size=page_size)
    t0 = time.perf_counter()
    B, res, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    need = T.tangram_pages_needed(B, res, wl.C, wl.P)
    n_pool = int(math.ceil(1.05 * need)) + headroom * wl.R * wl.C
    free = I.make_free_pages(wl, n_pool)
    t1 = time.perf_counter()
    tb, kv = T.tangram_build_ragged_tables(B, res, wl.C, wl.P, free, 0, kv, headroom_pages=headroom)
    t2 = time.perf_counter()
    if W is None:
        W = T.tangram_query_max_ctas(torch.cuda.current_device(), wl.d, wl.G)
    t3 = time.perf_counter()
    kv_plan = kv
    if plan_capacity:      # open-ended plan: built once for the tables' capacity, serves every decode step
        rows = np.arange(wl.R)[:, None] * tb.C + tb.cluster_of[None, :]
        kv_plan = ((tb.tbl_indptr[rows + 1] - tb.tbl_indptr[rows]) * wl.P).astype(np.int32)
    if dyn is None:        # the library's default: dynamic tail 500/6, or the static plan for a small batch
        dyn = T.tangram_default_dynamic_tail(kv_plan, W, wl.granule, c0)
    plan = T.tangram_plan_partitions(tb, B, kv_plan, W, wl.granule, c0, T.MODE_BALANCED if mode is None else mode, 0,
                                     dyn[0], dyn[1])
    t4 = time.perf_counter()
    q, pool = I.make_q_and_pool(wl, n_pool, device)
    host_ms = {"reserve_ms": (t1 - t0) * 1e3, "tables_ms": (t2 - t1) * 1e3, "plan_ms": (t4 - t3) * 1e3}
    return dict(wl=wl, B=B, res=res, kv=kv, tables=tb, plan=plan, W=W, q=q, pool=pool, n_pool=n_pool,
                host_ms=host_ms, c0=c0, dyn=dyn, free=free)


class L2Flusher:
    """Flushes the 126 MB L2 between timed iterations: writes a 256 MB buffer (evicts everything the
    previous step left), then reads a second 256 MB buffer so that the dirty lines of the write are
    themselves written back BEFORE the timed region starts -- otherwise up to ~126 MB of write-back
    traffic from the flush would be charged to the step being timed."""

    def __init__(self, device, nbytes=256 << 20):
        import torch
        self.buf = torch.empty(nbytes, dtype=torch.uint8, device=device)
        self.rd = torch.zeros(nbytes // 4, dtype=torch.int32, device=device)
        self.v = 0

    def __call__(self):
        self.v = (self.v + 1) & 0x7F
        self.buf.fill_(self.v)
        self.rd.max()


def time_steps(fn, steps, warmup, flush, torch):
    """Device time of `steps` calls of fn, CUDA events on the current stream, L2 flushed before
    every call (the flush is outside the event pair).  Returns per-step ms list."""
    for _ in range(warmup):
        flush()
        fn()
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        flush()
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (a reported baseline, not the target)
# ------------------------------------------------------------------------------------------------
def oracle_tables(O, t):
    return O.Tables(R=t.R, H=t.H, C=t.C, Hp=t.Hp, P=t.P, perm=t.perm, cluster_of=t.cluster_of,
                    slot_of=t.slot_of, tbl_indptr=t.tbl_indptr, tbl_pages=t.tbl_pages,
                    n_pages_used=t.n_pages_used)


def oracle_sample_pairs(wl, kv, budget_tokens_heads, rng):
    """A bounded random sample of (request, query head) pairs whose KV token-heads add up to about
    `budget_tokens_heads` (each pair streams kv_len[r][h] tokens of one KV head)."""
    pairs, tot = [], 0
    order = rng.permutation(wl.R * wl.Hq)
    for idx in order:
        r, j = int(idx // wl.Hq), int(idx % wl.Hq)
        n = int(kv[r, j // wl.G])
        if n == 0:
            continue
        pairs.append((r, j))
        tot += n
        if tot >= budget_tokens_heads:
            break
    return pairs, tot


def run_oracle_sample(O, S, q_cpu, pool_cpu, pairs, threads=0):
    wl = S["wl"]
    t0 = time.perf_counter()
    _, _, used = O.attention_pairs(q_cpu, pool_cpu, oracle_tables(O, S["tables"]), S["kv"], wl.Hq, wl.d, pairs, threads)
    return time.perf_counter() - t0, used


def cpu_baseline(O, S, target_s=15.0):
    """Times the oracle as it stands on this box's host cores on a bounded sample of the workload."""
    wl = S["wl"]
    q_cpu, pool_cpu = S["q"].cpu(), S["pool"].cpu()
    rng = np.random.default_rng(wl.seed + 1)
    probe_pairs, probe_tok = oracle_sample_pairs(wl, S["kv"], 200_000, rng)
    dt, used = run_oracle_sample(O, S, q_cpu, pool_cpu, probe_pairs)
    rate = probe_tok / max(dt, 1e-6)                      # query-head token visits per second
    total_visits = int(S["kv"].astype(np.int64).sum()) * wl.G
    pairs, tok = oracle_sample_pairs(wl, S["kv"], min(total_visits, rate * target_s / 8), rng)
    # about 10-30 s of CPU work in total: repeat the sample until ~1.5 s of wall time has passed
    dt, reps = 0.0, 0
    while dt < 1.5 and reps < 64:
        d1, used = run_oracle_sample(O, S, q_cpu, pool_cpu, pairs)
        dt, reps = dt + d1, reps + 1
    tok *= reps
    # the oracle re-reads K/V once per query head; the algorithmic KV bytes of the sample count each
    # KV head's tokens once per G query heads, as for the GPU path
    alg_bytes = tok / wl.G * 4 * wl.d
    tbs = alg_bytes / dt / 1e12
    return {"value": tbs, "unit": "TB/s", "cores": used, "kind": "oracle",
            "sample": f"{len(pairs)} of {wl.R * wl.Hq} (request, query head) rows of the {wl.name} workload x {reps} "
                      f"repetitions, {tok} token visits, {dt:.2f} s wall on {used} threads",
            "us_per_layer_step_extrapolated": total_visits / (tok / dt) * 1e6}


def reference_arm(args):
    """--impl reference: the fp64 CPU oracle timed on the host cores; each step a bounded sample."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import tangram_oracle as O
    from paper_2606_06302_b200 import inputs as I
    O.build_c()
    name = args.workload
    wl = I.make_workload(name)
    B, res, kv = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    # a pool that holds only what the sampled rows touch would change nothing for the oracle; keep
    # the recipe: 1.05 x pages needed, seeded free list, every slot random (CPU generator)
    upper = int(sum(wl.C * (-(-int(n) // wl.P)) for n in wl.ctx_len))
    t_probe, _ = O.build_ragged_tables(B, res, wl.C, wl.P, np.arange(upper, dtype=np.int32))
    n_pool = int(math.ceil(1.05 * t_probe.n_pages_used))
    t, kv = O.build_ragged_tables(B, res, wl.C, wl.P, I.make_free_pages(wl, n_pool), 0, kv)
    q, pool = I.make_q_and_pool(wl, n_pool, "cpu")
    S = dict(wl=wl, kv=kv, tables=t)
    rng = np.random.default_rng(wl.seed + 1)
    probe_pairs, probe_tok = oracle_sample_pairs(wl, kv, 100_000, rng)
    dt, used = run_oracle_sample(O, S, q, pool, probe_pairs)
    rate = probe_tok / max(dt, 1e-6)
    per_step_s = min(10.0, 120.0 / max(1, args.steps + args.warmup))
    times, toks = [], []
    for i in range(args.warmup + args.steps):
        pairs, tok = oracle_sample_pairs(wl, kv, max(1.0, rate * per_step_s), rng)
        dt, used = run_oracle_sample(O, S, q, pool, pairs)
        if i >= args.warmup:
            times.append(dt)
            toks.append(tok)
    alg_bytes = sum(toks) / wl.G * 4 * wl.d
    tbs = alg_bytes / sum(times) / 1e12
    n_rows = wl.R * wl.Hq
    sample = (f"each step = {len(pairs)} of the {n_rows} (request, query head) rows of the {name} workload "
              f"({int(np.mean(toks))} token visits, {np.mean(times):.3f} s of oracle time per step on {used} threads; "
              f"the sample is capped at the whole workload or ~{per_step_s:.0f} s, whichever is smaller)")
    line = {"impl": "reference", "metric": METRIC, "value": tbs, "unit": "TB/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(times) * 1e3),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": name, "note": "fp64 CPU oracle, bounded sample per step"},
            "cpu_baseline": {"value": tbs, "unit": "TB/s", "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": tbs, "unit": "TB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# NEXT-1: a real decode loop -- L layers x (KV append + attention) per step under ONE CUDA graph
# ------------------------------------------------------------------------------------------------
def decode_loop(T, I, name, device, layers, steps, torch):
    """Every layer has its own budgets, clusters, growable tables and an open-ended plan built once for the tables'
    slot capacity; one decode step = for each layer ONE launch of tangram_decode_step (KV append + attention +
    merge + length update + block-table growth for the next step), chained by programmatic dependent launch.  The
    L-layer step is captured in one CUDA graph and replayed: zero host work across steps and layers.
    The layers' pools are distinct and far larger than L2 together, so no flush is needed between layer-steps.
    `two_launches` is the round-1 loop (tangram_append_kv + tangram_decode_attention) on the same data."""
    headroom = (steps + 8) // 16 + 2                     # page slots for every token the loop appends
    Ls = []
    for l in range(layers):
        S = setup_workload(T, I, name, device, layer=l, plan_capacity=True, headroom=headroom)
        prepare(T, S, torch)
        S["kv_dev"] = torch.as_tensor(S["kv"], device=device)
        S["kv_dev2"] = S["kv_dev"].clone()
        S["free_dev"] = torch.as_tensor(S["free"], device=device)
        S["over"] = torch.zeros(2, dtype=torch.int32, device=device)
        S["pages0"] = int(S["tables"].n_pages_used)
        g = torch.Generator(device=device).manual_seed(S["wl"].seed + 17)
        S["k_new"] = torch.randn(S["wl"].R, S["wl"].H, S["wl"].d, generator=g, device=device).bfloat16()
        S["v_new"] = torch.randn(S["wl"].R, S["wl"].H, S["wl"].d, generator=g, device=device).bfloat16()
        Ls.append(S)

    def fused_step(stream=None):
        for S in Ls:
            T.tangram_decode_step(S["dp"], S["q"], S["k_new"], S["v_new"], S["pool"], S["kv_dev"], S["free_dev"], S["out"],
                                  S["lse"], S["ws"], overflow=S["over"][0:1], flags=T.STEP_OVERLAP, stream=stream)

    def two_launch_step(stream=None):
        for S in Ls:
            T.tangram_append_kv(S["dp"], S["k_new"], S["v_new"], S["pool"], S["kv_dev2"], S["over"][1:2], stream=stream)
            T.tangram_decode_attention(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"], kv_len=S["kv_dev2"],
                                       stream=stream)

    def timed(one_step, n):
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(st):
            one_step(st)                                  # warm-up outside the capture
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=st):
                one_step(st)
            for _ in range(3):
                graph.replay()
            st.synchronize()
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
            for a, b in evs:
                a.record(st)
                graph.replay()
                b.record(st)
            st.synchronize()
        torch.cuda.current_stream().wait_stream(st)
        return np.array([a.elapsed_time(b) for a, b in evs])

    for S in Ls:                                          # room for the first appended token
        T.tangram_extend_tables_device(S["dp"], S["kv_dev"], S["free_dev"])
    len0 = float(np.mean([int(S["kv_dev"].sum().item()) for S in Ls]))
    ms = timed(fused_step, steps - 4)                     # 1 eager + 3 warm replays + (steps - 4) timed = steps appends
    len1 = float(np.mean([int(S["kv_dev"].sum().item()) for S in Ls]))
    kv_bytes = 0.5 * (len0 + len1) * 4 * Ls[0]["wl"].d    # mean retained K/V over the loop (lengths grow every step)
    us_layer = float(np.median(ms)) * 1e3 / layers
    ms2 = timed(two_launch_step, max(4, (steps - 4) // 2))
    us_layer2 = float(np.median(ms2)) * 1e3 / layers
    torch.cuda.synchronize()
    starved = sum(T.tangram_download_tables(S["dp"], S["tables"]) for S in Ls)
    return {"layers": layers, "steps": steps, "us_per_layer_step": us_layer, "us_per_decode_step": us_layer * layers,
            "tbs": kv_bytes / (us_layer * 1e-6) / 1e12, "pct_of_8tbs": 100 * kv_bytes / (us_layer * 1e-6) / 1e12 / NOMINAL_TBS,
            "launches_per_layer_step": 1, "host_planning_per_step_ms": 0.0,
            "overflow": int(sum(int(S["over"][0].item()) for S in Ls)), "rows_starved": int(starved),
            "tokens_appended_per_head": steps,
            "pages_handed_out": int(sum(S["tables"].n_pages_used - S["pages0"] for S in Ls)),
            "overlap_state": T.tangram_overlap_state(),
            "two_launches": {"us_per_layer_step": us_layer2, "overflow": int(sum(int(S["over"][1].item()) for S in Ls)),
                             "note": "round-1 loop: tangram_append_kv + tangram_decode_attention, tables never grow"},
            "note": "one tangram_decode_step launch per layer (append + attention + merge + lengths + table growth), "
                    "chained by programmatic dependent launch, open-ended plans built once, whole L-layer step in one "
                    "CUDA graph; kv bytes = mean retained K/V over the loop"}


# ------------------------------------------------------------------------------------------------
# NEXT-2: per-head Top-k selection + compaction into the ragged pages (the step that fills the pool)
# ------------------------------------------------------------------------------------------------
def compact_topk_summary(T, I, name, device, steps, flush, torch, peak_gbs):
    """tangram_compact_topk on the workload's shape: scores [R,H,n_max] f32 and the uncompressed cache
    [R,H,n_max,d] bf16 are resident; one call = prepare + top-k select + gather (three launches).  The
    gather is the HBM-bound part: 4d bytes read + 4d bytes written per retained token-head."""
    S = setup_workload(T, I, name, device)
    wl, kv = S["wl"], S["kv"]
    dp = T.tangram_upload(S["tables"], S["plan"])
    n_max = int(wl.ctx_len.max())
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, device)
    ctx = torch.as_tensor(wl.ctx_len, device=device)
    keep = torch.as_tensor(np.ascontiguousarray(kv, dtype=np.int32), device=device)
    idx = torch.empty(wl.R, wl.H, n_max, dtype=torch.int32, device=device)
    ws = torch.empty(T.tangram_compact_workspace_bytes(wl.R, wl.H), dtype=torch.uint8, device=device)
    step = lambda: T.tangram_compact_topk(dp, scores, kd, vd, ctx, keep, S["pool"], idx_out=idx, workspace=ws)
    ms = time_steps(step, steps, 3, flush, torch)
    kept = int(kv.sum())
    gather_bytes = kept * 4 * wl.d * 2 + kept * 4            # rows read + rows written + indices read
    score_bytes = int(wl.ctx_len.astype(np.int64).sum()) * wl.H * 4
    us = float(np.median(ms) * 1e3)
    gbs = gather_bytes / (us * 1e-6) / 1e9
    roof = {"bound": "hbm", "achieved": gbs, "peak": peak_gbs, "unit": "GB/s", "frac": gbs / peak_gbs,
            "traffic": profiled_traffic(name, "tangram_compact_topk")}
    return {"workload": name, "us": us, "us_min": float(np.min(ms) * 1e3), "launches": 3, "roofline": roof,
            "retained_token_heads": kept, "gather_bytes": gather_bytes, "score_bytes_one_pass": score_bytes,
            "gbs_gather_bytes_over_total_time": gather_bytes / (us * 1e-6) / 1e9,
            "pct_of_measured_copy": 100 * gather_bytes / (us * 1e-6) / 1e9 / peak_gbs,
            "note": "whole call (select + gather) timed with CUDA events, L2 flushed; bytes = K/V rows read + "
                    "written; the select kernel reads the scores three times (first pass from HBM, then L2); "
                    "kernel shares: profiles/"}


# ------------------------------------------------------------------------------------------------
# NEXT-3: memory reclaimed vs heads per page, with and without Budget-Aware Clustering (host only)
# ------------------------------------------------------------------------------------------------
def page_accounting_summary(T, I, name):
    """Fig. 12 / Fig. 15 quantities on the synthetic profile of the workload: fraction of the full KV cache
    reclaimed when H_p heads share a page table, heads grouped by budget (clustered) or by index (adjacent)."""
    wl = I.make_workload(name)
    B, res, _ = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    out = {"workload": name, "unit": "fraction of the full (uncompressed, paged) KV cache of the layer"}
    for Hp in [d for d in (1, 2, 4, 8) if wl.H % d == 0]:
        clu = T.tangram_account_pages(B, res, wl.ctx_len, Hp, wl.P, T.GROUP_CLUSTERED)
        adj = T.tangram_account_pages(B, res, wl.ctx_len, Hp, wl.P, T.GROUP_ADJACENT)
        out[f"Hp{Hp}"] = {"reclaimed_clustered": clu["reclaimed_frac"], "reclaimed_adjacent": adj["reclaimed_frac"],
                          "extra_from_clustering": clu["reclaimed_frac"] - adj["reclaimed_frac"],
                          "fragmentation_clustered": clu["fragmentation"], "tables": clu["tables"],
                          "pages": clu["pages_alloc"]}
    return out


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def spread_of(T, S, torch, reps=5, detail=False):
    """Per-CTA elapsed-time spread (max - min) / mean of the worker CTAs' busy time, from the
    globaltimer stamps of the instrumented build (median over reps).  detail=True also returns the quantiles of the
    busy times (us), the spread of the bytes the plan assigned to the CTAs' own lists, and how stable the ranking of
    fast and slow CTAs (= SMs: one CTA per SM) is from launch to launch (correlation of the busy times)."""
    W = S["plan"].n_static
    ns = torch.zeros(W, 4, dtype=torch.int64, device=S["q"].device)
    dp = S["dp"]
    vals, runs = [], []
    live = np.diff(S["plan"].worker_indptr)[:W] > 0
    for _ in range(reps):
        T.tangram_decode_partials(dp, S["q"], S["pool"], S["out"], S["lse"], S["ws"], worker_ns=ns)
        torch.cuda.synchronize()
        a = ns.cpu().numpy().astype(np.float64)
        busy = (a[:, 1] - a[:, 0])[live]
        runs.append(busy)
        vals.append(float((busy.max() - busy.min()) / busy.mean()))
    if not detail:
        return float(np.median(vals))
    b = runs[-1] / 1e3
    items, wi = S["plan"].items, S["plan"].worker_indptr
    own = np.array([int((items[wi[k]:wi[k + 1], 5] - items[wi[k]:wi[k + 1], 4]).sum()) for k in range(W)], dtype=np.float64)[live]
    corr = [float(np.corrcoef(runs[i], runs[i + 1])[0, 1]) for i in range(len(runs) - 1)] if b.size > 2 else []
    return float(np.median(vals)), {
        "busy_us": {"min": float(b.min()), "p10": float(np.percentile(b, 10)), "median": float(np.median(b)),
                    "p90": float(np.percentile(b, 90)), "max": float(b.max())},
        "own_list_tokens_spread": float((own.max() - own.min()) / own.mean()) if own.size else 0.0,
        "busy_vs_own_tokens_corr": float(np.corrcoef(b, own)[0, 1]) if b.size > 2 and own.std() > 0 else None,
        "launch_to_launch_corr": corr}


def timeline_of(T, S, torch, flush, reps=5):
    """Where a step's time goes, from the instrumented kernel's globaltimer stamps (us after the first CTA starts,
    median over reps): the first and the last CTA running out of work lists, the last wait for a record's parts ended (in-grid merge),
    CTA, the last merge done.  The CUDA-event time of the same launch adds the launch / completion floor."""
    W = S["plan"].n_static
    ns = torch.zeros(W, 4, dtype=torch.int64, device=S["q"].device)
    rows = []
    for _ in range(reps):
        flush()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        T.tangram_decode_attention(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"], worker_ns=ns)
        b.record()
        torch.cuda.synchronize()
        w = ns.cpu().numpy().astype(np.float64)
        t0 = w[:, 0].min()
        merged = w[:, 3].max() if w[:, 3].max() > 0 else w[:, 1].max()
        # slot 2: when a CTA's last wait for a record's parts ended (in-grid merge); it holds the SM id otherwise
        barrier = w[:, 2].max() if w[:, 2].max() >= t0 else w[:, 1].max()
        rows.append([(w[:, 0].max() - t0) / 1e3, (w[:, 1].min() - t0) / 1e3, (w[:, 1].max() - t0) / 1e3,
                     (barrier - t0) / 1e3, (merged - t0) / 1e3, a.elapsed_time(b) * 1e3])
    m = np.median(np.array(rows), axis=0)
    return {"last_cta_start_us": float(m[0]), "first_cta_out_of_work_us": float(m[1]), "last_cta_out_of_work_us": float(m[2]),
            "last_wait_passed_us": float(m[3]), "merges_done_us": float(m[4]), "cuda_event_us": float(m[5])}


def prepare(T, S, torch):
    wl, plan = S["wl"], S["plan"]
    t0 = time.perf_counter()
    S["dp"] = T.tangram_upload(S["tables"], plan)      # packs the blob on the host, one H2D copy, stream sync
    S["host_ms"]["upload_ms"] = (time.perf_counter() - t0) * 1e3
    S["out"] = torch.empty_like(S["q"])
    S["lse"] = torch.empty(wl.R, wl.Hq, dtype=torch.float32, device=S["q"].device)
    S["ws"] = torch.empty(T.tangram_workspace_bytes(plan.n_part_slots, wl.G, wl.d), dtype=torch.uint8,
                          device=S["q"].device)
    S["bytes"] = algorithmic_bytes(wl, S["kv"], plan, S["tables"])


def measure_config(T, I, name, device, steps, warmup, flush, torch, peak_gbs, compare=True, dyn=None, R=None,
                   page_size=None):
    """µs per layer-step, achieved TB/s, kernel-only roofline, spread, and the same kernel run from the
    BALANCED plan without its dynamic tail, from STATIC_EVEN and from SPLITMAP."""
    S = setup_workload(T, I, name, device, dyn=dyn, R=R, page_size=page_size)
    prepare(T, S, torch)
    step = lambda: T.tangram_decode_attention(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"])
    ms = time_steps(step, steps, warmup, flush, torch)
    kern = lambda: T.tangram_decode_partials(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"])
    kms = time_steps(kern, steps, min(warmup, 3), flush, torch)
    b = S["bytes"]
    us, us_min = float(np.median(ms) * 1e3), float(np.min(ms) * 1e3)
    kus = float(np.mean(kms) * 1e3)
    res = {"us_per_layer_step": us, "us_min": us_min, "us_mean": float(np.mean(ms) * 1e3),
           "tbs": b["total"] / (us * 1e-6) / 1e12,
           "pct_of_8tbs": 100 * b["total"] / (us * 1e-6) / 1e12 / NOMINAL_TBS,
           "pct_of_measured_copy": 100 * b["total"] / (us * 1e-6) / 1e9 / peak_gbs,
           "decode_kernel_us": kus, "decode_kernel_gbs": (b["total"] - b["partials"] // 2) / (kus * 1e-6) / 1e9,
           "algorithmic_bytes": b, "W": S["W"], "items": int(S["plan"].n_items), "granule": S["wl"].granule,
           "c0": S["c0"], "dyn_permille": S["dyn"][0], "dyn_rounds": S["dyn"][1], "host_ms": S["host_ms"],
           "cta_spread": spread_of(T, S, torch), "timeline": timeline_of(T, S, torch, flush)}
    # DRAM bytes of the committed ncu capture of this configuration / the kernel's algorithmic bytes (None: no capture
    # of the current sources); only for the configuration as BASELINE.json names it
    tr = profiled_traffic(name) if R is None and page_size is None else None
    res["traffic_ratio"] = tr / (b["total"] - b["partials"] // 2) if tr else None
    if compare:
        legs = [(T.MODE_STATIC_EVEN, "static_even"), (T.MODE_SPLITMAP, "splitmap")]
        if S["dyn"][1] > 0:                   # the same equal-bytes plan, every CTA owning exactly one list
            legs.insert(0, (T.MODE_BALANCED, "balanced_static"))
        for mode, key in legs:
            S2 = dict(S)
            S2["host_ms"] = dict(S["host_ms"])
            S2["plan"] = T.tangram_plan_partitions(S["tables"], S["B"], S["kv"], S["W"], S["wl"].granule, S["c0"], mode)
            prepare(T, S2, torch)
            f2 = lambda: T.tangram_decode_attention(S2["dp"], S2["q"], S2["pool"], S2["out"], S2["lse"], S2["ws"])
            m2 = time_steps(f2, max(10, steps // 4), 3, flush, torch)
            res[key] = {"us_per_layer_step": float(np.median(m2) * 1e3), "items": int(S2["plan"].n_items),
                        "split_map": S2["plan"].split_map.tolist(), "cta_spread": spread_of(T, S2, torch, 3),
                        "slowdown_vs_balanced": float(np.median(m2) * 1e3) / us}
            if key == "balanced_static":  # the evidence behind the dynamic tail: equal bytes per CTA != equal time
                res[key]["cta_spread"], res[key]["per_cta"] = spread_of(T, S2, torch, 4, detail=True)
    return S, res, ms, kms


def e2e_steps(T, S, steps, warmup, flush, torch, zero_copy):
    """Same step through the public API with HOST buffers: q comes from pinned host memory and the result
    (out, lse) ends up in pinned host memory inside the timed region.  The KV page pool is the resident state
    of the serving system (written by prefill, like weights) and stays in HBM.
    zero_copy=True: tangram_decode_attention_host -- out / lse are HOST pointers (pinned memory is mapped into the
    device's address space and the kernel's posted stores go over the bus, so the result never waits for a copy
    engine); q is pulled from pinned host memory by the decode kernel itself: the consumer warps of CTA b stage query
    blocks b, b + grid, ... into device memory when the CTA starts and publish per-block flags, a producer waits for
    the flag of the block its item needs -- one launch, every block crosses the bus once, and the KV tile rings fill
    meanwhile (reading q in place from host memory with the kernel's bulk copies is refused by the library: every
    work item would re-read its query group over the bus, and bulk copies from mapped host memory hang now and then).
    zero_copy=False: explicit staging copies around the call (one H2D, one D2H)."""
    q_host = S["q"].cpu().pin_memory()
    R, Hq, d = S["q"].shape
    n_out, n_lse = R * Hq * d * 2, R * Hq * 4
    res_host = torch.empty(n_out + n_lse, dtype=torch.uint8).pin_memory()
    if zero_copy:
        out_host = res_host[:n_out].view(torch.bfloat16).view(R, Hq, d)
        lse_host = res_host[n_out:].view(torch.float32).view(R, Hq)

        q_dev = torch.empty_like(S["q"])

        def step():          # ONE C-ABI call, ONE launch: the decode kernel stages q itself
            T.tangram_decode_attention_host(S["dp"], q_host, q_dev, S["pool"], out_host, lse_host, S["ws"])
    else:
        # out and lse live in ONE device allocation, so the result goes back with a single device->host copy
        res_dev = torch.empty(n_out + n_lse, dtype=torch.uint8, device=S["q"].device)
        out_dev = res_dev[:n_out].view(torch.bfloat16).view(R, Hq, d)
        lse_dev = res_dev[n_out:].view(torch.float32).view(R, Hq)
        q_dev = torch.empty_like(S["q"])

        def step():
            q_dev.copy_(q_host, non_blocking=True)
            T.tangram_decode_attention(S["dp"], q_dev, S["pool"], out_dev, lse_dev, S["ws"])
            res_host.copy_(res_dev, non_blocking=True)

    ms = time_steps(step, steps, warmup, flush, torch)
    torch.cuda.synchronize()
    # the result the host sees is the one the device-resident path computes
    T.tangram_decode_attention(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"])
    torch.cuda.synchronize()
    got = res_host[:n_out].view(torch.bfloat16).view(R, Hq, d)
    assert torch.equal(got, S["out"].cpu()), "e2e result differs from the device-resident result"
    return ms, q_host.numel() * 2, n_out + n_lse


def guarded(fn, timeout_s, on_timeout):
    """fn() with a watchdog thread: if it has not returned after timeout_s seconds (a launch that never completes
    cannot be cancelled from inside the process), on_timeout() runs on the watchdog thread."""
    import threading
    done = threading.Event()

    def watch():
        if not done.wait(timeout_s):
            on_timeout()

    threading.Thread(target=watch, daemon=True).start()
    try:
        return fn()
    finally:
        done.set()


def read_stream_peak(T, device, flush, torch, nbytes=4 << 30, reps=5):
    """Builder-measured ceiling of a read-only HBM stream: tangram_read_stream (16-byte loads on all SMs) over 4 GiB,
    L2 flushed, CUDA events; best of `reps`, in GB/s."""
    buf = torch.empty(nbytes, dtype=torch.uint8, device=device)
    buf.random_(0, 255)
    sink = torch.zeros(1, dtype=torch.int32, device=device)
    ms = time_steps(lambda: T.tangram_read_stream(buf, sink), reps, 3, flush, torch)
    del buf
    torch.cuda.empty_cache()
    return nbytes / (min(ms) * 1e-3) / 1e9


def table_update_summary(T, I, device, torch, names=("8b", "32b"), steps=48):
    """NEXT-4: cost of one block-table update of the whole batch (every (request, cluster) row checked, full rows
    handed a page) per decode step, at H_p = 1 / 2 / 4 / 8: the host path (tangram_extend_tables, 1 thread and the
    OpenMP default) and the device path (tangram_extend_tables_device, CUDA events).  The paper's Table 1 quotes
    5.64-17.13 ms of per-step planning for its dynamic baseline; its own block-table cost is
    only shown in Fig. 8(c) (image not available)."""
    out = {"unit": "us per update of the whole batch", "paper_table1_dynamic_planning_ms": [5.64, 17.13]}
    for name in names:
        wl = I.make_workload(name)
        B, res, kv0 = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
        for Hp in (1, 2, 4, 8):
            C = wl.H // Hp
            need = T.tangram_pages_needed(B, res, C, wl.P)
            headroom = steps // 16 + 2
            free = I.make_free_pages(wl, need + headroom * wl.R * C)
            host_us = {}
            for nt in (1, 0):
                t, kv = T.tangram_build_ragged_tables(B, res, C, wl.P, free, 0, kv0, headroom_pages=headroom)
                # the C call itself, arguments marshalled once (the binding's per-call numpy -> ctypes conversion
                # costs ~15 us, more than the update)
                import ctypes
                ct, cur, ts, ext = t._c(), np.ascontiguousarray(kv, dtype=np.int32).copy(), [], 0
                e_out, s_out = ctypes.c_int64(0), ctypes.c_int64(0)
                args = (ctypes.byref(ct), cur.ctypes.data_as(ctypes.c_void_p), free.ctypes.data_as(ctypes.c_void_p),
                        ctypes.c_int64(free.shape[0]), ctypes.c_int32(nt), ctypes.byref(e_out), ctypes.byref(s_out))
                for _ in range(steps):
                    t0 = time.perf_counter()
                    rc = T._lib.tangram_extend_tables(*args)
                    ts.append(time.perf_counter() - t0)
                    assert rc == 0
                    ext += int(e_out.value)
                    cur += 1
                host_us["1_thread" if nt == 1 else "openmp_default"] = float(np.median(ts) * 1e6)
            t, kv = T.tangram_build_ragged_tables(B, res, C, wl.P, free, 0, kv0, headroom_pages=headroom)
            pl = T.tangram_plan_partitions(t, B, kv, 8, wl.granule, 1, T.MODE_BALANCED)
            dp = T.tangram_upload(t, pl)
            kv_dev, free_dev = torch.as_tensor(kv, device=device), torch.as_tensor(free, device=device)
            evs = []
            for _ in range(steps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                T.tangram_extend_tables_device(dp, kv_dev, free_dev)
                b.record()
                kv_dev += 1
                evs.append((a, b))
            torch.cuda.synchronize()
            starved = T.tangram_download_tables(dp, t)
            out[f"{name}_Hp{Hp}"] = {"rows": wl.R * C, "host_us": host_us,
                                     "device_us": float(np.median([a.elapsed_time(b) for a, b in evs]) * 1e3),
                                     "pages_handed_out_host": int(ext), "rows_starved_device": int(starved)}
    return out


def tiny_oracle_one_thread(O, T, I, torch):
    """SURVEY §8(d) 'Oracle timing': the whole Tiny workload through the fp64 oracle on ONE thread, wall seconds."""
    S = setup_workload(T, I, "tiny", "cpu", W=4)
    wl = S["wl"]
    pairs = [(r, j) for r in range(wl.R) for j in range(wl.Hq)]
    best = 1e9
    for _ in range(5):
        dt, used = run_oracle_sample(O, S, S["q"], S["pool"], pairs, threads=1)
        best = min(best, dt)
    return {"seconds": best, "threads": 1, "rows": len(pairs), "token_visits": int(S["kv"].sum()) * wl.G}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="8b", choices=["tiny", "8b", "32b", "skew", "uniform", "12b_d256"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the other configs' summary lines")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-compact", action="store_true", help="skip the Top-k compaction (NEXT-2) summary")
    ap.add_argument("--dyn-permille", type=int, default=None, help="dynamic-tail share of the BALANCED plan")
    ap.add_argument("--dyn-rounds", type=int, default=None)
    ap.add_argument("--decode-loop-layers", type=int, default=8,
                    help="layers of the multi-layer decode loop summary (0 = skip)")
    ap.add_argument("--decode-loop-only", action="store_true",
                    help="after the timed steps run only the multi-layer decode loop summary (short runs under ncu)")
    ap.add_argument("--plumbing-only", action="store_true",
                    help="exercise only the multi-rank plumbing (spawn, rendezvous, barrier, aggregation) on CPU / gloo")
    args = ap.parse_args()
    if args.impl == "reference":
        reference_arm(args)
        return
    # --gpus N does what it says: under torchrun the world must have N ranks; started bare, N ranks are spawned here
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        sys.exit(spawn_ranks(args.gpus, sys.argv[1:]))
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE', '1')}")
    if args.plumbing_only:
        plumbing_only(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2606_06302_b200 import binding as T      # raises if libtangram.so is missing
    from paper_2606_06302_b200 import inputs as I

    rank, local_rank, world = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")      # the communicator log shows the ranks that really joined
        dist.init_process_group("nccl", device_id=torch.device(device))
    peak_gbs, peak_src = measured_peak()
    flush = L2Flusher(device)

    dyn = None if args.dyn_permille is None else (args.dyn_permille, args.dyn_rounds or 0)
    S = setup_workload(T, I, args.workload, device, dyn=dyn)
    prepare(T, S, torch)
    step = lambda: T.tangram_decode_attention(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"])
    for _ in range(args.warmup):
        flush()
        step()
    # ---- the timed region: exactly K steps, barrier + synchronize on both sides
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    with ClockSampler(local_rank) as clocks:
        wall0 = time.perf_counter()
        ms = time_steps(step, args.steps, 0, flush, torch)
        torch.cuda.synchronize()
        wall = time.perf_counter() - wall0
    if world > 1:
        dist.barrier()
    ms_step_local = float(np.mean(ms))
    b = S["bytes"]
    ms_step, total_bytes = aggregate(ms_step_local, float(b["total"]), world, device)
    tbs = total_bytes / (ms_step * 1e-3) / 1e12

    # ---- kernel-only roofline for the dominant kernel (split-KV decode kernel alone: it does not read the partials
    #      back, so half of the partial bytes -- the merge's reads -- are not counted for it)
    kern = lambda: T.tangram_decode_partials(S["dp"], S["q"], S["pool"], S["out"], S["lse"], S["ws"])
    kms = time_steps(kern, args.steps, 3, flush, torch)
    k_bytes = b["total"] - b["partials"] // 2
    k_gbs = k_bytes / (float(np.mean(kms)) * 1e-3) / 1e9
    # ---- end to end with host buffers.  The copy-engine variant first (it cannot hang); the zero-copy variant has the
    #      SMs read pinned host memory, which on one box of this pool hung now and then: on one
    #      GPU it runs below under a watchdog, once the rest of the line is known.
    ems_staged, h2d, d2h = e2e_steps(T, S, max(10, args.steps // 4), 3, flush, torch, zero_copy=False)
    e_ms_staged, e_bytes = aggregate(float(np.mean(ems_staged)), float(b["total"]), world, device)
    e_ms = None
    if world > 1:
        ems, h2d, d2h = e2e_steps(T, S, args.steps, 3, flush, torch, zero_copy=True)
        e_ms, e_bytes = aggregate(float(np.mean(ems)), float(b["total"]), world, device)

    def e2e_entry(zero_copy_ms, hung=False):
        ms_ = zero_copy_ms if zero_copy_ms is not None else e_ms_staged
        note = ("one tangram_decode_attention_host call (one launch) per step: q pulled from pinned host memory by "
                "the decode kernel's own consumer warps (per-block flags), out+lse written "
                "by the kernel straight into pinned, device-mapped host memory, all inside the timed region; "
                "`staged_copies` = the same with copy-engine transfers (one H2D before, one D2H after the call); "
                "the KV page pool is resident serving state in HBM")
        if zero_copy_ms is None:
            note = ("copy-engine transfers (one H2D of q before, one D2H of out+lse after tangram_decode_attention) inside "
                    "the timed region; the zero-copy variant (tangram_decode_attention_host) "
                    + ("did not come back within its watchdog time on this box" if hung else
                       "is timed last and was not reached in this mode")
                    + "; the KV page pool is resident serving state in HBM")
        return {"value": e_bytes / (ms_ * 1e-3) / 1e12, "unit": "TB/s", "us_per_layer_step": ms_ * 1e3,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "us_per_layer_step_staged_copies": e_ms_staged * 1e3, "zero_copy": zero_copy_ms is not None,
                "zero_copy_hung": bool(hung), "note": note}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    read_peak = read_stream_peak(T, device, flush, torch)
    line = {
        "metric": METRIC, "value": tbs, "unit": "TB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "us_per_layer_step": ms_step * 1e3,
        "us_per_layer_step_median": float(np.median(ms) * 1e3), "us_per_layer_step_min": float(np.min(ms) * 1e3),
        "pct_of_8tbs_nominal": 100 * tbs / world / NOMINAL_TBS,
        "pct_of_measured_copy_peak": 100 * tbs * 1e3 / world / peak_gbs,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": args.workload, "R": S["wl"].R, "Hq": S["wl"].Hq, "H": S["wl"].H, "d": S["wl"].d,
                   "page_size": S["wl"].P, "clusters": S["wl"].C, "plan": "balanced", "W": S["W"], "dyn_permille": S["dyn"][0],
                   "dyn_rounds": S["dyn"][1], "work_lists": int(S["plan"].W),
                   "granule": S["wl"].granule, "c0": S["c0"], "items": int(S["plan"].n_items),
                   "kv_bytes": b["kv"], "algorithmic_bytes": b["total"], "pool_bytes": S["pool"].numel() * 2,
                   "l2": "inputs larger than L2 and an L2 flush (256 MB write, then 256 MB read) before every timed step",
                   "multi_gpu": "replicas only (path shards by request, no collective)",
                   "host_ms": {k: round(v, 3) for k, v in S["host_ms"].items()}},
        "e2e": e2e_entry(e_ms),
        # one cooperative launch per step (the merge runs inside the decode grid); the stand-alone merge
        # kernel is only launched when the grid cannot be co-resident, which bench.py never asks for
        "gpu_launches": args.steps,
        "roofline": {"bound": "hbm", "kernel": "tangram_decode_kernel", "achieved": k_gbs, "peak": peak_gbs,
                     "unit": "GB/s", "frac": k_gbs / peak_gbs, "traffic": profiled_traffic(args.workload),
                     "peak_source": peak_src,
                     "kernel_us": float(np.mean(kms) * 1e3), "algorithmic_bytes_per_launch": k_bytes,
                     # the peak above is a read+write copy; this kernel only reads.  Builder-measured in this run:
                     "read_peak_gbs": read_peak, "frac_of_read_peak": k_gbs / read_peak,
                     "read_peak_how": "tangram_read_stream: 16-byte loads on all SMs over 4 GiB, L2 flushed, CUDA events, best of 5",
                     "step_frac_of_read_peak": tbs * 1e3 / world / read_peak},
        "clocks": clocks.summary(),
        "host_ms": S["host_ms"], "wall_s_timed_region": wall,
        "paper_context": "Tangram reports ratios only: up to 1.7x decode-attention inflation from static "
                         "partitioning (Qwen3-4B, A100-80GB, PAPER.md:120) and up to 2.6x end-to-end throughput over "
                         "full KV (4xA100-80GB, PAPER.md:13); no absolute us or TB/s to compare with",
    }
    line["cta_spread"] = spread_of(T, S, torch)
    line["config"]["cta_spread"] = round(line["cta_spread"], 4)
    if args.decode_loop_only and world == 1:
        del S
        torch.cuda.empty_cache()
        line["decode_loop"] = decode_loop(T, I, args.workload, device, args.decode_loop_layers or 2, 12, torch)
        emit(line)
        return
    if not args.no_sweep and world == 1:
        per = {}
        del S
        torch.cuda.empty_cache()
        # batch-4 8b-shaped: the paper's own decode-attention comparison point (Fig. 13: batch 4)
        sweep = [("tiny", None, None), ("8b", None, None), ("32b", None, None), ("skew", None, None), ("uniform", None, None),
                 ("12b_d256", None, None), ("8b_batch4", 4, None), ("8b_page32", None, 32)]
        for key, R, P in sweep:
            name = "8b" if key in ("8b_batch4", "8b_page32") else key
            S2, res, _, _ = measure_config(T, I, name, device, min(args.steps, 100), 5, flush, torch, peak_gbs, dyn=dyn, R=R,
                                           page_size=P)
            if key == args.workload and not args.no_cpu_baseline:
                from oracle import tangram_oracle as O
                O.build_c()
                line["cpu_baseline"] = cpu_baseline(O, S2)
            per[key] = res
            del S2
            torch.cuda.empty_cache()
        line["per_config"] = per
        # compact copy the driver's record keeps: [us per layer-step, TB/s, kernel GB/s, per-CTA spread,
        # BALANCED-without-dynamic-tail slowdown (x), STATIC_EVEN slowdown (x)]
        line["config"]["per_config_summary"] = {
            "columns": ["us", "tbs", "kernel_gbs", "cta_spread", "balanced_static_x", "static_even_x"],
            "timeline_columns": ["first CTA out of work", "last CTA out of work", "last wait for parts passed", "merges done",
                                 "CUDA events"],
            "timeline_us": {k: [round(v["timeline"][c], 1) for c in ("first_cta_out_of_work_us", "last_cta_out_of_work_us",
                                                                      "last_wait_passed_us", "merges_done_us", "cuda_event_us")]
                            for k, v in per.items()},
            **{k: [round(v["us_per_layer_step"], 2), round(v["tbs"], 3), round(v["decode_kernel_gbs"], 0),
                   round(v["cta_spread"], 4),
                   round(v["balanced_static"]["slowdown_vs_balanced"], 3) if "balanced_static" in v else None,
                   round(v["static_even"]["slowdown_vs_balanced"], 3)] for k, v in per.items()}}
        if args.decode_loop_layers > 0:
            dl = decode_loop(T, I, args.workload, device, args.decode_loop_layers, 36, torch)
            line["decode_loop"] = dl
            line["config"]["decode_loop"] = {"us_per_layer_step": round(dl["us_per_layer_step"], 2),
                                             "launches_per_layer_step": dl["launches_per_layer_step"],
                                             "overflow": dl["overflow"], "layers": dl["layers"],
                                             "two_launches_us": round(dl["two_launches"]["us_per_layer_step"], 2),
                                             "two_launches_overflow": dl["two_launches"]["overflow"]}
            torch.cuda.empty_cache()
        tu = table_update_summary(T, I, device, torch)
        line["table_update"] = tu
        line["config"]["table_update_us"] = {k: [round(v["host_us"]["1_thread"], 1), round(v["host_us"]["openmp_default"], 1),
                                                 round(v["device_us"], 1)]
                                             for k, v in tu.items() if isinstance(v, dict)}
        line["config"]["table_update_us"]["columns"] = ["host 1 thread", "host OpenMP", "device kernel"]
    elif not args.no_cpu_baseline and world == 1:
        from oracle import tangram_oracle as O
        O.build_c()
        S = setup_workload(T, I, args.workload, device)
        line["cpu_baseline"] = cpu_baseline(O, S)
    if world == 1 and "cpu_baseline" in line:
        from oracle import tangram_oracle as O
        t1 = tiny_oracle_one_thread(O, T, I, torch)
        line["cpu_baseline"]["tiny_1thread_s"] = t1["seconds"]
        line["cpu_baseline"]["tiny_1thread"] = t1
    if world == 1:
        line["page_accounting"] = page_accounting_summary(T, I, args.workload)
    if world == 1 and not args.no_compact:
        S = None
        torch.cuda.empty_cache()
        line["compact_topk"] = compact_topk_summary(T, I, args.workload, device, 30, flush, torch, peak_gbs)
        line["config"]["compact_topk"] = {"us": round(line["compact_topk"]["us"], 1),
                                          "pct_of_measured_copy": round(line["compact_topk"]["pct_of_measured_copy"], 1)}
    if world == 1:
        # Last of all, so that a launch that never comes back costs nothing but this figure: the zero-copy e2e leg on
        # a freshly set-up workload, under a watchdog that prints the finished line (e2e = the copy-engine variant).
        S = None
        torch.cuda.empty_cache()
        S = setup_workload(T, I, args.workload, device, dyn=dyn)
        prepare(T, S, torch)

        def give_up():
            line["e2e"] = e2e_entry(None, hung=True)      # e2e.zero_copy_hung = true: the fall-back is on the record
            emit(line)
            os._exit(0)
        ems = guarded(lambda: e2e_steps(T, S, args.steps, 3, flush, torch, zero_copy=True)[0], 180.0, give_up)
        line["e2e"] = e2e_entry(float(np.mean(ems)))
    emit(line)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
