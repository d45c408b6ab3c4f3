"""tangram_decode_attention_static -- decode attention for callers that cannot allocate device memory.

Who needs it: a serving engine calls decode attention once per layer and step, long after it has handed every free
byte of HBM to its KV page pool, and a cudaMalloc in that loop would stall the whole device anyway; an attention
plug-in living under another component's allocator is in the same position.  Such a caller owns q, the pool, out and
lse, but has no split-KV workspace to pass.  The entry point takes the workspace from a fixed 8 MiB array inside the
library (one per GPU, shared by all calls, never cleared) and allocates nothing.

What is checked here, through the C ABI:
  * its output equals the ordinary path's (tangram_decode_attention with a caller workspace) within the tolerances
    every parity test uses -- and both equal the oracle's -- on two calls in a row with DIFFERENT queries, so a second
    call that picked up partials left behind by the first would be caught;
  * the array really is shared and really is reused: a different plan (other partition, other part count) runs through
    it in between and afterwards the first plan still gives the right answer;
  * a plan whose partials do not fit the array is refused with BUFFER_TOO_SMALL and a message that names the static
    workspace, and the outputs are not touched.

The file is named so that pytest collects it last: under `-x` a failure here cannot hide another test.  It keeps no
state between tests and needs none from the tests before it (it passes alone in a fresh process and at the end of the
suite alike)."""
import math

import numpy as np
import pytest
import torch

from oracle import tangram_oracle as O
from paper_2606_06302_b200 import binding as T
from paper_2606_06302_b200 import inputs as I

pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2, LSE_TOL = 2e-2, 5e-3, 1e-3      # BASELINE.json's tolerances, as in tests/test_gpu_parity.py


def _tables(wl):
    B, res, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    n_pool = int(math.ceil(1.05 * T.tangram_pages_needed(B, res, wl.C, wl.P)))
    free = I.make_free_pages(wl, n_pool)
    t, kv = T.tangram_build_ragged_tables(B, res, wl.C, wl.P, free, 0, kv)
    Bo, reso, kvo = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    to, kvo = O.build_ragged_tables(Bo, reso, wl.C, wl.P, free, 0, kvo)      # the oracle's own tables
    assert np.array_equal(kvo, kv) and np.array_equal(to.tbl_pages, t.tbl_pages)
    return B, kv, t, to, n_pool


def _close(out, lse, ref_out, ref_lse, what):
    out = out.float().cpu().numpy().astype(np.float64).reshape(ref_out.shape)
    lse = lse.float().cpu().numpy().astype(np.float64).reshape(ref_lse.shape)
    ref_out, ref_lse = np.asarray(ref_out, np.float64), np.asarray(ref_lse, np.float64)
    assert np.all(np.isfinite(out)), what
    err = np.abs(out - ref_out).max()
    rel = np.linalg.norm(out - ref_out) / max(np.linalg.norm(ref_out), 1e-30)
    assert np.array_equal(np.isneginf(lse), np.isneginf(ref_lse)), what
    fin = np.isfinite(ref_lse)
    dl = np.abs(lse[fin] - ref_lse[fin]).max() if fin.any() else 0.0
    assert err <= MAX_ABS and rel <= REL_L2 and dl <= LSE_TOL, f"{what}: max|err|={err:.3e} relL2={rel:.3e} dLSE={dl:.3e}"


def test_static_workspace_matches_the_ordinary_path_on_consecutive_calls():
    wl = I.make_workload("8b", R=4, ctx_div=8)          # many tiles per item, ragged tails, multi-part sequences
    B, kv, t, to, n_pool = _tables(wl)
    q1, pool = I.make_q_and_pool(wl, n_pool, "cuda")
    g = torch.Generator(device="cpu").manual_seed(20260611)
    q2 = torch.randn(q1.shape, generator=g, dtype=torch.float32).to(torch.bfloat16).cuda()
    W = T.tangram_query_max_ctas(0, wl.d, wl.G)
    plan_a = T.tangram_plan_partitions(t, B, kv, W, wl.granule, 1, T.MODE_BALANCED, 0, 300, 3)
    plan_b = T.tangram_plan_partitions(t, B, kv, 7, wl.granule, 1, T.MODE_STATIC_EVEN, 4)
    assert plan_a.n_part_slots > 0 and plan_b.n_part_slots > 0 and plan_a.n_part_slots != plan_b.n_part_slots
    G = wl.Hq // wl.H
    assert T.tangram_workspace_bytes(plan_a.n_part_slots, G, wl.d) <= T.STATIC_WORKSPACE_BYTES
    dp_a, dp_b = T.tangram_upload(t, plan_a), T.tangram_upload(t, plan_b)

    # two calls in a row on one plan, different queries; then another plan through the same array; then the first again
    for step, (dp, q) in enumerate(((dp_a, q1), (dp_a, q2), (dp_b, q1), (dp_a, q1))):
        got_out, got_lse = T.tangram_decode_attention_static(dp, q, pool)
        torch.cuda.synchronize()
        want_out, want_lse = T.tangram_decode_attention(dp, q, pool)        # the existing path, caller's workspace
        torch.cuda.synchronize()
        _close(got_out, got_lse, want_out.float().cpu().numpy(), want_lse.cpu().numpy(), f"call {step}: static vs ordinary path")
        ref_out, ref_lse, _ = O.attention(q.cpu(), pool.cpu(), to, kv, wl.Hq, wl.d)
        _close(got_out, got_lse, ref_out, ref_lse, f"call {step}: static vs oracle")


def test_static_workspace_with_runtime_lengths_and_caller_outputs():
    """Open-ended plan (run-time lengths on the device) and out / lse supplied by the caller: with those, not even
    the Python wrapper allocates."""
    wl = I.make_random_workload(5, R=3, H=4, G=2, d=64, C=2, max_ctx=700)
    B, kv, t, to, n_pool = _tables(wl)
    q, pool = I.make_q_and_pool(wl, n_pool, "cuda")
    pl = T.tangram_plan_partitions(t, B, kv, 40, wl.granule, 1, T.MODE_BALANCED, 0, 0, 0)
    dp = T.tangram_upload(t, pl)
    shorter = np.maximum(kv // 2, 0).astype(np.int32)
    kv_dev = torch.from_numpy(shorter).cuda()
    out = torch.full((wl.R, wl.Hq, wl.d), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((wl.R, wl.Hq), float("nan"), dtype=torch.float32, device="cuda")
    for _ in range(2):
        T.tangram_decode_attention_static(dp, q, pool, out=out, lse=lse, kv_len=kv_dev)
        torch.cuda.synchronize()
        want_out, want_lse = T.tangram_decode_attention(dp, q, pool, kv_len=kv_dev)
        torch.cuda.synchronize()
        _close(out, lse, want_out.float().cpu().numpy(), want_lse.cpu().numpy(), "static vs ordinary path, run-time lengths")
        ref_out, ref_lse, _ = O.attention(q.cpu(), pool.cpu(), to, shorter, wl.Hq, wl.d)
        _close(out, lse, ref_out, ref_lse, "static vs oracle, run-time lengths")


def test_static_workspace_refuses_a_plan_beyond_its_limit():
    wl = I.make_workload("8b")                           # host planning only: no full-size pool is made
    B, kv, t, to, n_pool = _tables(wl)
    pl = T.tangram_plan_partitions(t, B, kv, 148, wl.granule, 1, T.MODE_STATIC_EVEN, 32)
    G = wl.Hq // wl.H
    assert T.tangram_workspace_bytes(pl.n_part_slots, G, wl.d) > T.STATIC_WORKSPACE_BYTES
    dp = T.tangram_upload(t, pl)
    q = torch.zeros(wl.R, wl.Hq, wl.d, dtype=torch.bfloat16, device="cuda")
    pool = torch.zeros(1, wl.Hp, 2, wl.P, wl.d, dtype=torch.bfloat16, device="cuda")   # refused before the pool is looked at
    out = torch.full((wl.R, wl.Hq, wl.d), 7.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.full((wl.R, wl.Hq), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(T.TangramError) as ei:
        T.tangram_decode_attention_static(dp, q, pool, out=out, lse=lse)
    assert ei.value.code == T.ERR_BUFFER_TOO_SMALL and "static workspace" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all()) and bool((lse == 7.0).all())           # nothing was launched
