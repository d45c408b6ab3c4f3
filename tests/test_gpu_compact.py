"""GPU parity of NEXT-2 (per-head Top-k selection, Eq. 4, and compaction into the ragged pages,
Eq. 1) against oracle O7.  Index and byte work: bit-exact, including every pool byte the
compaction must NOT touch."""
import math

import numpy as np
import pytest
import torch

from oracle import tangram_oracle as O
from paper_2606_06302_b200 import binding as T
from paper_2606_06302_b200 import inputs as I

pytestmark = pytest.mark.gpu


def bits(x):
    return x.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def otables(t):
    if getattr(t, "oracle_side", None) is not None:
        return t.oracle_side
    return O.Tables(R=t.R, H=t.H, C=t.C, Hp=t.Hp, P=t.P, perm=t.perm, cluster_of=t.cluster_of, slot_of=t.slot_of,
                    tbl_indptr=t.tbl_indptr, tbl_pages=t.tbl_pages, n_pages_used=t.n_pages_used)


def setup(wl):
    """Tables through the product's C ABI and, independently, through the oracle (bit-exact agreement asserted);
    the oracle later works on its own copy."""
    B, res, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    n_pool = int(math.ceil(1.05 * T.tangram_pages_needed(B, res, wl.C, wl.P))) + 1
    free = I.make_free_pages(wl, n_pool)
    t, kv = T.tangram_build_ragged_tables(B, res, wl.C, wl.P, free, 0, kv)
    Bo, reso, kvo = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    to, kvo = O.build_ragged_tables(Bo, reso, wl.C, wl.P, free, 0, kvo)
    assert np.array_equal(kvo, kv) and all(np.array_equal(getattr(to, f), getattr(t, f))
                                           for f in ("perm", "cluster_of", "slot_of", "tbl_indptr", "tbl_pages"))
    t.oracle_side = to          # the oracle's own, independently built tables
    pl = T.tangram_plan_partitions(t, B, kv, 8, wl.granule, 1, T.MODE_BALANCED)
    return B, res, kv, t, n_pool, T.tangram_upload(t, pl)


def run_and_compare(wl, t, dp, n_pool, keep, scores, kd, vd, n_max):
    _, pool = I.make_q_and_pool(wl, n_pool, "cuda")
    before = bits(pool).copy()
    keep_dev = torch.from_numpy(np.ascontiguousarray(keep, dtype=np.int32)).cuda()
    ctx_dev = torch.from_numpy(wl.ctx_len.astype(np.int32)).cuda()
    idx_out = torch.full((wl.R, wl.H, n_max), -7, dtype=torch.int32, device="cuda")
    clamped = torch.zeros(1, dtype=torch.int32, device="cuda")
    T.tangram_compact_topk(dp, scores, kd, vd, ctx_dev, keep_dev, pool, idx_out=idx_out, clamped=clamped)
    torch.cuda.synchronize()
    assert int(clamped.item()) == 0
    ref_pool, ref_idx = O.compact_topk(before, otables(t), scores.cpu().numpy(), bits(kd), bits(vd), wl.ctx_len, keep)
    got_idx = idx_out.cpu().numpy()
    for r in range(wl.R):
        for h in range(wl.H):
            k = int(keep[r][h])
            assert np.array_equal(got_idx[r, h, :k], ref_idx[r][h]), (r, h, k)
            assert np.all(got_idx[r, h, k:] == -7)                      # nothing written behind the retained set
    assert np.array_equal(bits(pool), ref_pool)                          # every byte, slack included
    return pool, ref_pool


@pytest.mark.parametrize("seed,R,H,d,C,max_ctx,ties", [(21, 3, 4, 128, 2, 3000, "bf16"), (22, 2, 6, 64, 3, 2500, "none"),
                                                       (23, 4, 2, 128, 1, 700, "bf16"), (24, 2, 8, 64, 8, 5000, "bf16"),
                                                       (25, 1, 4, 128, 4, 40, "none"), (28, 2, 4, 256, 2, 1800, "bf16"),
                                                       # rows long enough for clusters of 4 and 8 CTAs
                                                       (26, 2, 2, 64, 2, 40000, "bf16"), (27, 1, 2, 64, 1, 70000, "bf16")])
def test_compact_random_shapes_bit_exact(seed, R, H, d, C, max_ctx, ties):
    wl = I.make_random_workload(seed, R=R, H=H, G=1, d=d, C=C, max_ctx=max_ctx)
    if max_ctx > 10000:
        wl.ctx_len[0] = max_ctx - 5           # make sure the longest cluster shape is exercised
        wl.demand = np.minimum(wl.demand, wl.ctx_len[:, None]).astype(np.int32)
        wl.demand[0] = np.maximum(1, (wl.ctx_len[0] * np.linspace(0.02, 0.9, H))).astype(np.int32)
    B, res, kv, t, n_pool, dp = setup(wl)
    n_max = int(wl.ctx_len.max()) + 3
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda", ties=ties)
    run_and_compare(wl, t, dp, n_pool, kv, scores, kd, vd, n_max)


@pytest.mark.parametrize("overlap", ["0", "1"])
@pytest.mark.parametrize("seed,R,H,d,C,max_ctx", [(41, 40, 8, 128, 4, 900), (42, 3, 4, 64, 2, 6000), (43, 2, 4, 256, 2, 1200)])
def test_compact_select_and_gather_overlap_modes(monkeypatch, overlap, seed, R, H, d, C, max_ctx):
    """The gather is launched behind the select programmatically and waits row by row for ready flags.  Both
    queue orders / occupancies (TANGRAM_COMPACT_OVERLAP = 0: the select keeps every CTA, longest row first; 1: one
    select CTA per SM, shortest row first, the gather co-resident from the start) must give the oracle's bytes;
    320 rows make the select queue several waves deep.  Empty and fully retained rows are in the mix."""
    monkeypatch.setenv("TANGRAM_COMPACT_OVERLAP", overlap)
    wl = I.make_random_workload(seed, R=R, H=H, G=1, d=d, C=C, max_ctx=max_ctx)
    B, res, kv, t, n_pool, dp = setup(wl)
    keep = kv.copy()
    keep[0, 0] = 0                                     # a row that keeps nothing
    keep[R - 1, H - 1] = min(int(wl.ctx_len[R - 1]), int(keep[R - 1, H - 1]))
    n_max = int(wl.ctx_len.max()) + 1
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda", ties="bf16")
    for _ in range(2):                                 # the second call re-arms flags and counters from the first
        run_and_compare(wl, t, dp, n_pool, keep, scores, kd, vd, n_max)


def test_compact_edge_keeps_and_heavy_ties():
    """keep in {0, 1, N-1, N, page multiples}; scores with four distinct values only, +-0, +-inf."""
    wl = I.make_random_workload(31, R=3, H=4, G=1, d=64, C=2, max_ctx=1500)
    wl.ctx_len[:] = [1500, 1024, 33]
    wl.mu[:] = 1.0                                     # capacity = the whole context for every head
    wl.demand = np.array([[0, 1, 1499, 1500], [1024, 16, 17, 512], [33, 32, 31, 2]], dtype=np.int32)
    B, res, kv, t, n_pool, dp = setup(wl)
    assert np.array_equal(kv, wl.demand)
    n_max = 1504
    g = torch.Generator(device="cuda").manual_seed(5)
    scores = torch.randint(0, 4, (3, 4, n_max), generator=g, device="cuda").float()
    scores[0, 2, ::7] = 0.0
    scores[0, 2, 3::7] = -0.0
    scores[0, 3, 5] = math.inf
    scores[1, 3, 11::13] = -math.inf
    scores[1, 1] = 2.5                                 # all equal: the first 16 tokens win
    scores[2, 2] = -scores[2, 2]
    _, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    run_and_compare(wl, t, dp, n_pool, kv, scores, kd, vd, n_max)


def test_compact_clamps_to_capacity_and_counts():
    """:176 -- the reserved budget is a hard capacity bound: a keep beyond min(N_r, pages x P) is clamped and
    counted (the oracle refuses such a call; with the clamped value the two agree bit for bit)."""
    wl = I.make_random_workload(41, R=2, H=4, G=1, d=128, C=2, max_ctx=900)
    B, res, kv, t, n_pool, dp = setup(wl)
    n_max = int(wl.ctx_len.max())
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    cap = np.zeros_like(kv)
    for r in range(wl.R):
        for h in range(wl.H):
            row = r * t.C + int(t.cluster_of[h])
            cap[r, h] = min(int(wl.ctx_len[r]), int(t.tbl_indptr[row + 1] - t.tbl_indptr[row]) * t.P)
    want = kv.copy()
    want[0, 1] = cap[0, 1] + 5
    want[1, 2] = 10 ** 9
    want[1, 0] = -3
    with pytest.raises(ValueError):
        O.compact_topk(np.zeros((n_pool, t.Hp, 2, t.P, wl.d), np.uint16), otables(t), scores.cpu().numpy(), bits(kd),
                       bits(vd), wl.ctx_len, np.maximum(want, 0))
    _, pool = I.make_q_and_pool(wl, n_pool, "cuda")
    before = bits(pool).copy()
    clamped = torch.zeros(1, dtype=torch.int32, device="cuda")
    idx = T.tangram_compact_topk(dp, scores, kd, vd, torch.from_numpy(wl.ctx_len).cuda(),
                                 torch.from_numpy(want.astype(np.int32)).cuda(), pool, clamped=clamped)
    torch.cuda.synchronize()
    assert int(clamped.item()) == 3
    eff = np.clip(want, 0, cap)
    ref_pool, ref_idx = O.compact_topk(before, otables(t), scores.cpu().numpy(), bits(kd), bits(vd), wl.ctx_len, eff)
    assert np.array_equal(bits(pool), ref_pool)
    assert np.array_equal(idx.cpu().numpy()[1, 2, :eff[1, 2]], ref_idx[1][2])


def test_compact_then_decode_attention_matches_oracle_pipeline():
    """The step before the path feeding the path: compaction (CUDA) -> decode attention (CUDA) against
    oracle compaction -> oracle attention."""
    wl = I.make_workload("8b", R=3, ctx_div=8)
    B, res, kv, t, n_pool = setup(wl)[:5]
    W = T.tangram_query_max_ctas(0, wl.d, wl.G)
    pl = T.tangram_plan_partitions(t, B, kv, W, wl.granule, 1, T.MODE_BALANCED, 0, T.DEFAULT_DYN_PERMILLE,
                                   T.DEFAULT_DYN_ROUNDS)
    dp = T.tangram_upload(t, pl)
    n_max = int(wl.ctx_len.max())
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    pool, ref_pool = run_and_compare(wl, t, dp, n_pool, kv, scores, kd, vd, n_max)
    q, _ = I.make_q_and_pool(wl, 1, "cuda")
    out, lse = T.tangram_decode_attention(dp, q, pool)
    torch.cuda.synchronize()
    ref_out, ref_lse, _ = O.attention(q.cpu(), torch.from_numpy(ref_pool.view(np.int16)).view(torch.bfloat16),
                                      otables(t), kv, wl.Hq, wl.d)
    got = out.float().cpu().numpy().astype(np.float64)
    assert np.abs(got - ref_out).max() <= 2e-2
    assert np.linalg.norm(got - ref_out) / np.linalg.norm(ref_out) <= 5e-3
    assert np.abs(lse.cpu().numpy() - ref_lse).max() <= 1e-3


def test_compact_full_size_every_row_and_properties():
    """8b at BASELINE size (bench.py's configuration): the index set of EVERY (request, head) against the oracle;
    and for every head the properties that hold at any size -- ascending unique indices below N_r, every kept
    score >= every dropped score, ties resolved towards the lower index, pool rows = dense rows at I."""
    wl = I.make_workload("8b")
    B, res, kv, t, n_pool, dp = setup(wl)
    n_max = int(wl.ctx_len.max())
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    pool = torch.zeros(n_pool, t.Hp, 2, t.P, wl.d, dtype=torch.bfloat16, device="cuda")
    idx = T.tangram_compact_topk(dp, scores, kd, vd, torch.from_numpy(wl.ctx_len).cuda(),
                                 torch.from_numpy(kv.astype(np.int32)).cuda(), pool)
    torch.cuda.synchronize()
    sc = scores.cpu().numpy()
    ix = idx.cpu().numpy()
    for r in range(wl.R):
        N = int(wl.ctx_len[r])
        for h in range(wl.H):
            k = int(kv[r, h])
            I_ = ix[r, h, :k].astype(np.int64)
            assert np.all(np.diff(I_) > 0) and (k == 0 or (I_[0] >= 0 and I_[-1] < N))
            keep_mask = np.zeros(N, bool)
            keep_mask[I_] = True
            s = sc[r, h, :N]
            if 0 < k < N:
                thr = s[keep_mask].min()
                assert thr >= s[~keep_mask].max()
                tie = np.flatnonzero(s == thr)
                kept_tie = keep_mask[tie]
                assert np.all(kept_tie[:kept_tie.sum()])               # the kept ties are the lowest indices
            assert np.array_equal(I_, O.topk_indices(s, k)), (r, h)
            # pool rows = dense rows at I (Eq. 1), checked on the device
            row = r * t.C + int(t.cluster_of[h])
            pages = torch.from_numpy(t.tbl_pages[int(t.tbl_indptr[row]):int(t.tbl_indptr[row]) + (k + t.P - 1) // t.P]
                                     .astype(np.int64)).cuda()
            sl = int(t.slot_of[h])
            got_k = pool[pages, sl, 0].reshape(-1, wl.d)[:k]
            got_v = pool[pages, sl, 1].reshape(-1, wl.d)[:k]
            It = torch.from_numpy(I_).cuda()
            assert torch.equal(got_k, kd[r, h, It]) and torch.equal(got_v, vd[r, h, It])


# ---------------------------------------------------------------------------- NEXT-4: implicit ratios (Eq. 3)
@pytest.mark.parametrize("seed,R,H,n_max,ties", [(51, 3, 4, 700, True), (52, 2, 8, 3001, False), (53, 1, 2, 45000, True),
                                                 (54, 4, 3, 64, True)])
def test_implicit_ratios_bit_exact(seed, R, H, n_max, ties):
    g = torch.Generator(device="cuda").manual_seed(seed)
    scores = torch.randn(R, H, n_max, generator=g, device="cuda").exp_()
    scores *= torch.linspace(0.5, 2.0, H, device="cuda")[None, :, None]       # heads of different importance
    if ties:
        scores = scores.bfloat16().float()
    rng = np.random.default_rng(seed)
    ctx = rng.integers(max(1, n_max // 3), n_max + 1, size=R).astype(np.int32)
    ctx[0] = n_max
    ctx_dev = torch.from_numpy(ctx).cuda()
    for rho in (0.0, 0.3, 0.5, 1.0, 1e-9):
        cnt, rat = T.tangram_implicit_ratios(scores, ctx_dev, rho)
        torch.cuda.synchronize()
        ref_cnt, ref_rat = O.implicit_ratios(scores.cpu().numpy(), ctx, rho)
        assert np.array_equal(cnt.cpu().numpy(), ref_cnt), rho
        assert rat.cpu().numpy().tobytes() == ref_rat.tobytes(), rho


def test_calibration_pipeline_scores_to_budgets():
    """Offline calibration end to end (:156-158): scores of 12 sample contexts -> Eq. 3 implicit ratios (CUDA) ->
    mu, sigma, B (host C++) against the same chain through the oracle; the budgets then drive a1."""
    H, n_max, n_samples, rho = 8, 2048, 12, 0.3
    g = torch.Generator(device="cuda").manual_seed(77)
    head_gain = torch.tensor([0.3, 0.5, 3.0, 0.4, 0.6, 2.5, 0.5, 0.7], device="cuda")   # two "retrieval" heads
    scores = (torch.randn(n_samples, H, n_max, generator=g, device="cuda").exp_() * head_gain[None, :, None]).bfloat16().float()
    ctx = np.random.default_rng(3).integers(700, n_max + 1, size=n_samples).astype(np.int32)
    _, rat = T.tangram_implicit_ratios(scores, torch.from_numpy(ctx).cuda(), rho)
    torch.cuda.synchronize()
    mu, sigma, B = T.tangram_calibrate_budgets(rat.cpu().numpy(), 2.0)
    _, ref_rat = O.implicit_ratios(scores.cpu().numpy(), ctx, rho)
    mo, so, Bo = O.calibrate_budgets(ref_rat, 2.0)
    assert mu.tobytes() == mo.tobytes() and sigma.tobytes() == so.tobytes() and B.tobytes() == Bo.tobytes()
    assert abs(mu.mean() - rho) < 1e-3                      # Eq. 3 keeps the global budget: mean_h mu_h = rho (+ ceil)
    assert set(np.argsort(B)[-2:]) == {2, 5}                # the high-gain heads get the large budgets
    B2, res, _ = T.tangram_reserve_budgets(mu, sigma, 2.0, np.array([4096], dtype=np.int32))
    assert B2.tobytes() == B.tobytes() and res.sum() >= math.ceil(rho * H * 4096) - H


def test_compact_topk_is_graph_capturable_and_repeatable():
    """Three launches, no host work: captured once, replayed on fresh pools, same bytes every time."""
    wl = I.make_random_workload(61, R=3, H=4, G=1, d=128, C=2, max_ctx=2000)
    B, res, kv, t, n_pool, dp = setup(wl)
    n_max = int(wl.ctx_len.max())
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    _, pool0 = I.make_q_and_pool(wl, n_pool, "cuda")
    pool = pool0.clone()
    keep = torch.from_numpy(kv.astype(np.int32)).cuda()
    ctx = torch.from_numpy(wl.ctx_len).cuda()
    idx = torch.empty(wl.R, wl.H, n_max, dtype=torch.int32, device="cuda")
    need = T.tangram_compact_workspace_bytes(wl.R, wl.H)
    ws_guarded = torch.full((need + 512,), 0xAB, dtype=torch.uint8, device="cuda")   # 256-byte guards on both sides
    ws = ws_guarded[256:256 + need]
    T.tangram_compact_topk(dp, scores, kd, vd, ctx, keep, pool, idx_out=idx, workspace=ws)
    torch.cuda.synchronize()
    assert bool((ws_guarded[:256] == 0xAB).all()) and bool((ws_guarded[256 + need:] == 0xAB).all())
    want = bits(pool).copy()
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            T.tangram_compact_topk(dp, scores, kd, vd, ctx, keep, pool, idx_out=idx, workspace=ws, stream=st)
        for _ in range(3):
            pool.copy_(pool0)
            g.replay()
            st.synchronize()
            assert np.array_equal(bits(pool), want)
    torch.cuda.current_stream().wait_stream(st)


def test_random_sweep_compaction_and_implicit_ratios():
    """100 seeded cases (shapes, unaligned n_max, three score distributions incl. five-valued scores, empty heads):
    index lists, every pool byte, implicit-ratio counts and fp64 ratios bit-exact against the oracle."""
    rng = np.random.default_rng(20260631)
    for case in range(100):
        H, d = int(rng.choice([1, 2, 4, 8])), int(rng.choice([64, 128, 256]))
        C = int(rng.choice([c for c in (1, 2, 4, 8) if H % c == 0]))
        R = int(rng.integers(1, 4))
        wl = I.make_random_workload(int(rng.integers(1 << 30)), R=R, H=H, G=1, d=d, C=C,
                                    max_ctx=int(rng.choice([20, 200, 1100, 2100, 6000])),
                                    P=int(rng.choice([16, 32])) if d <= 128 else 16)
        if rng.random() < 0.3:
            wl.demand[rng.integers(R), rng.integers(H)] = 0
        B, res, kv, t, n_pool, dp = setup(wl)
        n_max = int(wl.ctx_len.max()) + int(rng.integers(0, 5))
        g = torch.Generator(device="cuda").manual_seed(int(rng.integers(1 << 30)))
        kind = int(rng.integers(3))
        if kind == 0:
            scores = torch.randn(R, H, n_max, generator=g, device="cuda")
        elif kind == 1:
            scores = torch.randint(-2, 3, (R, H, n_max), generator=g, device="cuda").float()
        else:
            scores = torch.randn(R, H, n_max, generator=g, device="cuda").exp().bfloat16().float()
        _, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
        run_and_compare(wl, t, dp, n_pool, kv, scores, kd, vd, n_max)
        rho = float(rng.choice([0.0, 0.1, 0.37, 1.0]))
        cnt, rat = T.tangram_implicit_ratios(scores, torch.from_numpy(wl.ctx_len).cuda(), rho)
        ref_cnt, ref_rat = O.implicit_ratios(scores.cpu().numpy(), wl.ctx_len, rho)
        assert np.array_equal(cnt.cpu().numpy(), ref_cnt) and rat.cpu().numpy().tobytes() == ref_rat.tobytes(), case


@pytest.mark.parametrize("seed,d,C,P", [(81, 128, 2, 16), (82, 64, 4, 16), (83, 256, 1, 16), (84, 128, 2, 32), (85, 64, 1, 32)])
def test_chunked_prefill_compaction_bit_exact(seed, d, C, P):
    """Compression fused into chunked prefill (:152): four chunks of ragged lengths compressed one after the other,
    each appended behind the previous ones (chunk boundaries fall inside pages); pool, lengths and index lists
    bit-exact against oracle O11 after every chunk; then decode attention over the result; then an over-full
    chunk is clamped and counted."""
    R, H = 3, 4
    rng = np.random.default_rng(seed)
    wl = I.make_random_workload(seed, R=R, H=H, G=2, d=d, C=C, max_ctx=100, P=P)
    chunk_lens = [rng.integers(1, 700, size=R).astype(np.int32) for _ in range(4)]
    ratios = rng.uniform(0.05, 1.0, size=H)
    keeps = [np.minimum(cl[:, None], np.ceil(cl[:, None] * ratios[None, :] * rng.uniform(0.5, 1.0, size=(R, H)))).astype(np.int32)
             for cl in chunk_lens]
    keeps[1][0, 1] = 0
    total = sum(keeps)
    B = np.clip(total.max(0) / sum(chunk_lens).max(), 0.01, 1.0)
    need = T.tangram_pages_needed(B, total, C, P)
    t, _ = T.tangram_build_ragged_tables(B, total, C, P, np.random.default_rng(seed).permutation(need + 3).astype(np.int32))
    pl = T.tangram_plan_partitions(t, B, total, 148, 64, 1, T.MODE_BALANCED, 0, T.DEFAULT_DYN_PERMILLE, T.DEFAULT_DYN_ROUNDS)
    dp = T.tangram_upload(t, pl)
    g = torch.Generator(device="cuda").manual_seed(seed)
    pool = torch.randn(need + 3, t.Hp, 2, P, d, generator=g, device="cuda").bfloat16()
    ref_pool, ref_kv = bits(pool).copy(), np.zeros((R, H), dtype=np.int32)
    kv_dev = torch.zeros(R, H, dtype=torch.int32, device="cuda")
    clamped = torch.zeros(1, dtype=torch.int32, device="cuda")
    for cl, kp in zip(chunk_lens, keeps):
        n_max = int(cl.max()) + 1
        scores = torch.randn(R, H, n_max, generator=g, device="cuda").exp().bfloat16().float()
        kd = torch.randn(R, H, n_max, d, generator=g, device="cuda").bfloat16()
        vd = torch.randn(R, H, n_max, d, generator=g, device="cuda").bfloat16()
        idx = torch.full((R, H, n_max), -7, dtype=torch.int32, device="cuda")
        T.tangram_compact_topk_chunk(dp, scores, kd, vd, torch.from_numpy(cl).cuda(), torch.from_numpy(kp).cuda(), kv_dev,
                                     pool, idx_out=idx, clamped=clamped)
        torch.cuda.synchronize()
        ref_pool, ref_kv, ref_idx = O.compact_topk_chunk(ref_pool, otables(t), scores.cpu().numpy(), bits(kd), bits(vd), cl,
                                                         kp, ref_kv)
        assert np.array_equal(bits(pool), ref_pool) and np.array_equal(kv_dev.cpu().numpy(), ref_kv)
        gi = idx.cpu().numpy()
        for r in range(R):
            for h in range(H):
                assert np.array_equal(gi[r, h, :kp[r, h]], ref_idx[r][h]) and (gi[r, h, kp[r, h]:] == -7).all()
    assert int(clamped.item()) == 0 and np.array_equal(ref_kv, total)
    q = torch.randn(R, H * 2, d, generator=g, device="cuda").bfloat16()
    out, lse = T.tangram_decode_attention(dp, q, pool)
    torch.cuda.synchronize()
    ref_out, ref_lse, _ = O.attention(q.cpu(), pool.cpu(), otables(t), total, H * 2, d)
    got = out.float().cpu().numpy().astype(np.float64)
    assert np.abs(got - ref_out).max() <= 2e-2 and np.linalg.norm(got - ref_out) / np.linalg.norm(ref_out) <= 5e-3
    assert np.abs(lse.cpu().numpy() - ref_lse).max() <= 1e-3
    # one more chunk does not fit any more: every head is clamped to the room its table has left (:176)
    rows = np.arange(R)[:, None] * t.C + t.cluster_of[None, :]
    room = ((t.tbl_indptr[rows + 1] - t.tbl_indptr[rows]) * P - total).astype(np.int32)
    cl, kp = chunk_lens[0], np.minimum(chunk_lens[0][:, None], room + 5).astype(np.int32)
    eff = np.minimum(kp, room)
    T.tangram_compact_topk_chunk(dp, scores[:, :, :int(cl.max())].contiguous(), kd[:, :, :int(cl.max())].contiguous(),
                                 vd[:, :, :int(cl.max())].contiguous(), torch.from_numpy(cl).cuda(),
                                 torch.from_numpy(kp).cuda(), kv_dev, pool, clamped=clamped)
    torch.cuda.synchronize()
    assert int(clamped.item()) == int((eff != kp).sum()) and np.array_equal(kv_dev.cpu().numpy(), total + eff)


def test_global_flat_topk_compression_as_a_composition():
    """The non-uniform compressor of Eq. 3 run on the device: implicit per-head counts (tangram_implicit_ratios)
    fed as `keep` into the per-head compaction reproduce the global flat Top-k selection (oracle: one flat sort)."""
    wl = I.make_random_workload(91, R=3, H=4, G=1, d=64, C=1, max_ctx=1500)
    wl.mu[:] = 1.0                                        # tables sized for the whole context: any split fits
    wl.demand = np.repeat(wl.ctx_len[:, None], wl.H, 1).astype(np.int32)
    B, res, kv, t, n_pool, dp = setup(wl)
    n_max = int(wl.ctx_len.max())
    scores, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    scores *= torch.tensor([0.4, 1.0, 2.5, 0.7], device="cuda")[None, :, None]
    ctx_dev = torch.from_numpy(wl.ctx_len).cuda()
    cnt, _ = T.tangram_implicit_ratios(scores, ctx_dev, 0.3)
    _, pool = I.make_q_and_pool(wl, n_pool, "cuda")
    idx = T.tangram_compact_topk(dp, scores, kd, vd, ctx_dev, cnt, pool)
    torch.cuda.synchronize()
    sc, gi, c = scores.cpu().numpy(), idx.cpu().numpy(), cnt.cpu().numpy()
    for r in range(wl.R):
        N = int(wl.ctx_len[r])
        flat = np.concatenate([sc[r, h, :N] for h in range(wl.H)])
        sel = O.topk_indices(flat, int(math.ceil(0.3 * wl.H * N)))
        assert c[r].sum() == len(sel)
        for h in range(wl.H):
            mine = sel[(sel >= h * N) & (sel < (h + 1) * N)] - h * N
            assert np.array_equal(gi[r, h, :c[r, h]], mine)


def test_select_paths_buffered_and_fallback():
    """The select kernel buffers the entries that share the threshold's first radix digit when there are at most
    4096 of them, and falls back to whole-row passes otherwise: rows of 9 000 - 20 000 tokens with all-equal scores,
    three-valued scores (fallback), well-spread scores (buffered), and a row whose candidates are exactly the
    buffer size."""
    wl = I.make_random_workload(95, R=5, H=2, G=1, d=64, C=1, max_ctx=100)
    wl.ctx_len[:] = [9000, 20000, 12000, 4096, 16000]
    wl.mu[:] = 1.0
    wl.demand = (wl.ctx_len[:, None] * np.array([[0.3, 0.77]])).astype(np.int32)
    B, res, kv, t, n_pool, dp = setup(wl)
    n_max = 20000
    g = torch.Generator(device="cuda").manual_seed(95)
    scores = torch.randn(wl.R, wl.H, n_max, generator=g, device="cuda")
    scores[0] = 1.25                                                               # all equal: N candidates
    scores[1] = torch.randint(0, 3, (wl.H, n_max), generator=g, device="cuda").float()   # ~6 700 per value
    scores[3] = 3.0                                                                # exactly 4096 candidates
    scores[4, 0] = scores[4, 0].bfloat16().float()                                 # bf16-rounded normal scores
    _, kd, vd = I.make_scores_and_dense_kv(wl, n_max, "cuda")
    run_and_compare(wl, t, dp, n_pool, kv, scores, kd, vd, n_max)
