"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no product
code).  Each pin is chosen so that a plausible mistake in the oracle (dropped term, wrong sign
or index, transposed operand, wrong scale) fails at least one of them.  SURVEY.md §8(c) "Pins".
"""
import itertools
import json
import math
import os

import numpy as np
import pytest
import torch

from oracle import tangram_oracle as O
from paper_2606_06302_b200 import inputs as I

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_examples.json")))


def bf16(x):
    return torch.as_tensor(np.asarray(x), dtype=torch.float32).bfloat16()


# ---------------------------------------------------------------------------- helpers
def scatter_dense_into_pool(K, V, kv_len, t, n_pool_pages, fill=None, seed=0):
    """Independent inverse of the oracle's gather: write dense K,V [R][H][n][d] (bf16 tensors)
    page by page into a pool laid out [page][slot][kv][token][d].  Unwritten slots get random
    garbage (or `fill`)."""
    R, H, P = t.R, t.H, t.P
    d = K[0][0].shape[-1]
    g = torch.Generator().manual_seed(seed)
    pool = torch.randn(n_pool_pages, t.Hp, 2, P, d, generator=g).bfloat16()
    if fill is not None:
        pool[:] = fill
    for r in range(R):
        for h in range(H):
            n = int(kv_len[r][h])
            row = t.tbl_pages[t.tbl_indptr[r * t.C + t.cluster_of[h]]:
                              t.tbl_indptr[r * t.C + t.cluster_of[h] + 1]]
            for pi in range((n + P - 1) // P):
                lo, hi = pi * P, min(n, (pi + 1) * P)
                pool[int(row[pi]), int(t.slot_of[h]), 0, :hi - lo] = K[r][h][lo:hi]
                pool[int(row[pi]), int(t.slot_of[h]), 1, :hi - lo] = V[r][h][lo:hi]
    return pool


def simple_tables(kv_len, H, C, P, B=None, free=None):
    """Tables sized exactly by kv_len (reserved := kv_len)."""
    kv_len = np.asarray(kv_len, dtype=np.int32)
    R = kv_len.shape[0]
    if B is None:
        B = np.linspace(0.1, 1.0, H)
    n_pages = int(sum(-(-int(kv_len[r].max()) // P) for r in range(R)) * C + 8)
    if free is None:
        free = np.random.default_rng(1).permutation(n_pages).astype(np.int32)
    t, _ = O.build_ragged_tables(B, kv_len, C, P, free)
    return t, n_pages


def dense_case(R, H, G, d, lens, seed, C=1, P=16, B=None):
    g = torch.Generator().manual_seed(seed)
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    K = [[torch.randn(int(lens[r][h]), d, generator=g).bfloat16() for h in range(H)] for r in range(R)]
    V = [[torch.randn(int(lens[r][h]), d, generator=g).bfloat16() for h in range(H)] for r in range(R)]
    t, n_pages = simple_tables(lens, H, C, P, B=B)
    pool = scatter_dense_into_pool(K, V, lens, t, n_pages, seed=seed + 1)
    return q, K, V, t, pool


# ---------------------------------------------------------------------------- O2 reserve
@pytest.mark.parametrize("case", GOLD["reserve"])
def test_reserve_golden(case):
    B, res, kv = O.reserve_budgets(case["mu"], case["sigma"], case["alpha"], case["ctx_len"])
    assert B.tolist() == case["B"]
    assert res.tolist() == case["reserved"]
    assert kv.tolist() == case["reserved"]


def test_reserve_invariants_and_overflow():
    rng = np.random.default_rng(3)
    mu = rng.uniform(0.01, 1.0, 16)
    sg = rng.uniform(0, 0.1, 16)
    N = rng.integers(1, 5000, 9)
    dem = rng.integers(0, 5000, (9, 16))
    B, res, kv = O.reserve_budgets(mu, sg, 2.0, N, dem)
    assert np.all((B > 0) & (B <= 1))
    assert np.all(res >= 1) and np.all(res <= N[:, None])
    assert np.all(kv <= res) and np.all(kv <= dem) and np.all((kv == res) | (kv == dem))
    # monotone in B for a fixed N
    order = np.argsort(B)
    assert np.all(np.diff(res[:, order], axis=1) >= 0)
    # sigma = 0: sum_h ceil(B N) within [rho H N, rho H N + H)   (:160, "approximately")
    B0, res0, _ = O.reserve_budgets(mu, np.zeros(16), 2.0, N)
    exact = N[:, None] * mu[None, :]
    slack = res0.sum(1) - exact.sum(1)
    assert np.all(slack >= -1e-9) and np.all(slack < 16)
    with pytest.raises(ValueError):
        O.reserve_budgets([0.0], [0.0], 2.0, [10])
    with pytest.raises(ValueError):
        O.reserve_budgets([0.5], [0.0], 2.0, [0])


# ---------------------------------------------------------------------------- O3 clustering / tables
def test_cluster_properties_and_ties():
    B = np.array([0.5, 0.1, 0.5, 0.9, 0.1, 0.3, 1.0, 0.3])
    perm, cl, sl = O.cluster_heads(B, 4)
    assert sorted(perm.tolist()) == list(range(8))
    assert perm.tolist() == [1, 4, 5, 7, 0, 2, 3, 6]          # stable: ties keep head order
    assert cl.tolist() == [2, 0, 2, 3, 0, 1, 3, 1]
    assert sl.tolist() == [0, 0, 1, 0, 1, 0, 1, 1]
    for c in range(3):                                          # max of group i <= min of group i+1
        assert B[perm[2 * c:2 * c + 2]].max() <= B[perm[2 * c + 2:2 * c + 4]].min()
    p2, c2, s2 = O.cluster_heads(np.full(8, 0.4), 2)            # equal budgets => identity
    assert p2.tolist() == list(range(8)) and c2.tolist() == [0] * 4 + [1] * 4
    with pytest.raises(ValueError):
        O.cluster_heads(B, 3)


@pytest.mark.parametrize("H,Hp", [(4, 2), (6, 2), (6, 3), (8, 4), (8, 2)])
def test_sorted_grouping_minimises_allocation_bruteforce(H, Hp):
    """Sorted-consecutive grouping minimises sum_c H_p * max_c B over ALL equal-size partitions
    (the claim behind Budget-Aware Clustering)."""
    rng = np.random.default_rng(H * 10 + Hp)
    B = rng.uniform(0.01, 1.0, H)
    perm, cl, _ = O.cluster_heads(B, H // Hp)
    ours = sum(Hp * B[perm[c * Hp:(c + 1) * Hp]].max() for c in range(H // Hp))

    def parts(rest):
        if not rest:
            yield []
            return
        first = rest[0]
        for combo in itertools.combinations(rest[1:], Hp - 1):
            grp = (first,) + combo
            left = [x for x in rest if x not in grp]
            for p in parts(left):
                yield [grp] + p

    best = min(sum(Hp * max(B[list(g)]) for g in p) for p in parts(list(range(H))))
    assert ours <= best + 1e-12


def test_tables_structure():
    wl = I.make_workload("8b", R=3, ctx_div=16)
    B, res, kv = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    free = I.make_free_pages(wl, 4000)
    t, kv2 = O.build_ragged_tables(B, res, wl.C, wl.P, free, 0, kv)
    assert np.array_equal(kv2, kv)
    assert len(set(t.tbl_pages.tolist())) == len(t.tbl_pages) == t.n_pages_used
    assert np.array_equal(t.tbl_pages, free[:t.n_pages_used])         # prefix of the free list, in order
    for r in range(wl.R):
        for c in range(wl.C):
            members = t.perm[c * t.Hp:(c + 1) * t.Hp]
            want = -(-int(res[r, members].max()) // wl.P)
            assert t.tbl_indptr[r * wl.C + c + 1] - t.tbl_indptr[r * wl.C + c] == want
    # H_p = H: one table per request sized by the global max (the monolithic page, :89/:188)
    t1, _ = O.build_ragged_tables(B, res, 1, wl.P, free)
    assert [int(x) for x in np.diff(t1.tbl_indptr)] == [-(-int(res[r].max()) // wl.P) for r in range(wl.R)]
    assert t1.n_pages_used * t1.Hp >= t.n_pages_used * t.Hp - wl.R * wl.C * t.Hp   # bytes: ragged <= monolithic (+ page rounding)
    # FILL_GROUP (:235)
    _, kvf = O.build_ragged_tables(B, res, wl.C, wl.P, free, O.FLAG_FILL_GROUP, kv)
    for r in range(wl.R):
        for h in range(wl.H):
            members = t.perm[t.cluster_of[h] * t.Hp:(t.cluster_of[h] + 1) * t.Hp]
            assert kvf[r, h] == res[r, members].max() <= wl.ctx_len[r]
    with pytest.raises(MemoryError):
        O.build_ragged_tables(B, res, wl.C, wl.P, free[:t.n_pages_used - 1])


# ---------------------------------------------------------------------------- O4 plans
@pytest.mark.parametrize("case", GOLD["split_map"])
def test_split_map_golden(case):
    B = np.array(case["B"])
    perm, _, _ = O.cluster_heads(B, len(B) // case["Hp"])
    assert O.split_map(B, perm, case["Hp"], case["n_cta"]).tolist() == case["S"]


def test_split_map_scale_invariance_and_zero():
    B = np.array([0.05, 0.05, 0.1, 0.1, 0.2, 0.3, 0.9, 1.0])
    perm, _, _ = O.cluster_heads(B, 4)
    for lam in (0.5, 0.25, 0.125):            # ratios only (:254); dyadic lam keeps fp exact
        assert O.split_map(lam * B, perm, 2, 108).tolist() == O.split_map(B, perm, 2, 108).tolist()
    assert O.split_map(np.zeros(8), perm, 2, 108).tolist() == [1, 1, 1, 1]


def _one_request_tables(lens, P=16):
    H = len(lens)
    B = np.linspace(0.1, 0.9, H)              # increasing => identity perm, seq i = head i
    t, _ = simple_tables([lens], H, 1, P, B=B)
    return t, B


@pytest.mark.parametrize("case", GOLD["balanced"])
def test_balanced_golden(case):
    t, B = _one_request_tables(case["kv_len"])
    pl = O.plan_partitions(t, B, [case["kv_len"]], case["W"], case["g"], case["c0"], O.MODE_BALANCED)
    got = [[[int(it[1]), int(it[4]), int(it[5])] for it in pl.items[pl.worker_indptr[w]:pl.worker_indptr[w + 1]]]
           for w in range(case["W"])]
    assert got == case["workers"]


@pytest.mark.parametrize("case", GOLD["balanced_dynamic"])
def test_balanced_dynamic_tail_golden(case):
    assert O.list_weights(case["W"], case["dyn_permille"], case["dyn_rounds"]) == case["weights"]
    if "lists" not in case:
        return
    t, B = _one_request_tables(case["kv_len"])
    pl = O.plan_partitions(t, B, [case["kv_len"]], case["W"], case["g"], case["c0"], O.MODE_BALANCED, 0,
                           case["dyn_permille"], case["dyn_rounds"])
    assert pl.n_static == case["W"] and pl.W == len(case["weights"])
    got = [[[int(it[1]), int(it[4]), int(it[5])] for it in pl.items[pl.worker_indptr[w]:pl.worker_indptr[w + 1]]]
           for w in range(pl.W)]
    assert got == case["lists"]
    check_plan_valid(pl, t, np.array([case["kv_len"]]), case["g"])


def test_dynamic_tail_shares_and_validity():
    wl = I.make_workload("8b", R=6, ctx_div=4)
    B, res, kv = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    t, _ = O.build_ragged_tables(B, res, wl.C, wl.P, np.arange(200000, dtype=np.int32))
    W = 16
    pl = O.plan_partitions(t, B, kv, W, 64, 1, O.MODE_BALANCED, 0, 200, 3)
    check_plan_valid(pl, t, kv, 64)
    assert pl.W == W * 4 and pl.n_static == W
    tok = np.array([sum(int(it[5] - it[4]) for it in pl.items[pl.worker_indptr[w]:pl.worker_indptr[w + 1]])
                    for w in range(pl.W)], dtype=float)
    tot = tok.sum()
    share = [tok[r * W:(r + 1) * W].sum() / tot for r in range(4)]
    assert np.allclose(share, [0.8, 0.1, 0.05, 0.05], atol=0.01)
    # no tail requested => identical to the static plan; tail args are ignored by the other modes
    p0 = O.plan_partitions(t, B, kv, W, 64, 1, O.MODE_BALANCED)
    assert p0.W == p0.n_static == W
    for mode in (O.MODE_SPLITMAP, O.MODE_STATIC_EVEN):
        a = O.plan_partitions(t, B, kv, W, 64, 1, mode)
        b = O.plan_partitions(t, B, kv, W, 64, 1, mode, 0, 200, 3)
        assert a.items.tobytes() == b.items.tobytes() and b.W == W
    with pytest.raises(ValueError):
        O.plan_partitions(t, B, kv, W, 64, 1, O.MODE_BALANCED, 0, 200, 0)


def check_plan_valid(pl, t, kv_len, g):
    """Every token of every (r, h) is covered exactly once; slots and counts are consistent."""
    kv_len = np.asarray(kv_len)
    cover = {}
    for it in pl.items:
        r, h, c, s, tb, te, slot, npart = (int(x) for x in it)
        assert c == t.cluster_of[h] and s == t.slot_of[h]
        assert 0 <= tb < te <= kv_len[r, h]
        assert tb % g == 0 and (te % g == 0 or te == kv_len[r, h])
        cover.setdefault((r, h), []).append((tb, te, slot, npart))
    seen_slots = set()
    for r in range(t.R):
        for h in range(t.H):
            lst = sorted(cover.get((r, h), []))
            n = int(kv_len[r, h])
            seq = r * t.H + h
            assert pl.part_indptr[seq + 1] - pl.part_indptr[seq] == len(lst)
            pos = 0
            for o, (tb, te, slot, npart) in enumerate(lst):
                assert tb == pos and npart == len(lst) and slot == pl.part_indptr[seq] + o
                assert slot not in seen_slots
                seen_slots.add(slot)
                pos = te
            assert pos == n
    assert pl.n_part_slots == pl.part_indptr[-1] == pl.n_items == len(pl.items)
    assert pl.worker_indptr[0] == 0 and pl.worker_indptr[-1] == pl.n_items
    assert np.all(np.diff(pl.worker_indptr) >= 0)


@pytest.mark.parametrize("mode", [O.MODE_BALANCED, O.MODE_SPLITMAP, O.MODE_STATIC_EVEN])
@pytest.mark.parametrize("name,kw", [("tiny", {}), ("8b", dict(R=4, ctx_div=8)), ("skew", dict(R=2, ctx_div=8)),
                                     ("uniform", dict(R=8, ctx_div=4)), ("32b", dict(R=5, ctx_div=8))])
def test_plan_invariants(name, kw, mode):
    wl = I.make_workload(name, **kw)
    B, res, kv = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    t, _ = O.build_ragged_tables(B, res, wl.C, wl.P, np.arange(200000, dtype=np.int32))
    for W, c0 in ((4, 0), (37, 1), (296, 2)):
        pl = O.plan_partitions(t, B, kv, W, wl.granule, c0, mode)
        check_plan_valid(pl, t, kv, wl.granule)
        pl2 = O.plan_partitions(t, B, kv, W, wl.granule, c0, mode)
        assert pl.items.tobytes() == pl2.items.tobytes()             # deterministic
        if mode == O.MODE_BALANCED:
            assert pl.n_items <= wl.R * wl.H + W - 1
            u = -(-kv.astype(np.int64) // wl.granule)
            T = int((u + np.where(u > 0, c0, 0)).sum())
            for w in range(W):
                its = pl.items[pl.worker_indptr[w]:pl.worker_indptr[w + 1]]
                gran = sum(-(-(int(it[5]) - int(it[4])) // wl.granule) for it in its)
                assert gran <= T / W + 1                              # never more than the fair share (+ rounding)
                assert gran >= T // W - (c0 * (len(its) + 1)) - 1     # overhead positions carry no tokens


def test_balanced_equal_lengths_even_tokens():
    lens = [[256] * 8] * 4                     # 32 sequences x 4 granules = 128; W = 16 divides it
    B = np.full(8, 0.5)
    t, _ = simple_tables(lens, 8, 2, 16, B=B)
    pl = O.plan_partitions(t, B, lens, 16, 64, 0, O.MODE_BALANCED)
    tok = [sum(int(it[5] - it[4]) for it in pl.items[pl.worker_indptr[w]:pl.worker_indptr[w + 1]]) for w in range(16)]
    assert tok == [512] * 16
    plw = O.plan_partitions(t, B, lens, 1000, 64, 0, O.MODE_BALANCED)   # W > T: empty workers allowed
    check_plan_valid(plw, t, np.array(lens), 64)
    assert plw.n_items == 128


def test_static_even_default_and_splitmap_expansion():
    lens = [[640, 64, 100, 0]]
    B = np.array([0.9, 0.1, 0.2, 0.05])
    t, _ = simple_tables(lens, 4, 2, 16, B=B)
    pl = O.plan_partitions(t, B, lens, 16, 64, 0, O.MODE_STATIC_EVEN)      # S = ceil(16/4) = 4
    assert pl.split_map.tolist() == [4, 4]
    check_plan_valid(pl, t, np.array(lens), 64)
    by = {}
    for it in pl.items:
        by.setdefault(int(it[1]), []).append((int(it[4]), int(it[5])))
    assert sorted(by[0]) == [(0, 128), (128, 320), (320, 448), (448, 640)]   # 10 granules -> 2,3,2,3
    assert by[1] == [(0, 64)] and sorted(by[2]) == [(0, 64), (64, 100)] and 3 not in by
    # SPLITMAP: perm = [3,1,2,0]; Phi = [.15, 1.1]; tau = 1.25/16 -> S = [2, 14]
    pls = O.plan_partitions(t, B, lens, 16, 64, 0, O.MODE_SPLITMAP)
    assert pls.split_map.tolist() == [2, 14]
    check_plan_valid(pls, t, np.array(lens), 64)
    # items dealt round-robin in global order: item k -> worker k mod W
    assert [int(x) for x in np.diff(pls.worker_indptr)] == [1] * pls.n_items + [0] * (16 - pls.n_items)


# ---------------------------------------------------------------------------- O5 merge
def test_merge_properties():
    rng = np.random.default_rng(5)
    parts = [(rng.normal(size=8), float(rng.normal())) for _ in range(5)]
    o, L = O.merge(parts)
    o1, L1 = O.merge([parts[0]])
    assert np.array_equal(o1, parts[0][0]) and L1 == parts[0][1]           # one part is returned unchanged
    o2, L2 = O.merge(parts[::-1])                                          # commutative
    assert np.allclose(o, o2, rtol=0, atol=1e-14) and abs(L - L2) < 1e-14
    oa, La = O.merge([O.merge(parts[:2]), O.merge(parts[2:])])             # associative
    assert np.allclose(o, oa, rtol=0, atol=1e-14) and abs(L - La) < 1e-14
    oi, Li = O.merge(parts + [(np.full(8, np.nan), -math.inf)])            # -inf part is the identity
    assert np.array_equal(o, oi) and L == Li
    # independent closed form: weights softmax(lse)
    lses = np.array([p[1] for p in parts])
    w = np.exp(lses) / np.exp(lses).sum()
    assert np.allclose(o, sum(wi * p[0] for wi, p in zip(w, parts)), atol=1e-14)
    assert abs(L - math.log(np.exp(lses).sum())) < 1e-14
    z, Lz = O.merge([(np.zeros(4), -math.inf)])
    assert np.all(z == 0) and Lz == -math.inf


# ---------------------------------------------------------------------------- O1 attention
def test_attention_vs_dense_library_equal_budgets():
    """(i) all budgets equal => dense fp64 softmax(QK^T/sqrt(d))V on contiguous arrays (torch)."""
    R, H, G, d, n = 3, 4, 3, 64, 197
    lens = [[n] * H] * R
    q, K, V, t, pool = dense_case(R, H, G, d, lens, seed=11, C=2, B=np.full(H, 0.5))
    out, lse, _ = O.attention(q, pool, t, lens, H * G, d)
    Kd = torch.stack([torch.stack(K[r]) for r in range(R)]).double()      # [R,H,n,d]
    Vd = torch.stack([torch.stack(V[r]) for r in range(R)]).double()
    qd = q.double().view(R, H, G, d)
    ref = torch.nn.functional.scaled_dot_product_attention(qd, Kd, Vd)      # [R,H,G,d], scale 1/sqrt(d)
    s = torch.einsum("rhgd,rhnd->rhgn", qd, Kd) / math.sqrt(d)
    assert np.allclose(out, ref.reshape(R, H * G, d).numpy(), rtol=0, atol=1e-12)
    assert np.allclose(lse, torch.logsumexp(s, -1).reshape(R, H * G).numpy(), rtol=0, atol=1e-12)


def test_attention_vs_bruteforce_ragged():
    """(ii) brute force without max-subtraction, pure Python loops, ragged lengths, GQA 5."""
    R, H, G, d = 2, 4, 5, 64
    lens = [[33, 1, 16, 50], [7, 64, 0, 17]]
    q, K, V, t, pool = dense_case(R, H, G, d, lens, seed=12, C=2)
    out, lse, _ = O.attention(q, pool, t, lens, H * G, d)
    for r in range(R):
        for j in range(H * G):
            h = j // G
            n = lens[r][h]
            if n == 0:
                assert np.all(out[r, j] == 0) and lse[r, j] == -math.inf
                continue
            qv = q[r, j].double().numpy()
            Kn, Vn = K[r][h].double().numpy(), V[r][h].double().numpy()
            e = [math.exp(sum(qv[x] * Kn[tk][x] for x in range(d)) / math.sqrt(d)) for tk in range(n)]
            Z = sum(e)
            ref = [sum(e[tk] * Vn[tk][x] for tk in range(n)) / Z for x in range(d)]
            assert np.allclose(out[r, j], ref, rtol=0, atol=1e-12)
            assert abs(lse[r, j] - math.log(Z)) < 1e-12


def test_attention_closed_forms():
    cf = GOLD["attention_closed_forms"]
    d, H, G = 64, 2, 2
    # n = 1  =>  out = v0, lse = q.k0/sqrt(d)
    q, K, V, t, pool = dense_case(1, H, G, d, [[1, 1]], seed=13)
    out, lse, _ = O.attention(q, pool, t, [[1, 1]], H * G, d)
    for j in range(H * G):
        assert np.array_equal(out[0, j], V[0][j // G][0].double().numpy())
        want = float(q[0, j].double() @ K[0][j // G][0].double()) / 8.0
        assert abs(lse[0, j] - want) < 1e-13
    # q = 0 => out = mean(v), lse = ln n
    n = 512
    q, K, V, t, pool = dense_case(1, H, G, d, [[n, n]], seed=14)
    out, lse, _ = O.attention(torch.zeros_like(q), pool, t, [[n, n]], H * G, d)
    assert np.allclose(lse, cf[1]["lse_n512"], rtol=0, atol=1e-12)
    assert np.allclose(out[0, 0], V[0][0].double().mean(0).numpy(), atol=1e-13)
    # pins the 1/sqrt(d) scale and the natural log: q = 8 e0, k0 = e0, k1 = 0, v0 = 1, v1 = 0
    qq = torch.zeros(1, H * G, d).bfloat16()
    qq[0, :, 0] = 8.0
    Kc = [[torch.zeros(2, d).bfloat16() for _ in range(H)]]
    Vc = [[torch.zeros(2, d).bfloat16() for _ in range(H)]]
    for h in range(H):
        Kc[0][h][0, 0] = 1.0
        Vc[0][h][0, :] = 1.0
    t2, npg = simple_tables([[2, 2]], H, 1, 16)
    pool2 = scatter_dense_into_pool(Kc, Vc, [[2, 2]], t2, npg)
    out, lse, _ = O.attention(qq, pool2, t2, [[2, 2]], H * G, d)
    assert np.allclose(out, cf[0]["w0"], rtol=0, atol=1e-15) and np.allclose(lse, cf[0]["lse"], rtol=0, atol=1e-15)
    # the same inputs under a caller-supplied scale (sm_scale of tangram.h): x = [8 * 0.25, 0] = [2, 0]
    out, lse, _ = O.attention(qq, pool2, t2, [[2, 2]], H * G, d, sm_scale=cf[2]["sm_scale"])
    assert np.allclose(out, cf[2]["w0"], rtol=0, atol=1e-15) and np.allclose(lse, cf[2]["lse"], rtol=0, atol=1e-15)
    o_r, l_r = O.attend_range(qq, pool2, t2, H * G, d, 0, 1, 0, 2, sm_scale=cf[2]["sm_scale"])
    assert np.allclose(o_r, cf[2]["w0"], rtol=0, atol=1e-15) and abs(l_r - cf[2]["lse"]) < 1e-15
    # and against dense library attention at a third scale on random data
    q3, K3, V3, t3, pool3 = dense_case(2, 2, 3, d, [[37, 90], [64, 5]], seed=131)
    out3, lse3, _ = O.attention(q3, pool3, t3, [[37, 90], [64, 5]], 6, d, sm_scale=0.05)
    for r in range(2):
        for j in range(6):
            sc = (K3[r][j // 3].double() @ q3[r, j].double()) * 0.05
            assert np.allclose(out3[r, j], (torch.softmax(sc, 0) @ V3[r][j // 3].double()).numpy(), rtol=0, atol=1e-12)
            assert abs(lse3[r, j] - float(torch.logsumexp(sc, 0))) < 1e-12
    # V_h == h + 1 => out_j = floor(j / G) + 1 (pins the GQA map, reading A20) -- G = 3, H = 4
    H4, G3 = 4, 3
    lens = [[40, 9, 23, 31]]
    q, K, V, t, pool = dense_case(1, H4, G3, d, lens, seed=15, C=2)
    Vh = [[torch.full((lens[0][h], d), float(h + 1)).bfloat16() for h in range(H4)]]
    pool = scatter_dense_into_pool(K, Vh, lens, t, pool.shape[0])
    out, _, _ = O.attention(q, pool, t, lens, H4 * G3, d)
    for j in range(H4 * G3):
        assert np.allclose(out[0, j], j // G3 + 1, rtol=0, atol=1e-12)


def test_split_then_merge_equals_unsplit():
    """(iv) any partition of [0, n) merged by O5 equals the unsplit result."""
    R, H, G, d = 2, 2, 4, 128
    lens = [[300, 45], [77, 129]]
    q, K, V, t, pool = dense_case(R, H, G, d, lens, seed=16)
    out, lse, _ = O.attention(q, pool, t, lens, H * G, d)
    rng = np.random.default_rng(17)
    for r in range(R):
        for j in range(H * G):
            n = lens[r][j // G]
            cuts = sorted(set(rng.integers(0, n + 1, size=4).tolist()) | {0, n})
            parts = [O.attend_range(q, pool, t, H * G, d, r, j, a, b) for a, b in zip(cuts[:-1], cuts[1:])]
            parts.append(O.attend_range(q, pool, t, H * G, d, r, j, n, n))         # an empty part
            o, L = O.merge(parts)
            assert np.allclose(o, out[r, j], rtol=0, atol=1e-12) and abs(L - lse[r, j]) < 1e-12


def test_page_permutation_invariance():
    """(v) same logical KV under a different physical page assignment: bit-identical in fp64."""
    R, H, G, d = 2, 4, 2, 64
    lens = np.array([[100, 20, 64, 3], [16, 90, 33, 48]], dtype=np.int32)
    g = torch.Generator().manual_seed(18)
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    K = [[torch.randn(int(lens[r][h]), d, generator=g).bfloat16() for h in range(H)] for r in range(R)]
    V = [[torch.randn(int(lens[r][h]), d, generator=g).bfloat16() for h in range(H)] for r in range(R)]
    B = np.array([0.9, 0.2, 0.6, 0.3])
    res = []
    for seed in (1, 2):
        free = np.random.default_rng(seed).permutation(64).astype(np.int32)
        t, _ = O.build_ragged_tables(B, lens, 2, 16, free)
        pool = scatter_dense_into_pool(K, V, lens, t, 64, seed=seed)               # different garbage too
        res.append(O.attention(q, pool, t, lens, H * G, d)[:2])
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])


def test_slack_is_never_read():
    """NaN in every slot outside [0, kv_len) must not reach the output (reading A28)."""
    R, H, G, d = 1, 4, 2, 64
    lens = [[70, 5, 33, 16]]
    q, K, V, t, _ = dense_case(R, H, G, d, lens, seed=19, C=2)
    pool = scatter_dense_into_pool(K, V, lens, t, 32, fill=float("nan"))
    out, lse, _ = O.attention(q, pool, t, lens, H * G, d)
    assert np.all(np.isfinite(out)) and np.all(np.isfinite(lse))


# ---------------------------------------------------------------------------- O6 KV append (NEXT-1)
def test_append_kv_round_trip_against_dense_attention():
    """Tokens appended one decode step at a time into empty sequences are found again, in order, by the
    (already pinned) gather of O1: attention over the appended cache equals dense library attention over
    the appended rows.  Also: bytes outside the written rows never change, kv_len counts the rows, and
    rows beyond the table capacity are dropped and counted."""
    R, H, G, d, P, steps = 2, 4, 2, 64, 16, 37
    B = np.array([0.9, 0.2, 0.6, 0.3])
    cap_tokens = np.array([[48, 16, 32, 16], [32, 16, 48, 32]], dtype=np.int32)     # reservation per head
    free = np.random.default_rng(3).permutation(40).astype(np.int32)
    t, _ = O.build_ragged_tables(B, cap_tokens, 2, P, free)
    g = torch.Generator().manual_seed(21)
    pool0 = torch.randn(40, t.Hp, 2, P, d, generator=g).bfloat16()
    bits = pool0.view(torch.int16).numpy().view(np.uint16).copy()
    kv = np.zeros((R, H), dtype=np.int32)
    Ks = torch.randn(steps, R, H, d, generator=g).bfloat16()
    Vs = torch.randn(steps, R, H, d, generator=g).bfloat16()
    total_over = 0
    for sidx in range(steps):
        kb = Ks[sidx].view(torch.int16).numpy().view(np.uint16)
        vb = Vs[sidx].view(torch.int16).numpy().view(np.uint16)
        new_bits, new_kv, over = O.append_kv(bits, t, kv, kb, vb)
        assert np.array_equal(new_kv - kv, (new_kv > kv).astype(np.int32)) and over == int((new_kv == kv).sum())
        assert (new_bits != bits).sum() <= int((new_kv > kv).sum()) * 2 * d        # only the written rows change
        bits, kv, total_over = new_bits, new_kv, total_over + over
    # capacity of head h = pages of its cluster x P (cluster = pair of heads sorted by B: (1,3) and (2,0))
    cap = np.zeros((R, H), dtype=np.int32)
    for r in range(R):
        for h in range(H):
            c = t.cluster_of[h]
            cap[r, h] = (t.tbl_indptr[r * 2 + c + 1] - t.tbl_indptr[r * 2 + c]) * P
    assert np.array_equal(kv, np.minimum(steps, cap)) and total_over == int((steps - kv).sum())
    assert cap[0].tolist() == [48, 16, 48, 16]                                      # cluster max, page-rounded
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    pool = torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16)
    out, lse, _ = O.attention(q, pool, t, kv, H * G, d)
    for r in range(R):
        for j in range(H * G):
            h = j // G
            n = int(kv[r, h])
            Kd, Vd = Ks[:n, r, h].double(), Vs[:n, r, h].double()
            sc = (Kd @ q[r, j].double()) / math.sqrt(d)
            ref = torch.softmax(sc, 0) @ Vd
            assert np.allclose(out[r, j], ref.numpy(), rtol=0, atol=1e-12)
            assert abs(lse[r, j] - float(torch.logsumexp(sc, 0))) < 1e-12


# ---------------------------------------------------------------------------- O7 Top-k + compaction (NEXT-2)
def test_topk_indices_definition_and_ties():
    """Brute-force definition: token i is retained iff fewer than k tokens beat it, where j beats i when
    s_j > s_i, or s_j == s_i and j < i.  Includes heavy ties, negative scores, +-0 and infinities."""
    rng = np.random.default_rng(31)
    cases = [rng.normal(size=40).astype(np.float32),
             rng.integers(0, 4, size=50).astype(np.float32),                # many ties
             np.array([0.0, -0.0, 1.0, -1.0, np.inf, -np.inf, 1.0, 0.0], dtype=np.float32),
             np.full(9, 2.5, dtype=np.float32)]
    for s in cases:
        n = len(s)
        for k in (0, 1, n // 3, n - 1, n):
            want = [i for i in range(n)
                    if sum(1 for j in range(n) if s[j] > s[i] or (s[j] == s[i] and j < i)) < k]
            got = O.topk_indices(s, k)
            assert got.tolist() == want
            if 0 < k < n:
                dropped = np.setdiff1d(np.arange(n), got)
                assert s[got].min() >= s[dropped].max()
    assert O.topk_indices(np.array([3, 1, 2], dtype=np.float32), 2).tolist() == [0, 2]   # ascending token order


def test_compact_topk_round_trip_against_dense_attention():
    """Eq. 1 through the pages: attention over the compacted cache (pinned gather O1) equals dense library
    attention over K[I,:], V[I,:] with I from the brute-force-pinned selection; untouched pool bytes survive."""
    R, H, G, d, P, n_max = 2, 4, 2, 64, 16, 90
    ctx = np.array([90, 57], dtype=np.int32)
    keep = np.array([[90, 20, 45, 1], [57, 0, 30, 16]], dtype=np.int32)
    B = np.array([1.0, 0.25, 0.5, 0.2])
    t, _ = O.build_ragged_tables(B, keep, 2, P, np.random.default_rng(4).permutation(60).astype(np.int32))
    g = torch.Generator().manual_seed(33)
    scores = torch.randn(R, H, n_max, generator=g).numpy()
    Kd = torch.randn(R, H, n_max, d, generator=g).bfloat16()
    Vd = torch.randn(R, H, n_max, d, generator=g).bfloat16()
    pool0 = torch.randn(60, t.Hp, 2, P, d, generator=g).bfloat16()
    b0 = pool0.view(torch.int16).numpy().view(np.uint16)
    kb = Kd.view(torch.int16).numpy().view(np.uint16)
    vb = Vd.view(torch.int16).numpy().view(np.uint16)
    b1, idx = O.compact_topk(b0, t, scores, kb, vb, ctx, keep)
    assert (b1 != b0).sum() <= int(keep.sum()) * 2 * d
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    out, lse, _ = O.attention(q, torch.from_numpy(b1.view(np.int16)).view(torch.bfloat16), t, keep, H * G, d)
    for r in range(R):
        for j in range(H * G):
            h = j // G
            I_ = idx[r][h]
            assert len(I_) == keep[r, h] and (len(I_) == 0 or I_.max() < ctx[r])
            if len(I_) == 0:
                assert np.all(out[r, j] == 0) and lse[r, j] == -math.inf
                continue
            sc = (Kd[r, h, I_].double() @ q[r, j].double()) / math.sqrt(d)
            ref = torch.softmax(sc, 0) @ Vd[r, h, I_].double()
            assert np.allclose(out[r, j], ref.numpy(), rtol=0, atol=1e-12)
    with pytest.raises(ValueError):
        O.compact_topk(b0, t, scores, kb, vb, ctx, keep + 100)


# ---------------------------------------------------------------------------- O8 page accounting (NEXT-3)
def test_account_pages_hand_example_fig7():
    """Fig. 7 (:168) in numbers: six heads, one request of 64 tokens, P = 16, two long heads (64) among short
    ones (16).  Monolithic: every page blocked by a long head.  Adjacent groups of 3: each group holds a long
    head, nothing freed.  Clustered: the short heads share a group and free their pages."""
    res = np.array([[16, 64, 16, 16, 64, 16]])
    B = res[0] / 64.0
    ctx = [64]
    mono = O.account_pages(B, res, ctx, 6, 16, O.GROUP_ADJACENT)
    adj = O.account_pages(B, res, ctx, 3, 16, O.GROUP_ADJACENT)
    clu = O.account_pages(B, res, ctx, 3, 16, O.GROUP_CLUSTERED)
    one = O.account_pages(B, res, ctx, 1, 16, O.GROUP_CLUSTERED)
    assert mono["slots_alloc"] == 6 * 64 and mono["pages_alloc"] == 4 and mono["reclaimed_frac"] == 0.0
    assert adj["slots_alloc"] == 384 and adj["pages_alloc"] == 8 and adj["tables"] == 2
    assert clu["slots_alloc"] == 3 * 16 + 3 * 64 == 240 and clu["reclaimed_frac"] == 1.0 - 240 / 384
    assert one["slots_alloc"] == one["slots_exact"] == one["slots_used"] == 4 * 16 + 2 * 64 and one["fragmentation"] == 0.0
    assert clu["fragmentation"] == (240 - 192) / 240 and one["tables"] == 6


def test_account_pages_invariants_and_optimality():
    rng = np.random.default_rng(8)
    for _ in range(30):
        H = int(rng.choice([4, 6, 8]))
        R = int(rng.integers(1, 4))
        P = int(rng.choice([1, 16]))
        B = rng.uniform(0.05, 1.0, size=H)
        ctx = rng.integers(50, 400, size=R)
        res = np.ceil(B[None, :] * ctx[:, None]).astype(np.int64)
        for Hp in [d for d in (1, 2, 4, 8, H) if H % d == 0]:
            clu = O.account_pages(B, res, ctx, Hp, P, O.GROUP_CLUSTERED)
            adj = O.account_pages(B, res, ctx, Hp, P, O.GROUP_ADJACENT)
            assert clu["slots_exact"] == adj["slots_exact"] <= clu["slots_alloc"] <= adj["slots_alloc"] <= clu["slots_full"]
            assert clu["slots_alloc"] == Hp * P * clu["pages_alloc"] and clu["tables"] == R * H // Hp
            if Hp == 1:
                assert clu["slots_alloc"] == clu["slots_exact"]
            if Hp == H:                                   # one group: the policy cannot matter
                assert clu["slots_alloc"] == adj["slots_alloc"] == H * P * sum(-(-int(m) // P) for m in res.max(1))
            # the tables the pinned builder O3 makes use exactly this many pages
            t, _ = O.build_ragged_tables(B, res.astype(np.int32), H // Hp, P, np.arange(10 ** 5, dtype=np.int32))
            assert t.n_pages_used == clu["pages_alloc"]
            if H <= 6 and Hp in (2, 3) and P == 1 and R == 1:   # brute force over all equal-size groupings
                best = min(sum(max(res[0, list(g)]) for g in part) * Hp for part in _equal_partitions(list(range(H)), Hp))
                assert clu["slots_alloc"] == best
    same = O.account_pages(np.full(4, 0.5), np.full((2, 4), 100), [200, 200], 2, 16, O.GROUP_CLUSTERED)
    assert same == O.account_pages(np.full(4, 0.5), np.full((2, 4), 100), [200, 200], 2, 16, O.GROUP_ADJACENT)


def _equal_partitions(items, size):
    if not items:
        yield []
        return
    first, rest = items[0], items[1:]
    import itertools
    for mates in itertools.combinations(rest, size - 1):
        left = [x for x in rest if x not in mates]
        for tail in _equal_partitions(left, size):
            yield [(first,) + mates] + tail


# ---------------------------------------------------------------------------- O9 calibration (NEXT-4)
def test_calibrate_budgets_closed_forms_and_library():
    mu, sd, B = O.calibrate_budgets([[0.25, 0.5], [0.75, 0.5]], 1.0)
    assert mu.tolist() == [0.5, 0.5] and sd.tolist() == [0.25, 0.0]        # population sigma (ddof = 0), not 0.3536
    assert B.tolist() == [0.75, 0.5]
    assert O.calibrate_budgets([[0.25], [0.75]], 2.0)[2].tolist() == [1.0]  # min(1, .) of Eq. 5
    assert O.calibrate_budgets([[0.375]], 2.0)[2].tolist() == [0.375]       # one sample: sigma = 0
    rng = np.random.default_rng(12)
    x = rng.uniform(0.01, 1.0, size=(50, 8))                                # 50 samples (:262)
    mu, sd, B = O.calibrate_budgets(x, 2.0)
    assert np.allclose(mu, x.mean(0), rtol=1e-14, atol=0) and np.allclose(sd, x.std(0, ddof=0), rtol=1e-12, atol=0)
    assert np.array_equal(B, np.minimum(1.0, mu + 2.0 * sd))
    # feeds Eq. 5 of O2 unchanged: reserve_budgets(mu, sigma, alpha) reproduces B
    B2, _, _ = O.reserve_budgets(mu, sd, 2.0, np.array([1000], dtype=np.int32))
    assert np.array_equal(B, B2)
    # Cantelli: at most 1/(1 + alpha^2) of the samples exceed mu + alpha * sigma (holds for the empirical
    # distribution with the population sigma)
    assert ((x > (mu + 2.0 * sd)[None, :]).mean(0) <= 0.2 + 1e-12).all()


# ---------------------------------------------------------------------------- O10 implicit ratios (Eq. 3, NEXT-4)
def test_implicit_ratios_brute_force_and_closed_forms():
    rng = np.random.default_rng(17)
    R, H, n_max = 3, 4, 37
    ctx = np.array([37, 20, 5])
    sc = rng.integers(0, 6, size=(R, H, n_max)).astype(np.float32)          # heavy ties across heads
    for rho in (0.0, 0.13, 0.5, 0.99, 1.0):
        cnt, rat = O.implicit_ratios(sc, ctx, rho)
        for r in range(R):
            N = int(ctx[r])
            flat = [(float(sc[r, h, t]), h * N + t) for h in range(H) for t in range(N)]
            k = min(H * N, max(0, math.ceil(rho * H * N)))
            # definition: entry i is selected iff fewer than k entries beat it (higher score, or equal and lower flat index)
            sel = [i for (v, i) in flat if sum(1 for (w, j) in flat if w > v or (w == v and j < i)) < k]
            want = np.bincount(np.array(sel, dtype=np.int64) // N, minlength=H) if sel else np.zeros(H, int)
            assert cnt[r].tolist() == want.tolist() and cnt[r].sum() == k
            assert np.array_equal(rat[r], cnt[r] / N)
    # heads on disjoint score bands: the flat selection eats the highest heads first
    N = 10
    band = np.stack([np.linspace(0, 0.9, N) + 10 * h for h in range(4)])[None].astype(np.float32)
    cnt, rat = O.implicit_ratios(band, [N], 0.625)                          # k = 25
    assert cnt[0].tolist() == [0, 5, 10, 10] and rat[0].tolist() == [0.0, 0.5, 1.0, 1.0]
    # identical score vectors in every head, no ties inside a head: equal shares, the remainder to the lower heads
    same = np.tile(np.arange(8, dtype=np.float32)[None, None, :], (1, 3, 1))
    assert O.implicit_ratios(same, [8], 10 / 24)[0][0].tolist() == [4, 3, 3]
    # mean over heads of the implicit ratios = k / (H N) >= rho  (Eq. 3 keeps the global budget exactly)
    big = rng.normal(size=(2, 8, 300)).astype(np.float32)
    cnt, rat = O.implicit_ratios(big, [300, 211], 0.3)
    assert cnt.sum(1).tolist() == [math.ceil(0.3 * 8 * 300), math.ceil(0.3 * 8 * 211)]
    # a global selection over ONE head is the per-head selection of Eq. 4
    one = rng.normal(size=(1, 1, 50)).astype(np.float32)
    assert O.implicit_ratios(one, [50], 0.2)[0][0, 0] == len(O.topk_indices(one[0, 0], 10))


# ---------------------------------------------------------------------------- O11 chunked compaction (:152)
def test_compact_topk_chunk_round_trip_and_single_chunk_case():
    """A context compressed chunk by chunk: attention over the resulting cache (pinned gather O1) equals dense
    library attention over the union, in chunk order, of the per-chunk brute-force-pinned selections; with one
    chunk and an empty cache the result is compact_topk's, byte for byte."""
    R, H, G, d, P = 2, 4, 2, 64, 16
    chunks = [np.array([40, 33]), np.array([25, 40]), np.array([7, 1])]
    keeps = [np.array([[40, 10, 21, 1], [33, 0, 16, 9]]), np.array([[25, 6, 11, 0], [40, 3, 17, 16]]),
             np.array([[7, 2, 3, 1], [1, 1, 0, 1]])]
    total = sum(keeps)
    B = np.array([1.0, 0.25, 0.5, 0.3])
    t, _ = O.build_ragged_tables(B, total.astype(np.int32), 2, P, np.random.default_rng(6).permutation(80).astype(np.int32))
    g = torch.Generator().manual_seed(44)
    pool0 = torch.randn(80, t.Hp, 2, P, d, generator=g).bfloat16()
    bits_ = lambda x: x.view(torch.int16).numpy().view(np.uint16)
    pool, kv = bits_(pool0).copy(), np.zeros((R, H), dtype=np.int32)
    kept_k = [[[] for _ in range(H)] for _ in range(R)]
    kept_v = [[[] for _ in range(H)] for _ in range(R)]
    for ci, (cl, kp) in enumerate(zip(chunks, keeps)):
        n_max = int(cl.max())
        sc = torch.randn(R, H, n_max, generator=g).numpy()
        Kc, Vc = torch.randn(R, H, n_max, d, generator=g).bfloat16(), torch.randn(R, H, n_max, d, generator=g).bfloat16()
        if ci == 0:
            single, sidx = O.compact_topk(pool, t, sc, bits_(Kc), bits_(Vc), cl, kp)
        pool, kv, idx = O.compact_topk_chunk(pool, t, sc, bits_(Kc), bits_(Vc), cl, kp, kv)
        if ci == 0:
            assert np.array_equal(pool, single) and all(np.array_equal(idx[r][h], sidx[r][h]) for r in range(R) for h in range(H))
        for r in range(R):
            for h in range(H):
                assert idx[r][h].tolist() == O.topk_indices(sc[r, h, :cl[r]], kp[r, h]).tolist()
                kept_k[r][h].append(Kc[r, h, idx[r][h]]), kept_v[r][h].append(Vc[r, h, idx[r][h]])
    assert np.array_equal(kv, total)
    assert (pool != bits_(pool0)).sum() <= int(total.sum()) * 2 * d
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    out, lse, _ = O.attention(q, torch.from_numpy(pool.view(np.int16)).view(torch.bfloat16), t, kv, H * G, d)
    for r in range(R):
        for j in range(H * G):
            Kd, Vd = torch.cat(kept_k[r][j // G]).double(), torch.cat(kept_v[r][j // G]).double()
            sc_ = (Kd @ q[r, j].double()) / math.sqrt(d)
            assert np.allclose(out[r, j], (torch.softmax(sc_, 0) @ Vd).numpy(), rtol=0, atol=1e-12)
    with pytest.raises(ValueError):                      # the tables are full now (:176)
        O.compact_topk_chunk(pool, t, sc, bits_(Kc), bits_(Vc), chunks[-1], np.full((R, H), 1), kv + 200)


def test_global_flat_topk_equals_per_head_topk_with_its_own_counts():
    """Eq. 3 decomposes exactly: the global flat Top-k set, split by head, is each head's Top-(its implicit count)
    under the same tie rule -- so the non-uniform compressor Tangram replaces (and Eq. 2, keep = ceil(rho N) for
    every head) are the per-head selection of Eq. 4 with particular `keep` inputs."""
    rng = np.random.default_rng(23)
    R, H, n_max = 2, 5, 60
    ctx = np.array([60, 41])
    sc = rng.integers(0, 7, size=(R, H, n_max)).astype(np.float32) * rng.uniform(0.5, 2.0, size=(1, H, 1)).astype(np.float32)
    for rho in (0.1, 0.45, 0.8):
        cnt, _ = O.implicit_ratios(sc, ctx, rho)
        for r in range(R):
            N = int(ctx[r])
            flat = np.concatenate([sc[r, h, :N] for h in range(H)])
            sel = O.topk_indices(flat, int(cnt[r].sum()))
            for h in range(H):
                mine = sel[(sel >= h * N) & (sel < (h + 1) * N)] - h * N
                assert mine.tolist() == O.topk_indices(sc[r, h, :N], int(cnt[r, h])).tolist()


def test_topk_indices_against_a_stable_library_sort():
    """O7 once more against a library routine: a stable descending argsort keeps equal scores in index order, so its
    first k entries are the oracle's selection (random rows with ties, +-0, infinities)."""
    rng = np.random.default_rng(77)
    for _ in range(200):
        n = int(rng.integers(1, 400))
        s = rng.choice([rng.normal(size=n), rng.integers(-3, 4, size=n).astype(float)]).astype(np.float32)
        if n > 4:
            s[rng.integers(n)], s[rng.integers(n)], s[rng.integers(n)] = 0.0, -0.0, np.inf
        k = int(rng.integers(0, n + 1))
        want = np.sort(np.argsort(-s.astype(np.float64), kind="stable")[:k])
        assert O.topk_indices(s, k).tolist() == want.tolist()


# ---------------------------------------------------------------------------- O12 block-table growth (NEXT-4)
def test_extend_tables_hand_example():
    """Hand-evaluated updates (tests/golden): which rows take a page, from where in the free list, and which starve."""
    for case in GOLD["extend_tables"]:
        free = np.array(case["free_pages"], dtype=np.int32)
        t, _ = O.build_ragged_tables(np.array(case["B"]), np.array(case["reserved"], dtype=np.int32), case["n_clusters"],
                                     case["P"], free, headroom_pages=case["headroom_pages"])
        b = case["built"]
        assert t.tbl_indptr.tolist() == b["tbl_indptr"] and t.tbl_pages.tolist() == b["tbl_pages"]
        assert t.row_pages.tolist() == b["row_pages"] and t.n_pages_used == b["n_pages_used"]
        for u in case["updates"]:
            t, starved = O.extend_tables(t, np.array(u["kv_len"], dtype=np.int32), free)
            assert t.tbl_pages.tolist() == u["tbl_pages"] and t.row_pages.tolist() == u["row_pages"]
            assert t.n_pages_used == u["n_pages_used"] and starved == u["starved"]
            assert t.tbl_indptr.tolist() == b["tbl_indptr"]                       # rows never move


def test_headroom_zero_is_the_tight_table_and_slots_do_not_change_the_gather():
    """headroom_pages = 0 reproduces the pinned builder bit for bit; with headroom the assigned pages are the same
    ones in the same order (only -1 slots are interleaved), so the pinned gather O1 reads the same bytes."""
    R, H, G, d = 2, 4, 2, 64
    lens = np.array([[100, 20, 64, 3], [16, 90, 33, 48]], dtype=np.int32)
    B = np.array([0.9, 0.2, 0.6, 0.3])
    free = np.random.default_rng(5).permutation(64).astype(np.int32)
    t0, _ = O.build_ragged_tables(B, lens, 2, 16, free)
    t1, _ = O.build_ragged_tables(B, lens, 2, 16, free, headroom_pages=3)
    assert t0.row_pages is None and t1.n_pages_used == t0.n_pages_used
    assert t1.tbl_pages[t1.tbl_pages >= 0].tolist() == t0.tbl_pages.tolist()
    for row in range(R * 2):
        n = t0.tbl_indptr[row + 1] - t0.tbl_indptr[row]
        assert t1.row_pages[row] == n == t1.assigned(row) and t1.tbl_indptr[row + 1] - t1.tbl_indptr[row] == n + 3
        assert np.array_equal(t1.tbl_pages[t1.tbl_indptr[row]:t1.tbl_indptr[row] + n],
                              t0.tbl_pages[t0.tbl_indptr[row]:t0.tbl_indptr[row + 1]])
        assert np.all(t1.tbl_pages[t1.tbl_indptr[row] + n:t1.tbl_indptr[row + 1]] == -1)
    g = torch.Generator().manual_seed(6)
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    pool = torch.randn(64, 2, 2, 16, d, generator=g).bfloat16()
    a, b = O.attention(q, pool, t0, lens, H * G, d)[:2], O.attention(q, pool, t1, lens, H * G, d)[:2]
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_extend_then_append_round_trip_through_page_boundaries():
    """A decode loop of 70 steps (extend the tables, then append one row per head) crosses several page
    boundaries in every row and drops nothing; the pinned gather O1 then finds the prefill rows followed by all
    appended rows: attention = dense library attention over them.  The pages are a duplicate-free prefix of the
    free list, and every row ends with exactly the pages the pinned builder gives a batch whose reservation is
    the final length + 1 (the same tables up to which physical page sits where)."""
    R, H, G, d, P, steps, C = 2, 4, 2, 64, 16, 70, 2
    B = np.array([0.9, 0.2, 0.6, 0.3])
    lens0 = np.array([[40, 10, 33, 16], [16, 5, 20, 7]], dtype=np.int32)
    free = np.random.default_rng(8).permutation(80).astype(np.int32)
    t, _ = O.build_ragged_tables(B, lens0, C, P, free, headroom_pages=6)
    g = torch.Generator().manual_seed(9)
    K0 = [[torch.randn(int(lens0[r][h]), d, generator=g).bfloat16() for h in range(H)] for r in range(R)]
    V0 = [[torch.randn(int(lens0[r][h]), d, generator=g).bfloat16() for h in range(H)] for r in range(R)]
    pool = scatter_dense_into_pool(K0, V0, lens0, t, 80, seed=10)
    bits = pool.view(torch.int16).numpy().view(np.uint16).copy()
    Ks = torch.randn(steps, R, H, d, generator=g).bfloat16()
    Vs = torch.randn(steps, R, H, d, generator=g).bfloat16()
    kv = lens0.copy()
    for s_ in range(steps):
        t, starved = O.extend_tables(t, kv, free)
        assert starved == 0
        bits, kv, over = O.append_kv(bits, t, kv, Ks[s_].view(torch.int16).numpy().view(np.uint16),
                                     Vs[s_].view(torch.int16).numpy().view(np.uint16))
        assert over == 0
    assert np.array_equal(kv, lens0 + steps)
    used = t.tbl_pages[t.tbl_pages >= 0]
    assert len(set(used.tolist())) == len(used) == t.n_pages_used
    assert sorted(used.tolist()) == sorted(free[:t.n_pages_used].tolist())
    tight, _ = O.build_ragged_tables(B, kv, C, P, free)          # reservation = final length: ceil(n / P) pages
    for row in range(R * C):
        # the row grew when its longest head filled a page, i.e. it holds floor((longest - 1) / P) + 1 pages
        # (the page of the last appended token) -- the pinned builder's count for these lengths
        assert t.assigned(row) == tight.tbl_indptr[row + 1] - tight.tbl_indptr[row]
    q = torch.randn(R, H * G, d, generator=g).bfloat16()
    out, lse, _ = O.attention(q, torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16), t, kv, H * G, d)
    for r in range(R):
        for j in range(H * G):
            h = j // G
            Kd = torch.cat([K0[r][h], Ks[:, r, h]]).double()
            Vd = torch.cat([V0[r][h], Vs[:, r, h]]).double()
            sc = (Kd @ q[r, j].double()) / math.sqrt(d)
            assert np.allclose(out[r, j], (torch.softmax(sc, 0) @ Vd).numpy(), rtol=0, atol=1e-12)
            assert abs(lse[r, j] - float(torch.logsumexp(sc, 0))) < 1e-12


def test_extend_tables_starvation_drops_exactly_the_unserved_rows():
    """Free list shorter than the growth: rows are served in (request, cluster) order until it runs out; the heads
    of an unserved row that are full drop their row and are counted (reading A29), the others keep growing."""
    R, H, P, C, d = 2, 2, 16, 2, 8
    B = np.array([0.3, 0.8])
    lens0 = np.array([[16, 32], [16, 16]], dtype=np.int32)        # every row is exactly full
    free = np.arange(100, 107, dtype=np.int32)                    # 5 pages to build with, 2 left for 4 rows
    t, _ = O.build_ragged_tables(B, lens0, C, P, free, headroom_pages=2)
    assert t.n_pages_used == 5
    t, starved = O.extend_tables(t, lens0, free)
    assert starved == 2 and t.row_pages.tolist() == [2, 3, 1, 1] and t.n_pages_used == 7
    bits = np.zeros((107, 1, 2, P, d), dtype=np.uint16)
    k = np.full((R, H, d), 7, dtype=np.uint16)
    _, kv, over = O.append_kv(bits, t, lens0, k, k)
    assert over == 2 and kv.tolist() == [[17, 33], [16, 16]]
    t2, starved2 = O.extend_tables(t, kv, free)                   # nothing left: the same two rows starve again
    assert starved2 == 2 and np.array_equal(t2.tbl_pages, t.tbl_pages)
