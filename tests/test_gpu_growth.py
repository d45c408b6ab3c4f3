"""GPU parity of the block-table growth (NEXT-4, PAPER.md:244 / :89) and of the one-launch decode step
(tangram_decode_step: KV append + attention + merge + length update + table growth) against the oracle's
extend_tables (O12) -> append_kv (O6) -> attention (O1).  Byte / index work is compared bit for bit (pool, lengths,
page tables, free-list cursor, dropped-row and starved-row counts); the attention output within the a4 tolerances."""
import math

import numpy as np
import pytest
import torch

from oracle import tangram_oracle as O
from paper_2606_06302_b200 import binding as T
from paper_2606_06302_b200 import inputs as I

from test_gpu_parity import DYN_PERMILLE, DYN_ROUNDS, bits, check, n_cta

pytestmark = pytest.mark.gpu


def growable_setup(wl, headroom, extra_free=None, Hp=None):
    """Growable tables through the product and, independently, through the oracle (they must agree bit for bit)."""
    C = wl.C if Hp is None else wl.H // Hp
    B, res, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    need = T.tangram_pages_needed(B, res, C, wl.P)
    n_free = need + (headroom * wl.R * C if extra_free is None else extra_free)
    free = I.make_free_pages(wl, n_free)
    t, kv = T.tangram_build_ragged_tables(B, res, C, wl.P, free, 0, kv, headroom_pages=headroom)
    Bo, reso, kvo = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    to, kvo = O.build_ragged_tables(Bo, reso, C, wl.P, free, 0, kvo, headroom_pages=headroom)
    same_tables(to, t)
    assert np.array_equal(kv, kvo)
    return B, kv, t, to, free


def same_tables(to, t):
    assert np.array_equal(to.tbl_indptr, t.tbl_indptr) and np.array_equal(to.tbl_pages, t.tbl_pages)
    assert np.array_equal(to.row_pages, t.row_pages) and to.n_pages_used == t.n_pages_used


def slot_capacity(t, wl):
    rows = np.arange(wl.R)[:, None] * t.C + t.cluster_of[None, :]
    return ((t.tbl_indptr[rows + 1] - t.tbl_indptr[rows]) * wl.P).astype(np.int32)


def make_pool(wl, t, n_pages, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    q = torch.randn(wl.R, wl.Hq, wl.d, generator=g, device="cuda").bfloat16()
    pool = torch.randn(n_pages, t.Hp, 2, wl.P, wl.d, generator=g, device="cuda").bfloat16()
    return q, pool


@pytest.mark.parametrize("name,kw,Hp", [("8b", dict(R=6, ctx_div=16), 1), ("8b", dict(R=6, ctx_div=16), 2),
                                        ("32b", dict(R=5, ctx_div=16), 4), ("uniform", dict(R=40, ctx_div=8), 8),
                                        ("32b", dict(), 1), ("uniform", dict(), 8)])
def test_extend_tables_device_bit_exact(name, kw, Hp):
    """The device update (one block, ordered scan) against O12 over 50 updates with rising lengths, a free list that
    runs out and headroom that runs out: tables, cursor and starved count equal after every update.  The full-size
    32b shape at H_p = 1 has 512 rows, uniform 256: more rows than one warp, fewer than one 1024-thread chunk; the
    2500-row case below covers several chunks."""
    wl = I.make_workload(name, **kw)
    C = wl.H // Hp
    B, kv, t, to, free = growable_setup(wl, headroom=3, extra_free=2 * wl.R * C + 3, Hp=Hp)
    pl = T.tangram_plan_partitions(t, B, kv, 8, wl.granule, 1, T.MODE_BALANCED)
    dp = T.tangram_upload(t, pl)
    free_dev = torch.from_numpy(free).cuda()
    rng = np.random.default_rng(3)
    rows = np.arange(wl.R)[:, None] * C + t.cluster_of[None, :]
    cur = np.maximum(to.row_pages[rows] * wl.P - rng.integers(0, 21, size=kv.shape), 0).astype(np.int32)
    starved_total = 0
    for step in range(50):
        to, starved = O.extend_tables(to, cur, free)
        starved_total += starved
        T.tangram_extend_tables_device(dp, torch.from_numpy(cur).cuda(), free_dev)
        got_starved = T.tangram_download_tables(dp, t)
        same_tables(to, t)
        assert got_starved == starved_total
        cur = np.minimum(cur + 1, to.row_pages[rows] * wl.P).astype(np.int32)
    assert starved_total > 0 and to.n_pages_used == len(free)


def test_extend_tables_device_many_rows():
    """2500 (request, cluster) rows: the ordered scan runs over three 1024-row chunks and must keep the row order
    across them."""
    wl = I.make_random_workload(77, R=625, H=4, G=1, d=64, C=4, max_ctx=80)
    B, kv, t, to, free = growable_setup(wl, headroom=2, extra_free=3000)
    pl = T.tangram_plan_partitions(t, B, kv, 4, wl.granule, 1, T.MODE_BALANCED)
    dp = T.tangram_upload(t, pl)
    free_dev = torch.from_numpy(free).cuda()
    rows = np.arange(wl.R)[:, None] * t.C + t.cluster_of[None, :]
    cur = (to.row_pages[rows] * wl.P).astype(np.int32)          # every row is full: all 2500 rows ask at once
    cur[::7] -= 1                                                # ... except some
    starved_total = 0
    for step in range(3):
        to, starved = O.extend_tables(to, cur, free)
        starved_total += starved
        T.tangram_extend_tables_device(dp, torch.from_numpy(cur).cuda(), free_dev)
        assert T.tangram_download_tables(dp, t) == starved_total
        same_tables(to, t)
        cur = (to.row_pages[rows] * wl.P).astype(np.int32)
    assert starved_total > 0


def run_decode_steps(wl, B, kv0, t, to, free, steps, d_check_every=1, flags=0, W=None, seed=5, dyn=(DYN_PERMILLE, DYN_ROUNDS),
                     with_growth=True):
    """`steps` fused decode steps against the oracle composition; returns the final oracle-side state."""
    cap = slot_capacity(t, wl)
    W = W or n_cta(wl)
    pl = T.tangram_plan_partitions(t, B, cap, W, wl.granule, 1, T.MODE_BALANCED, 0, *dyn)
    dp = T.tangram_upload(t, pl)
    n_pages = int(max(free.max(), t.tbl_pages.max())) + 1
    q, pool = make_pool(wl, t, n_pages, seed)
    free_dev = torch.from_numpy(free).cuda()
    kv_dev = torch.from_numpy(kv0.copy()).cuda()
    over_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    g = torch.Generator(device="cuda").manual_seed(seed + 1)
    ref_bits, ref_kv, ref_over, ref_starved = bits(pool).copy(), kv0.copy(), 0, 0
    if with_growth:                                                  # room for the first token
        T.tangram_extend_tables_device(dp, kv_dev, free_dev)
        to, s = O.extend_tables(to, ref_kv, free)
        ref_starved += s
    for step in range(steps):
        k_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        v_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        out, lse = T.tangram_decode_step(dp, q, k_new, v_new, pool, kv_dev, free_dev if with_growth else None,
                                         overflow=over_dev, flags=flags)
        torch.cuda.synchronize()
        ref_bits, ref_kv, o = O.append_kv(ref_bits, to, ref_kv, bits(k_new), bits(v_new))
        ref_over += o
        if step % d_check_every == 0 or step == steps - 1:
            ro, rl, _ = O.attention(q.cpu(), torch.from_numpy(ref_bits.view(np.int16)).view(torch.bfloat16), to, ref_kv,
                                    wl.Hq, wl.d)
            check(out, lse, ro, rl, f"decode step {step}")
        if with_growth:
            to, s = O.extend_tables(to, ref_kv, free)
            ref_starved += s
        assert np.array_equal(kv_dev.cpu().numpy(), ref_kv), f"lengths after step {step}"
        assert int(over_dev.item()) == ref_over, f"dropped rows after step {step}"
        assert np.array_equal(bits(pool), ref_bits), f"pool after step {step}"
        if with_growth:
            assert T.tangram_download_tables(dp, t) == ref_starved
            same_tables(to, t)
    return ref_kv, ref_over, ref_starved


@pytest.mark.parametrize("name,kw", [("8b", dict(R=3, ctx_div=32)), ("32b", dict(R=3, ctx_div=32)),
                                     ("skew", dict(R=2, ctx_div=32)), ("tiny", dict())])
def test_decode_step_equals_extend_append_attend(name, kw):
    """40 fused steps (more than two page boundaries per row) on scaled configs: after EVERY step the pool, the
    lengths, the tables and the counters equal the oracle's, the output is within tolerance, nothing is dropped."""
    wl = I.make_workload(name, **kw)
    B, kv, t, to, free = growable_setup(wl, headroom=4)
    ref_kv, over, starved = run_decode_steps(wl, B, kv, t, to, free, steps=40)
    assert over == 0 and starved == 0 and np.array_equal(ref_kv, kv + 40)


def test_decode_step_full_size_8b_in_the_decode_loop_configuration():
    """The fused step at BASELINE.json's full 8b size in the configuration bench.py's decode loop times (W = N_CTA,
    open-ended plan over the tables' capacity, default dynamic tail, TANGRAM_STEP_OVERLAP): after each of three steps
    the whole 0.9 GB pool, the lengths, the tables and the counters equal the oracle's bit for bit and every output
    row is within tolerance of the oracle's attention over the grown cache."""
    wl = I.make_workload("8b")
    B, kv, t, to, free = growable_setup(wl, headroom=2)
    W = n_cta(wl)
    dyn = T.tangram_default_dynamic_tail(slot_capacity(t, wl), W, wl.granule, 1)
    ref_kv, over, starved = run_decode_steps(wl, B, kv, t, to, free, steps=3, flags=T.STEP_OVERLAP, W=W, dyn=dyn)
    assert over == 0 and starved == 0 and np.array_equal(ref_kv, kv + 3)


def test_decode_step_page_size_32():
    """The fused step on 32-token pages: growth hands out a page every 32 tokens per row."""
    wl = I.make_workload("8b", R=3, ctx_div=32, page_size=32)
    B, kv, t, to, free = growable_setup(wl, headroom=3)
    ref_kv, over, starved = run_decode_steps(wl, B, kv, t, to, free, steps=70)
    assert over == 0 and starved == 0


def test_decode_step_small_grid_and_static_plan():
    """W = 1 (the single CTA merges AND grows) and W = 5 with a static plan."""
    wl = I.make_random_workload(41, R=3, H=4, G=2, d=128, C=2, max_ctx=300)
    for W in (1, 5):
        B, kv, t, to, free = growable_setup(wl, headroom=3)
        run_decode_steps(wl, B, kv, t, to, free, steps=20, W=W, dyn=(0, 0))


@pytest.mark.parametrize("flags", [0, T.STEP_OVERLAP])
def test_decode_step_on_a_grid_larger_than_the_device(flags):
    """W = 300 work lists = 300 CTAs, more than fit the device: a plain launch whose first 152 CTAs to finish leave at
    once and whose last 148 merge; the CTA with the last ticket updates the lengths and grows the tables.  With
    TANGRAM_STEP_OVERLAP such a grid waits for its predecessor but does not let its own dependents start early."""
    wl = I.make_workload("8b", R=3, ctx_div=16)
    B, kv, t, to, free = growable_setup(wl, headroom=3)
    ref_kv, over, starved = run_decode_steps(wl, B, kv, t, to, free, steps=24, W=300, flags=flags, dyn=(300, 2))
    assert over == 0 and starved == 0


def test_decode_step_starvation_drops_and_counts():
    """A free list that runs out and headroom that runs out: exactly the oracle's rows are dropped and counted, the
    other heads keep growing, and nothing outside the written rows changes (the pool is compared bit for bit)."""
    wl = I.make_random_workload(43, R=4, H=4, G=2, d=64, C=2, max_ctx=200)
    B, kv, t, to, free = growable_setup(wl, headroom=2, extra_free=7)
    ref_kv, over, starved = run_decode_steps(wl, B, kv, t, to, free, steps=45)
    assert over > 0 and starved > 0


def test_decode_step_without_free_list_is_append_plus_attention():
    """free_pages = NULL: no growth; tight tables drop rows at the end of their last page (reading A29)."""
    wl = I.make_random_workload(44, R=3, H=2, G=4, d=128, C=1, max_ctx=100)
    B, res, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    need = T.tangram_pages_needed(B, res, wl.C, wl.P)
    free = I.make_free_pages(wl, need + 4)
    t, kv = T.tangram_build_ragged_tables(B, res, wl.C, wl.P, free, 0, kv)
    to, _ = O.build_ragged_tables(B, res, wl.C, wl.P, free, 0, kv)
    ref_kv, over, _ = run_decode_steps(wl, B, kv, t, to, free, steps=20, with_growth=False)
    assert over > 0


def test_decode_step_head_dim_256_uses_the_follow_up_kernels():
    """d = 256: the merge and the growth run as follow-up kernels (no in-grid tail phase); same results."""
    wl = I.make_random_workload(45, R=3, H=4, G=2, d=256, C=2, max_ctx=400)
    B, kv, t, to, free = growable_setup(wl, headroom=3)
    ref_kv, over, starved = run_decode_steps(wl, B, kv, t, to, free, steps=24)
    assert over == 0 and starved == 0


def test_host_extend_then_sync_tables():
    """The host path: tangram_extend_tables on the host tables, tangram_sync_tables to the device copy, then
    tangram_append_kv + tangram_decode_attention -- the same state as the device path."""
    wl = I.make_workload("8b", R=3, ctx_div=32)
    B, kv, t, to, free = growable_setup(wl, headroom=3)
    cap = slot_capacity(t, wl)
    pl = T.tangram_plan_partitions(t, B, cap, n_cta(wl), wl.granule, 1, T.MODE_BALANCED, 0, DYN_PERMILLE, DYN_ROUNDS)
    dp = T.tangram_upload(t, pl)
    q, pool = make_pool(wl, t, int(free.max()) + 1, 9)
    kv_dev = torch.from_numpy(kv.copy()).cuda()
    over_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    g = torch.Generator(device="cuda").manual_seed(10)
    ref_bits, ref_kv = bits(pool).copy(), kv.copy()
    for step in range(36):
        ext, starved = T.tangram_extend_tables(t, ref_kv, free)
        to, s = O.extend_tables(to, ref_kv, free)
        same_tables(to, t)
        assert starved == s == 0
        if ext:
            T.tangram_sync_tables(t, dp)
        k_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        v_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        T.tangram_append_kv(dp, k_new, v_new, pool, kv_dev, over_dev)
        out, lse = T.tangram_decode_attention(dp, q, pool, kv_len=kv_dev)
        torch.cuda.synchronize()
        ref_bits, ref_kv, o = O.append_kv(ref_bits, to, ref_kv, bits(k_new), bits(v_new))
        assert o == 0 and int(over_dev.item()) == 0
        assert np.array_equal(bits(pool), ref_bits) and np.array_equal(kv_dev.cpu().numpy(), ref_kv)
    ro, rl, _ = O.attention(q.cpu(), torch.from_numpy(ref_bits.view(np.int16)).view(torch.bfloat16), to, ref_kv, wl.Hq, wl.d)
    check(out, lse, ro, rl, "host-extended tables")


def test_200_decode_steps_on_a_3_layer_graph_through_page_boundaries():
    """200 decode steps of a 3-layer model, ONE launch per layer-step (tangram_decode_step with
    TANGRAM_STEP_OVERLAP), the 3-layer step captured in one CUDA graph and replayed: every row crosses ten or more
    page boundaries; afterwards pool, lengths, page tables and free-list cursor of every layer equal the oracle's bit
    for bit, no row was dropped, and the last step's output matches the oracle."""
    L, steps = 3, 200
    headroom = steps // 16 + 2
    layers = []
    for l in range(L):
        wl = I.make_workload("32b", R=2, ctx_div=32, layer=l)
        B, kv, t, to, free = growable_setup(wl, headroom=headroom)
        cap = slot_capacity(t, wl)
        plan = T.tangram_plan_partitions(t, B, cap, n_cta(wl), wl.granule, 1, T.MODE_BALANCED, 0, DYN_PERMILLE, DYN_ROUNDS)
        dp = T.tangram_upload(t, plan)
        q, pool = make_pool(wl, t, int(free.max()) + 1, 100 + l)
        g = torch.Generator(device="cuda").manual_seed(200 + l)
        Ks = torch.randn(steps, wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        Vs = torch.randn(steps, wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        layers.append(dict(wl=wl, t=t, to=to, free=free, kv=kv.copy(), q=q, pool=pool, dp=dp, Ks=Ks, Vs=Vs,
                           kv_dev=torch.from_numpy(kv.copy()).cuda(), free_dev=torch.from_numpy(free).cuda(),
                           k=torch.empty_like(Ks[0]), v=torch.empty_like(Vs[0]),
                           over=torch.zeros(1, dtype=torch.int32, device="cuda"),
                           out=torch.empty_like(q), lse=torch.empty(wl.R, wl.Hq, device="cuda"),
                           ws=torch.empty(T.tangram_workspace_bytes(plan.n_part_slots, wl.G, wl.d), dtype=torch.uint8,
                                          device="cuda"),
                           ref_bits=bits(pool).copy()))

    def step(st):
        for S in layers:
            T.tangram_decode_step(S["dp"], S["q"], S["k"], S["v"], S["pool"], S["kv_dev"], S["free_dev"], S["out"], S["lse"],
                                  S["ws"], overflow=S["over"], flags=T.STEP_OVERLAP, stream=st)

    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        for S in layers:
            T.tangram_extend_tables_device(S["dp"], S["kv_dev"], S["free_dev"], stream=st)
            S["k"].copy_(S["Ks"][0]), S["v"].copy_(S["Vs"][0])
        step(st)                                                               # decode step 1 (eager)
        graph = torch.cuda.CUDAGraph()
        for S in layers:
            S["k"].copy_(S["Ks"][1]), S["v"].copy_(S["Vs"][1])
        with torch.cuda.graph(graph, stream=st):
            step(st)                                                           # decode step 2 runs at the first replay
        for s_ in range(1, steps):
            for S in layers:
                S["k"].copy_(S["Ks"][s_]), S["v"].copy_(S["Vs"][s_])
            graph.replay()
    torch.cuda.synchronize()
    for S in layers:
        wl, to, free = S["wl"], S["to"], S["free"]
        rb, rk = S["ref_bits"], S["kv"]
        to, s0 = O.extend_tables(to, rk, free)
        assert s0 == 0
        for s_ in range(steps):
            rb, rk, o = O.append_kv(rb, to, rk, bits(S["Ks"][s_]), bits(S["Vs"][s_]))
            assert o == 0
            to, s1 = O.extend_tables(to, rk, free)
            assert s1 == 0
        assert int(S["over"].item()) == 0
        assert np.array_equal(S["kv_dev"].cpu().numpy(), rk) and np.array_equal(rk, S["kv"] + steps)
        assert np.array_equal(bits(S["pool"]), rb)
        assert T.tangram_download_tables(S["dp"], S["t"]) == 0
        same_tables(to, S["t"])
        grew = to.row_pages - S["to"].row_pages
        assert grew.min() >= steps // 16 - 2                               # every row crossed at least 10 page boundaries
        ro, rl, _ = O.attention(S["q"].cpu(), torch.from_numpy(rb.view(np.int16)).view(torch.bfloat16), to, rk, wl.Hq, wl.d)
        check(S["out"], S["lse"], ro, rl, "200-step graph loop")


def _poisoned_free_list(wl, headroom):
    """Growable tables from a valid free list whose NOT YET USED part then gets entries that are no pages of the pool
    (beyond its end, huge, negative) mixed in; -> (B, kv, tables, free list, pages of the pool, the bad entries)."""
    B, kv, t, to, free = growable_setup(wl, headroom=headroom)
    n_pages = int(free.max()) + 1
    free = free.copy()
    tail = np.arange(t.n_pages_used, free.shape[0])
    bad_at = tail[::3][:12]
    bad = np.array([n_pages, n_pages + 5, 2 ** 30, -7, 2 ** 31 - 1, n_pages + 1] * 2, dtype=np.int64)[:bad_at.shape[0]]
    free[bad_at] = bad.astype(np.int32)
    return B, kv, t, free, n_pages, set(int(x) for x in bad)


def test_decode_step_never_hands_out_a_free_list_entry_outside_the_pool():
    """The appends store through the page tables without a hardware bound (the TMA reads are clamped, plain stores are
    not), so a wrong free-list entry must not become a store address.  tangram_decode_step knows the pool's size: a
    free-list entry outside [0, n_pool_pages) is consumed but never written into the tables, the row counts as starved
    and takes the next entry at the next step.  Checked: guard pages behind the pool and every page no table names
    keep their bits; the tables hold only pages of the pool; rows were starved; and the attention result of the last
    step equals the oracle's over the final pool, tables and lengths."""
    wl = I.make_random_workload(46, R=4, H=4, G=2, d=64, C=2, max_ctx=200)
    B, kv, t, free, n_pages, bad = _poisoned_free_list(wl, headroom=6)
    n_guard = 6
    g = torch.Generator(device="cuda").manual_seed(9)
    big = torch.randn(n_pages + n_guard, t.Hp, 2, wl.P, wl.d, generator=g, device="cuda").bfloat16()
    pool = big[:n_pages]                                              # the pool the calls are told about
    before = bits(big).copy()
    q = torch.randn(wl.R, wl.Hq, wl.d, generator=g, device="cuda").bfloat16()
    cap = slot_capacity(t, wl)
    pl = T.tangram_plan_partitions(t, B, cap, n_cta(wl), wl.granule, 1, T.MODE_BALANCED, 0, 300, 3)
    dp = T.tangram_upload(t, pl)
    free_dev, kv_dev = torch.from_numpy(free).cuda(), torch.from_numpy(kv.copy()).cuda()
    over = torch.zeros(1, dtype=torch.int32, device="cuda")
    for step in range(70):                                            # through several page boundaries of every row
        k_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        v_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
        out, lse = T.tangram_decode_step(dp, q, k_new, v_new, pool, kv_dev, free_dev, overflow=over)
    torch.cuda.synchronize()
    starved = T.tangram_download_tables(dp, t)
    assert t.n_pages_used > int(np.flatnonzero(np.isin(free, list(bad)))[0]), "no bad entry was reached"
    assert starved > 0
    held = t.tbl_pages[t.tbl_pages >= 0]
    assert held.max() < n_pages and not np.isin(held, list(bad)).any()
    after = bits(big)
    assert np.array_equal(after[n_pages:], before[n_pages:]), "a guard page behind the pool was written"
    unnamed = np.setdiff1d(np.arange(n_pages), held)
    assert np.array_equal(after[unnamed], before[unnamed]), "a page that no table names was written"
    kv_now = kv_dev.cpu().numpy()
    assert (kv_now > kv).all()
    to = O.Tables(R=t.R, H=t.H, C=t.C, Hp=t.Hp, P=t.P, perm=t.perm, cluster_of=t.cluster_of, slot_of=t.slot_of,
                  tbl_indptr=t.tbl_indptr, tbl_pages=t.tbl_pages, n_pages_used=t.n_pages_used)
    ro, rl, _ = O.attention(q.cpu(), pool.cpu(), to, kv_now, wl.Hq, wl.d)
    check(out, lse, ro, rl, "last step after poisoned free-list entries")


def test_append_kv_never_stores_through_a_page_id_outside_the_pool():
    """tangram_extend_tables_device does not know the pool's size, so a wrong free-list entry can reach the tables;
    tangram_append_kv then keeps the row's length, counts it in overflow and stores nothing for it."""
    wl = I.make_random_workload(47, R=3, H=4, G=2, d=128, C=2, max_ctx=150)
    B, kv, t, free, n_pages, bad = _poisoned_free_list(wl, headroom=4)
    # full rows, so that the very next token of every row needs the page handed out below
    full = slot_capacity(t, wl) - 4 * wl.P
    g = torch.Generator(device="cuda").manual_seed(10)
    big = torch.randn(n_pages + 4, t.Hp, 2, wl.P, wl.d, generator=g, device="cuda").bfloat16()
    pool = big[:n_pages]
    before = bits(big).copy()
    pl = T.tangram_plan_partitions(t, B, slot_capacity(t, wl), 8, wl.granule, 1, T.MODE_BALANCED, 0, 0, 0)
    dp = T.tangram_upload(t, pl)
    kv_dev = torch.from_numpy(full.astype(np.int32)).cuda()
    T.tangram_extend_tables_device(dp, kv_dev, torch.from_numpy(free).cuda())
    T.tangram_download_tables(dp, t)
    rows = np.arange(wl.R)[:, None] * t.C + t.cluster_of[None, :]
    new_page = t.tbl_pages[t.tbl_indptr[rows] + full // wl.P]            # the page every head's next token falls in
    is_bad = (new_page < 0) | (new_page >= n_pages)
    assert is_bad.any() and not is_bad.all()
    k_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
    v_new = torch.randn(wl.R, wl.H, wl.d, generator=g, device="cuda").bfloat16()
    over = torch.zeros(1, dtype=torch.int32, device="cuda")
    T.tangram_append_kv(dp, k_new, v_new, pool, kv_dev, overflow=over)
    torch.cuda.synchronize()
    assert np.array_equal(kv_dev.cpu().numpy(), full + (~is_bad).astype(np.int32))
    assert int(over.item()) == int(is_bad.sum())
    after = bits(big)
    assert np.array_equal(after[n_pages:], before[n_pages:])
    good_pages = np.unique(new_page[~is_bad])
    untouched = np.setdiff1d(np.arange(n_pages), good_pages)
    assert np.array_equal(after[untouched], before[untouched])
    assert not np.array_equal(after[good_pages], before[good_pages])
