"""Host side of the product (C ABI: reserve / tables / planner) against the CPU oracle: bit-exact
budgets, page tables and plans on the five BASELINE configs (full size) and on random shapes, the
error contract, and the exported symbols.  No GPU needed: these calls are host-pure."""
import ctypes
import os
import re

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

from oracle import tangram_oracle as O
from paper_2606_06302_b200 import binding as T
from paper_2606_06302_b200 import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "tangram.h")).read()
    declared = set(re.findall(r"\b(tangram_[a-z_]+)\s*\(", hdr))
    assert declared == set(T.EXPORTS)
    lib = ctypes.CDLL(T.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def both_sides(wl, n_pool_pages=None, flags=0, identity=False):
    Bo, reso, kvo = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    Bp, resp, kvp = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    assert Bo.tobytes() == Bp.tobytes() and np.array_equal(reso, resp) and np.array_equal(kvo, kvp)
    need = T.tangram_pages_needed(Bp, resp, wl.C, wl.P)
    n_pool = n_pool_pages or int(np.ceil(1.05 * need))
    free = I.make_free_pages(wl, n_pool, identity=identity)
    to, kvo2 = O.build_ragged_tables(Bo, reso, wl.C, wl.P, free, flags, kvo)
    tp, kvp2 = T.tangram_build_ragged_tables(Bp, resp, wl.C, wl.P, free, flags, kvp)
    assert need == to.n_pages_used == tp.n_pages_used
    for f in ("perm", "cluster_of", "slot_of", "tbl_indptr", "tbl_pages"):
        a, b = getattr(to, f), getattr(tp, f)
        assert a.dtype == b.dtype and np.array_equal(a, b), f
    assert (to.R, to.H, to.C, to.Hp, to.P) == (tp.R, tp.H, tp.C, tp.Hp, tp.P)
    assert np.array_equal(kvo2, kvp2)
    return Bo, kvo2, to, tp


def plans_equal(po, pp):
    assert (po.W, po.n_static, po.mode, po.n_items, po.n_part_slots) == \
        (pp.W, pp.n_static, pp.mode, pp.n_items, pp.n_part_slots)
    assert np.array_equal(po.split_map, pp.split_map)
    assert po.items.shape == pp.items.shape and np.array_equal(po.items, pp.items)
    assert np.array_equal(po.worker_indptr, pp.worker_indptr)
    assert np.array_equal(po.part_indptr, pp.part_indptr)


@pytest.mark.parametrize("name", I.CONFIG_NAMES)
def test_full_configs_bit_exact(name):
    wl = I.make_workload(name)
    B, kv, to, tp = both_sides(wl)
    for mode in (O.MODE_BALANCED, O.MODE_SPLITMAP, O.MODE_STATIC_EVEN):
        for W, c0 in ((148, 1), (296, 0)):
            po = O.plan_partitions(to, B, kv, W, wl.granule, c0, mode)
            pp = T.tangram_plan_partitions(tp, B, kv, W, wl.granule, c0, mode)
            plans_equal(po, pp)
    for dyn, J in ((250, 4), (100, 1), (999, 16)):
        po = O.plan_partitions(to, B, kv, 148, wl.granule, 1, O.MODE_BALANCED, 0, dyn, J)
        pp = T.tangram_plan_partitions(tp, B, kv, 148, wl.granule, 1, T.MODE_BALANCED, 0, dyn, J)
        plans_equal(po, pp)
        assert pp.W == 148 * (1 + J) and pp.n_static == 148


def test_fill_group_and_identity_free_list():
    wl = I.make_workload("skew", R=2, ctx_div=16)
    B, kv, to, tp = both_sides(wl, flags=O.FLAG_FILL_GROUP, identity=True)
    assert kv[0, 7] == kv[0, 0] == wl.ctx_len[0] and kv[0, 1] < 100   # the short heads sharing the long head's cluster fill up
    po = O.plan_partitions(to, B, kv, 8, 64, 1, O.MODE_BALANCED)
    plans_equal(po, T.tangram_plan_partitions(tp, B, kv, 8, 64, 1, T.MODE_BALANCED))


@settings(max_examples=60, deadline=None)
@given(seed=st.integers(0, 10**6), R=st.integers(1, 5), Hp=st.integers(1, 4), C=st.integers(1, 4),
       W=st.integers(1, 40), c0=st.integers(0, 3), gmul=st.integers(1, 4), mode=st.integers(0, 2),
       splits=st.integers(0, 5), dyn=st.integers(0, 999), J=st.integers(0, 6))
def test_random_shapes_bit_exact(seed, R, Hp, C, W, c0, gmul, mode, splits, dyn, J):
    if dyn == 0 or J == 0:
        dyn = J = 0
    wl = I.make_random_workload(seed, R=R, H=Hp * C, G=1, d=64, C=C, max_ctx=700)
    B, kv, to, tp = both_sides(wl)
    g = wl.P * gmul
    po = O.plan_partitions(to, B, kv, W, g, c0, mode, splits, dyn, J)
    pp = T.tangram_plan_partitions(tp, B, kv, W, g, c0, mode, splits, dyn, J)
    plans_equal(po, pp)


def test_zero_length_sequences():
    wl = I.make_random_workload(5, R=3, H=4, G=1, d=64, C=2)
    wl.demand[:, 1] = 0
    wl.demand[2, :] = 0
    B, kv, to, tp = both_sides(wl)
    assert kv[2].sum() == 0
    for mode in range(3):
        plans_equal(O.plan_partitions(to, B, kv, 7, 64, 1, mode), T.tangram_plan_partitions(tp, B, kv, 7, 64, 1, mode))


def test_error_contract():
    with pytest.raises(T.TangramError) as e:
        T.tangram_reserve_budgets([0.0], [0.0], 2.0, [10])
    assert e.value.code == T.ERR_INVALID_ARG and "B=" in str(e.value)
    with pytest.raises(T.TangramError):
        T.tangram_reserve_budgets([0.5], [0.0], 2.0, [0])
    with pytest.raises(T.TangramError):
        T.tangram_reserve_budgets([0.5], [0.0], 2.0, [5], [[-1]])
    B, res, kv = T.tangram_reserve_budgets([0.5, 0.25, 0.5], [0, 0, 0], 2.0, [100])
    with pytest.raises(T.TangramError) as e:
        T.tangram_build_ragged_tables(B, res, 2, 16, np.arange(100))           # H % C != 0
    assert e.value.code == T.ERR_INVALID_ARG
    with pytest.raises(T.TangramError) as e:
        T.tangram_build_ragged_tables(B, res, 3, 0, np.arange(100))            # page_size <= 0
    assert e.value.code == T.ERR_INVALID_ARG
    with pytest.raises(T.TangramError) as e:
        T.tangram_build_ragged_tables(B, res, 3, 16, np.arange(3))             # needs 4+2+4 pages
    assert e.value.code == T.ERR_OUT_OF_PAGES
    t, _ = T.tangram_build_ragged_tables(B, res, 3, 16, np.arange(100))
    with pytest.raises(T.TangramError) as e:
        T.tangram_plan_partitions(t, B, kv, 4, 24, 0, T.MODE_BALANCED)          # granule % P != 0
    assert e.value.code == T.ERR_INVALID_ARG
    with pytest.raises(T.TangramError):
        T.tangram_plan_partitions(t, B, kv, 0, 64, 0, T.MODE_BALANCED)
    with pytest.raises(T.TangramError):
        T.tangram_plan_partitions(t, B, kv + 1000, 4, 64, 0, T.MODE_BALANCED)   # kv_len beyond the table
    with pytest.raises(T.TangramError):
        T.tangram_plan_partitions(t, B, kv, 4, 64, 0, 7)
    for dyn, J in ((250, 0), (0, 2), (1000, 2), (100, 17)):
        with pytest.raises(T.TangramError) as e:
            T.tangram_plan_partitions(t, B, kv, 4, 64, 0, T.MODE_BALANCED, 0, dyn, J)
        assert e.value.code == T.ERR_INVALID_ARG


def test_skew_balance_numbers():
    """SURVEY §8(d) scratch check: Skew, W=296, g=64 -> at most R*H+W-1 items, token spread < 1 %; STATIC_EVEN S=3 leaves 43 691-token
    chunks next to a ~7.3K-token fair share."""
    wl = I.make_workload("skew")
    B, kv, to, tp = both_sides(wl)
    pl = T.tangram_plan_partitions(tp, B, kv, 296, 64, 0, T.MODE_BALANCED)
    assert 296 <= pl.n_items <= wl.R * wl.H + 296 - 1
    tok = np.array([sum(int(it[5] - it[4]) for it in pl.items[pl.worker_indptr[w]:pl.worker_indptr[w + 1]])
                    for w in range(296)])
    assert (tok.max() - tok.min()) / tok.mean() < 0.01
    ps = T.tangram_plan_partitions(tp, B, kv, 296, 64, 0, T.MODE_STATIC_EVEN)
    assert ps.split_map.tolist() == [3, 3]
    assert max(int(it[5] - it[4]) for it in ps.items) == 43712           # ceil(2048/3)=683 granules * 64


# ---------------------------------------------------------------------------- NEXT-3 / NEXT-4 (host, bit-exact)
@pytest.mark.parametrize("name", I.CONFIG_NAMES)
def test_account_pages_bit_exact_on_the_configs(name):
    wl = I.make_workload(name)
    B, res, _ = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    for Hp in [d for d in (1, 2, 4, 8) if wl.H % d == 0]:
        for pol in (T.GROUP_CLUSTERED, T.GROUP_ADJACENT):
            got = T.tangram_account_pages(B, res, wl.ctx_len, Hp, wl.P, pol)
            want = O.account_pages(B, res, wl.ctx_len, Hp, wl.P, pol)
            assert got == want, (Hp, pol)                 # integers and the two fp64 ratios, bit for bit
    # the tables the product builds occupy exactly the accounted pages
    assert T.tangram_account_pages(B, res, wl.ctx_len, wl.Hp, wl.P, T.GROUP_CLUSTERED)["pages_alloc"] == \
        T.tangram_pages_needed(B, res, wl.C, wl.P)


@settings(max_examples=60, deadline=None)
@given(st.integers(1, 5), st.sampled_from([2, 4, 6, 8, 12]), st.integers(0, 2 ** 31 - 1))
def test_account_pages_random(R, H, seed):
    rng = np.random.default_rng(seed)
    B = np.round(rng.uniform(0.01, 1.0, size=H), 2)          # rounded: equal budgets (ties) do occur
    ctx = rng.integers(1, 3000, size=R).astype(np.int32)
    res = np.maximum(1, np.ceil(B[None, :] * ctx[:, None])).astype(np.int32)
    P = int(rng.choice([1, 8, 16, 32]))
    for Hp in [d for d in range(1, H + 1) if H % d == 0]:
        for pol in (T.GROUP_CLUSTERED, T.GROUP_ADJACENT):
            assert T.tangram_account_pages(B, res, ctx, Hp, P, pol) == O.account_pages(B, res, ctx, Hp, P, pol)


def test_account_pages_error_contract():
    B, res, ctx = np.array([0.5, 0.5]), np.array([[5, 5]], dtype=np.int32), np.array([10], dtype=np.int32)
    for args in ((B, res, ctx, 3, 16, 0), (B, res, ctx, 2, 0, 0), (B, res, ctx, 2, 16, 7), (B, -res, ctx, 2, 16, 0),
                 (B, res, ctx * 0, 2, 16, 0)):
        with pytest.raises(T.TangramError) as e:
            T.tangram_account_pages(*args)
        assert e.value.code == T.ERR_INVALID_ARG


@settings(max_examples=60, deadline=None)
@given(st.integers(1, 60), st.integers(1, 9), st.integers(0, 2 ** 31 - 1), st.sampled_from([0.0, 1.0, 2.0, 2.5]))
def test_calibrate_budgets_bit_exact(n, H, seed, alpha):
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.0, 1.0, size=(n, H))
    mo, so, Bo = O.calibrate_budgets(x, alpha)
    mp, sp, Bp = T.tangram_calibrate_budgets(x, alpha)
    assert mo.tobytes() == mp.tobytes() and so.tobytes() == sp.tobytes() and Bo.tobytes() == Bp.tobytes()


def test_calibrate_then_reserve_pipeline_and_errors():
    """Calibration feeds Budget Reservation: 50 synthetic samples of the 8b head profile (:262)."""
    wl = I.make_workload("8b")
    x = I.make_calibration_ratios(wl, 50)
    mu, sigma, B = T.tangram_calibrate_budgets(x, wl.alpha)
    B2, res, kv = T.tangram_reserve_budgets(mu, sigma, wl.alpha, wl.ctx_len, wl.demand)
    assert B.tobytes() == B2.tobytes()
    assert (np.abs(mu - wl.mu) < 0.1 * wl.mu).all()           # the samples were drawn around the nominal ratios
    with pytest.raises(T.TangramError):
        T.tangram_calibrate_budgets(np.array([[np.nan]]), 2.0)
    with pytest.raises(T.TangramError):
        T.tangram_calibrate_budgets(np.zeros((0, 3)), 2.0)


def test_header_is_plain_c_and_host_path_runs_from_c(tmp_path):
    """include/tangram.h compiles as strict C99 and a plain C program drives the host side of the path through
    the shared library (no Python, no torch types): hand-evaluated values of a1 / a2 / a3 / NEXT-3 / NEXT-4."""
    import subprocess
    src = os.path.join(ROOT, "tests", "c_abi", "host_path.c")
    exe = str(tmp_path / "host_path")
    libdir = os.path.dirname(T.LIB_PATH)
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(ROOT, "include"),
                           src, "-o", exe, "-L", libdir, "-ltangram", "-Wl,-rpath," + libdir])
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    assert "c_abi host path ok" in out.stdout


def test_host_code_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the host side (tangram_host.cpp: reserve, tables, growth, planner, accounting, calibration) built
    with -fsanitize=address,undefined together with the plain-C caller and run: no report, same hand-evaluated
    values.  The CUDA side cannot be built this way; it is covered by guard regions / NaN poison on the GPU."""
    import subprocess
    csrc = os.path.join(ROOT, "paper_2606_06302_b200", "csrc")
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]
    obj_c, obj_cpp, exe = str(tmp_path / "host_path.o"), str(tmp_path / "tangram_host.o"), str(tmp_path / "host_path_san")
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", *san, "-I", os.path.join(ROOT, "include"),
                           "-c", os.path.join(ROOT, "tests", "c_abi", "host_path.c"), "-o", obj_c])
    subprocess.check_call(["g++", "-std=c++17", "-Wall", "-Wextra", "-ffp-contract=off", "-fopenmp", *san,
                           "-I", os.path.join(ROOT, "include"), "-I", csrc, "-c", os.path.join(csrc, "tangram_host.cpp"),
                           "-o", obj_cpp])
    subprocess.check_call(["g++", *san, "-fopenmp", obj_c, obj_cpp, "-o", exe])
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    out = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=120)
    assert out.returncode == 0, out.stderr + out.stdout
    assert "c_abi host path ok" in out.stdout and "runtime error" not in out.stderr and "AddressSanitizer" not in out.stderr


def test_default_dynamic_tail_rule():
    for name in I.CONFIG_NAMES:
        wl = I.make_workload(name)
        _, _, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
        for W in (1, 148, 296):
            assert T.tangram_default_dynamic_tail(kv, W, wl.granule, 1) == O.default_dynamic_tail(kv, W, wl.granule, 1)
    wl = I.make_workload("tiny")
    _, _, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    assert T.tangram_default_dynamic_tail(kv, 148, 64, 1) == (0, 0)                      # little work per CTA: static
    wl = I.make_workload("8b")
    _, _, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    assert T.tangram_default_dynamic_tail(kv, 148, 64, 1) == (500, 4)                    # 167 cost units per CTA
    wl = I.make_workload("uniform")
    _, _, kv = T.tangram_reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    assert T.tangram_default_dynamic_tail(kv, 148, 64, 1) == (500, 6)                    # 900 cost units per CTA
    for units, want in ((47, (0, 0)), (48, (500, 4)), (383, (500, 4)), (384, (500, 6))):
        edge = np.full((1, 1), 64 * (units - 1), dtype=np.int32)                          # units - 1 granules + 1 overhead
        assert T.tangram_default_dynamic_tail(edge, 1, 64, 1) == O.default_dynamic_tail(edge, 1, 64, 1) == want


# ---------------------------------------------------------------------------- NEXT-4: growable tables (host path)
def tables_equal(to, tp):
    for f in ("tbl_indptr", "tbl_pages", "row_pages"):
        a, b = getattr(to, f), getattr(tp, f)
        assert a.dtype == b.dtype and np.array_equal(a, b), f
    assert to.n_pages_used == tp.n_pages_used


@pytest.mark.parametrize("name,Hp", [("8b", 1), ("8b", 2), ("8b", 8), ("32b", 1), ("32b", 4), ("uniform", 8), ("skew", 4)])
def test_growable_tables_and_vectorized_update_bit_exact(name, Hp):
    """Tables with growth headroom and 60 block-table updates of a decode loop (lengths + 1 per step, every head
    started a few tokens before its page boundary) on the full-size configs at several heads per page: slot
    layout, page ids, row_pages, free-list cursor and the extended / starved counts equal the oracle's, with one
    thread and with four (the OpenMP row scan) -- and the AVX-512 path equals the scalar path wherever it runs."""
    wl = I.make_workload(name)
    C = wl.H // Hp
    Bo, reso, kvo = O.reserve_budgets(wl.mu, wl.sigma, wl.alpha, wl.ctx_len, wl.demand)
    need = T.tangram_pages_needed(Bo, reso, C, wl.P)
    free = I.make_free_pages(wl, need + 2 * wl.R * C + 3)            # short: every row wants 3 more pages, some a 4th
    to, _ = O.build_ragged_tables(Bo, reso, C, wl.P, free, 0, kvo, headroom_pages=3)
    tp, _ = T.tangram_build_ragged_tables(Bo, reso, C, wl.P, free, 0, kvo, headroom_pages=3)
    tp4, _ = T.tangram_build_ragged_tables(Bo, reso, C, wl.P, free, 0, kvo, headroom_pages=3)
    tables_equal(to, tp)
    rng = np.random.default_rng(7)
    # every row starts between 0 and 20 tokens before the end of its pages
    rows = np.arange(wl.R)[:, None] * C + to.cluster_of[None, :]
    kv = np.maximum(to.row_pages[rows] * wl.P - rng.integers(0, 21, size=(wl.R, wl.H)), 0).astype(np.int32)
    tot_ext = tot_starved = 0
    for step in range(60):
        to, starved = O.extend_tables(to, kv, free)
        ext_p, starved_p = T.tangram_extend_tables(tp, kv, free, n_threads=1)
        ext_4, starved_4 = T.tangram_extend_tables(tp4, kv, free, n_threads=4)
        assert starved == starved_p == starved_4 and ext_p == ext_4
        tables_equal(to, tp)
        tables_equal(to, tp4)
        tot_ext, tot_starved = tot_ext + ext_p, tot_starved + starved
        cap = to.row_pages[rows] * wl.P
        kv = np.minimum(kv + 1, cap).astype(np.int32)                # what append_kv leaves (full rows drop)
    assert tot_ext == to.n_pages_used - need and tot_ext > 0 and tot_starved > 0
    assert to.n_pages_used == len(free)                              # the free list was used up, in order
    used = to.tbl_pages[to.tbl_pages >= 0]
    assert sorted(used.tolist()) == sorted(free.tolist())


@settings(max_examples=40, deadline=None)
@given(seed=st.integers(0, 10 ** 6), R=st.integers(1, 40), Hp=st.sampled_from([1, 2, 3, 4]), C=st.integers(1, 4),
       headroom=st.integers(1, 3), P=st.sampled_from([1, 4, 16]))
def test_growable_tables_random_shapes(seed, R, Hp, C, headroom, P):
    rng = np.random.default_rng(seed)
    H = Hp * C
    B = rng.uniform(0.05, 1.0, size=H)
    res = rng.integers(1, 70, size=(R, H)).astype(np.int32)
    need = T.tangram_pages_needed(B, res, C, P)
    free = rng.permutation(need + int(rng.integers(0, 2 * R * C + 1))).astype(np.int32)
    to, _ = O.build_ragged_tables(B, res, C, P, free, headroom_pages=headroom)
    tp, _ = T.tangram_build_ragged_tables(B, res, C, P, free, headroom_pages=headroom)
    tables_equal(to, tp)
    kv = res.copy()
    for step in range(3 * P + 2):
        to, starved = O.extend_tables(to, kv, free)
        ext, starved_p = T.tangram_extend_tables(tp, kv, free, n_threads=int(rng.integers(0, 3)))
        assert starved == starved_p
        tables_equal(to, tp)
        rows = np.arange(R)[:, None] * C + to.cluster_of[None, :]
        kv = np.minimum(kv + rng.integers(0, 2, size=kv.shape), to.row_pages[rows] * P).astype(np.int32)


def test_growable_tables_error_contract():
    B = np.array([0.5, 0.25])
    res = np.array([[20, 10]], dtype=np.int32)
    free = np.arange(10, dtype=np.int32)
    tight, _ = T.tangram_build_ragged_tables(B, res, 2, 16, free)
    assert tight.row_pages is None and len(tight.tbl_pages) == tight.n_pages_used == 3
    with pytest.raises(T.TangramError) as e:                          # no headroom, no row_pages: nothing to grow into
        T._check(T._lib.tangram_extend_tables(ctypes.byref(tight._c()), T._ptr(res), T._ptr(free), ctypes.c_int64(10),
                                              ctypes.c_int32(0), None, None))
    assert e.value.code == T.ERR_INVALID_ARG
    ct = tight._c()
    ct.headroom_pages = 2                                             # headroom asked for without the row_pages array
    rc = T._lib.tangram_build_ragged_tables(T._ptr(B), T._ptr(res), 1, 2, 2, 16, T._ptr(free), ctypes.c_int64(10), 0, None,
                                            ctypes.byref(ct))
    assert rc == T.ERR_INVALID_ARG
    ct.headroom_pages = -1
    rc = T._lib.tangram_build_ragged_tables(T._ptr(B), T._ptr(res), 1, 2, 2, 16, T._ptr(free), ctypes.c_int64(10), 0, None,
                                            ctypes.byref(ct))
    assert rc == T.ERR_INVALID_ARG
    grow, _ = T.tangram_build_ragged_tables(B, res, 2, 16, free, headroom_pages=2)
    assert len(grow.tbl_pages) == 3 + 2 * 2 and grow.row_pages.tolist() == [1, 2]
    # the planner accepts lengths up to the slot capacity (an open-ended plan covers the growth)
    pl = T.tangram_plan_partitions(grow, B, np.array([[64, 48]], dtype=np.int32), 4, 64, 1, T.MODE_BALANCED)
    assert int(pl.items[:, 5].max()) == 64
