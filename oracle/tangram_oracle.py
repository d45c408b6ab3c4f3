"""TEST INFRASTRUCTURE -- CPU oracle for the Tangram hot path (PAPER.md = arxiv/paper_2606_06302).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this.  It shares no code with the CUDA/C++ product (paper_2606_06302_b200/csrc): own
source, own address arithmetic, plain Python / numpy fp64 (the attention part is plain C in
attention_oracle.c, called through ctypes).

What each function follows (citations are PAPER.md lines; "reading Ax" = DESIGN.md §Readings):
  O2 reserve_budgets      Eq. 5 (:158)  B = min(1, mu + alpha*sigma);  Eq. 4 (:154) n = ceil(B N);
                          overflow truncation (:176)
  O3 build_ragged_tables  Budget-Aware Clustering (:192-194, :227-233), per-group page table sized
                          by the group's max budget (:190), slack use (:235)
  O4 split_map            Algorithm 1 (:196-225)
     plan_partitions      modes SPLITMAP (Alg. 1 expanded, reading A16), BALANCED (north_star's
                          equal-bytes work list, reading A2), STATIC_EVEN (FlashDecoding-style
                          uniform num_splits, :120)
  O5 merge                log-sum-exp merge of split-KV partials (implied by split-KV :91, :120)
  O7 topk_indices /       per-head Top-ceil(B N) selection (Eq. 4 :154) and K~ = K[I,:], V~ = V[I,:] (Eq. 1
     compact_topk         :57) written into the ragged pages (NEXT-2; tie rule = reading A30)
  O11 compact_topk_chunk  the same for one prefill chunk, appended behind what the head already holds (compression
                          fused into chunked prefill, :152; NEXT-2 extension)
  O6 append_kv            one decode step's new K/V rows written into the ragged pages (NEXT-1;
                          page layout :190, reading A29: a row is dropped only when its table has no page for it)
  O12 extend_tables       block-table growth during decode (NEXT-4; :85-89 "for every iteration, the scheduler
                          allocates pages", :244 per-group block mappings updated for all groups at once;
                          reading A33)
  O8 account_pages        pages / token-head slots a batch occupies under a grouping policy (monolithic,
                          adjacent, Budget-Aware Clustering; Fig. 7 :168, Fig. 8 :186, Fig. 15 :316-320; NEXT-3)
  O9 calibrate_budgets    mu, sigma of the recorded per-head implicit retention ratios and Eq. 5 (:156-158;
                          population sigma = reading A10; NEXT-4)
  O10 implicit_ratios     the per-head retention ratios a global flat Top-ceil(rho H N) selection implies (Eq. 3
                          :68-77; what Budget Calibration records per sample, :156; NEXT-4)
  O1 attention*           plain softmax(q K~^T / sqrt(d)) V~ through the page tables (Eq. 1 :57)

Pins (every function is pinned; nothing here is "parity unpinned"): tests/test_oracle_pins.py.
Fidelity to the authors' unseen code for the rounding mode of Alg. 1 line 10 (reading A14) and
for how S maps to CTAs (reading A16) cannot be pinned from the paper; they are pinned to the
DESIGN.md readings.
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import subprocess
from typing import List, Optional, Sequence, Tuple

import numpy as np

FLAG_FILL_GROUP = 1
MODE_BALANCED, MODE_SPLITMAP, MODE_STATIC_EVEN = 0, 1, 2


# --------------------------------------------------------------------------------------------
# O2  Budget Reservation  (Eq. 5 :158, Eq. 4 :154, overflow :176)
# --------------------------------------------------------------------------------------------
def reserve_budgets(mu, sigma, alpha: float, ctx_len, demand=None):
    """Returns (B [H] f64, reserved [R][H] i32, kv_len [R][H] i32).

    B_h = min(1, mu_h + alpha*sigma_h) evaluated as one fp64 multiply then one fp64 add
    (reading A9; Python floats never fuse).  reserved = ceil(B_h * N_r) clamped to [1, N_r].
    kv_len = min(demand, reserved) (the overflow rule, :176) or reserved if demand is None."""
    H, R = len(mu), len(ctx_len)
    B = np.empty(H, dtype=np.float64)
    for h in range(H):
        prod = float(alpha) * float(sigma[h])
        b = float(mu[h]) + prod
        b = min(1.0, b)
        if not (b > 0.0):
            raise ValueError(f"budget ratio of head {h} is not in (0,1] (reading A11)")
        B[h] = b
    reserved = np.empty((R, H), dtype=np.int32)
    kv_len = np.empty((R, H), dtype=np.int32)
    for r in range(R):
        N = int(ctx_len[r])
        if N < 1:
            raise ValueError("ctx_len < 1")
        for h in range(H):
            n = int(math.ceil(float(B[h]) * float(N)))
            n = max(1, min(N, n))
            reserved[r, h] = n
            if demand is None:
                kv_len[r, h] = n
            else:
                dm = int(demand[r][h])
                if dm < 0:
                    raise ValueError("demand < 0")
                kv_len[r, h] = min(dm, n)
    return B, reserved, kv_len


# --------------------------------------------------------------------------------------------
# O3  Budget-Aware Clustering + per-(request, cluster) page tables  (§4.2 :190-235)
# --------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Tables:
    R: int
    H: int
    C: int
    Hp: int
    P: int
    perm: np.ndarray        # [H]  pi: sorted position -> head
    cluster_of: np.ndarray  # [H]  head -> cluster
    slot_of: np.ndarray     # [H]  head -> slot inside the cluster's pages
    tbl_indptr: np.ndarray  # [R*C+1] int64, row = r*C + c; a row owns the page SLOTS [indptr[row], indptr[row+1])
    tbl_pages: np.ndarray   # [indptr[-1]] int32 page id of every slot; -1 = slot not assigned yet (growth headroom)
    n_pages_used: int       # pages taken from the free list so far
    row_pages: Optional[np.ndarray] = None   # [R*C] int32 assigned pages per row (None: every slot is assigned)

    def assigned(self, row: int) -> int:
        """Pages row `row` holds (its first `assigned` slots)."""
        if self.row_pages is None:
            return int(self.tbl_indptr[row + 1] - self.tbl_indptr[row])
        return int(self.row_pages[row])


def cluster_heads(B, n_clusters: int):
    """pi = heads stably sorted by B ascending (ties keep head order, reading A6);
    group i = H_p consecutive heads of the sorted order (:231-233)."""
    H = len(B)
    if n_clusters <= 0 or H % n_clusters != 0:
        raise ValueError("H must be a multiple of n_clusters (reading A17)")
    Hp = H // n_clusters
    perm = sorted(range(H), key=lambda h: (float(B[h]), h))
    cluster_of = [0] * H
    slot_of = [0] * H
    for j, h in enumerate(perm):
        cluster_of[h] = j // Hp
        slot_of[h] = j % Hp
    return (np.array(perm, dtype=np.int32), np.array(cluster_of, dtype=np.int32),
            np.array(slot_of, dtype=np.int32))


def build_ragged_tables(B, reserved, n_clusters: int, page_size: int, free_pages,
                        flags: int = 0, kv_len=None, headroom_pages: int = 0):
    """Returns (Tables, kv_len').  Row (r, c) of the tables has ceil(max_{h in c} reserved / P)
    pages (:190) and takes the next entries of `free_pages` in order (reading A27).  With
    FLAG_FILL_GROUP every head's kv_len is raised to its cluster's max reserved (:235).
    headroom_pages > 0 (reading A33): every row is followed by that many page slots that hold no
    page yet (-1) -- room for extend_tables to grow the row during decode without moving it."""
    reserved = np.asarray(reserved)
    R, H = reserved.shape
    if page_size <= 0:
        raise ValueError("page_size <= 0")
    perm, cluster_of, slot_of = cluster_heads(B, n_clusters)
    C, Hp = n_clusters, H // n_clusters
    indptr = [0]
    pages: List[int] = []
    row_pages: List[int] = []
    cursor = 0
    gmax = np.zeros((R, C), dtype=np.int64)
    for r in range(R):
        for c in range(C):
            members = [int(perm[c * Hp + k]) for k in range(Hp)]
            mx = max(int(reserved[r, h]) for h in members)
            gmax[r, c] = mx
            n_pg = -(-mx // page_size)
            if cursor + n_pg > len(free_pages):
                raise MemoryError("out of pages")
            pages.extend(int(free_pages[cursor + i]) for i in range(n_pg))
            pages.extend([-1] * int(headroom_pages))
            cursor += n_pg
            row_pages.append(n_pg)
            indptr.append(len(pages))
    kv_out = None if kv_len is None else np.array(kv_len, dtype=np.int32, copy=True)
    if (flags & FLAG_FILL_GROUP) and kv_out is not None:
        for r in range(R):
            for h in range(H):
                kv_out[r, h] = gmax[r, cluster_of[h]]
    t = Tables(R=R, H=H, C=C, Hp=Hp, P=page_size, perm=perm, cluster_of=cluster_of,
               slot_of=slot_of, tbl_indptr=np.array(indptr, dtype=np.int64),
               tbl_pages=np.array(pages, dtype=np.int32), n_pages_used=cursor,
               row_pages=np.array(row_pages, dtype=np.int32) if headroom_pages else None)
    return t, kv_out


# --------------------------------------------------------------------------------------------
# O12  block-table growth during decode (NEXT-4; :85-89, :244; reading A33)
# --------------------------------------------------------------------------------------------
def extend_tables(t: Tables, kv_len, free_pages):
    """One block-table update for ALL (request, cluster) rows of a batch, run between two decode steps
    ("between consecutive forward passes, a scheduling step requests the pages required for the next
    pass", :89; the per-group block mappings of all groups updated together, :244).

    Reading A33: the free list is the one the tables were built from; its first t.n_pages_used entries are
    taken.  The rows are visited r-major then by cluster.  A row whose LONGEST head has filled the row's
    pages (max_{h in c} kv_len[r][h] >= assigned pages x P) has no room for the next token; it takes the
    next free page, free_pages[n_pages_used], into its first unassigned slot.  A row with no unassigned
    slot left, or reached after the free list ran out, stays as it is and is counted as starved (its full
    heads then drop their next row: append_kv).  At most one page per row and call: a decode step appends
    one token per head.
    Returns (Tables' (a modified copy), n_starved)."""
    if t.row_pages is None:
        raise ValueError("tables were built without growth headroom")
    kv = np.asarray(kv_len)
    P, C, Hp = t.P, t.C, t.Hp
    pages = np.array(t.tbl_pages, dtype=np.int32, copy=True)
    row_pages = np.array(t.row_pages, dtype=np.int32, copy=True)
    cursor = int(t.n_pages_used)
    starved = 0
    for r in range(t.R):
        for c in range(C):
            row = r * C + c
            longest = max(int(kv[r, int(t.perm[c * Hp + k])]) for k in range(Hp))
            have = int(row_pages[row])
            if longest < have * P:
                continue                                  # the next token of every head still fits
            lo, hi = int(t.tbl_indptr[row]), int(t.tbl_indptr[row + 1])
            if have >= hi - lo or cursor >= len(free_pages):
                starved += 1
                continue
            pages[lo + have] = int(free_pages[cursor])
            cursor += 1
            row_pages[row] = have + 1
    return dataclasses.replace(t, tbl_pages=pages, row_pages=row_pages, n_pages_used=cursor), starved


# --------------------------------------------------------------------------------------------
# O4  AoT plans
# --------------------------------------------------------------------------------------------
def split_map(B, perm, Hp: int, n_cta: int) -> np.ndarray:
    """Algorithm 1 (:196-225) for one layer, de-garbled per reading A13:
    Omega = sum_h B_h; if Omega = 0: S = 1; tau = Omega / N_CTA;
    Phi_i = sum_{h in G_i} B_h;  S_i = max(1, round(Phi_i / tau)), round = half-up (A14)."""
    H = len(B)
    C = H // Hp
    S = [1] * C
    omega = 0.0
    for h in range(H):           # head-index order
        omega += float(B[h])
    if omega == 0.0:
        return np.array(S, dtype=np.int32)
    tau = omega / float(n_cta)
    for i in range(C):
        phi = 0.0
        for k in range(Hp):      # perm order inside the group
            phi += float(B[int(perm[i * Hp + k])])
        S[i] = max(1, int(math.floor(phi / tau + 0.5)))
    return np.array(S, dtype=np.int32)


@dataclasses.dataclass
class Plan:
    W: int                      # work lists in total (= n_static * (1 + dyn_rounds) with a dynamic tail)
    n_static: int               # lists 0..n_static-1 are the CTAs' own
    mode: int
    split_map: np.ndarray       # [C] int32 (SPLITMAP: Alg. 1; STATIC_EVEN: constant; BALANCED: Alg. 1, informational)
    items: np.ndarray           # [n_items, 8] int32: req, kv_head, cluster, slot, tok_begin, tok_end, part_slot, n_parts
    worker_indptr: np.ndarray   # [W+1] int64
    part_indptr: np.ndarray     # [R*H+1] int64, seq = r*H + h
    n_items: int
    n_part_slots: int


def _finish(raw: List[Tuple[int, int, int, int, int]], t: Tables, W: int, mode: int, S,
            n_static: Optional[int] = None) -> Plan:
    """raw: (worker, r, h, tok_begin, tok_end) in plan order.  Assigns part_slot / n_parts and
    lays the items out worker-major, plan order kept inside a worker."""
    R, H = t.R, t.H
    count = [0] * (R * H)
    for (_, r, h, _, _) in raw:
        count[r * H + h] += 1
    part_indptr = [0] * (R * H + 1)
    for s in range(R * H):
        part_indptr[s + 1] = part_indptr[s] + count[s]
    # ordinal of an item inside its sequence = token order
    by_seq: dict = {}
    for idx, (_, r, h, tb, _) in enumerate(raw):
        by_seq.setdefault(r * H + h, []).append((tb, idx))
    ordinal = [0] * len(raw)
    for s, lst in by_seq.items():
        for o, (_, idx) in enumerate(sorted(lst)):
            ordinal[idx] = o
    per_worker: List[List[int]] = [[] for _ in range(W)]
    for idx, it in enumerate(raw):
        per_worker[it[0]].append(idx)
    items = np.zeros((len(raw), 8), dtype=np.int32)
    worker_indptr = [0]
    k = 0
    for w in range(W):
        for idx in per_worker[w]:
            _, r, h, tb, te = raw[idx]
            s = r * H + h
            items[k] = (r, h, int(t.cluster_of[h]), int(t.slot_of[h]), tb, te,
                        part_indptr[s] + ordinal[idx], count[s])
            k += 1
        worker_indptr.append(k)
    return Plan(W=W, n_static=W if n_static is None else n_static, mode=mode,
                split_map=np.asarray(S, dtype=np.int32), items=items,
                worker_indptr=np.array(worker_indptr, dtype=np.int64),
                part_indptr=np.array(part_indptr, dtype=np.int64), n_items=len(raw),
                n_part_slots=part_indptr[-1])


def list_weights(n_workers: int, dyn_permille: int, dyn_rounds: int) -> List[int]:
    """Relative sizes of the BALANCED work lists.  No dynamic tail: n_workers
    lists of weight 1.  With a tail of dyn_permille/1000 of the cost handed out in J = dyn_rounds
    rounds (round j < J takes 2^-j of the tail, the last round the rest): the n_workers static
    lists weigh (1000 - dyn) 2^(J-1) each, a list of round j < J weighs dyn 2^(J-1-j), a list of the
    last round weighs dyn."""
    if dyn_rounds == 0:
        return [1] * n_workers
    J = dyn_rounds
    w = [(1000 - dyn_permille) * 2 ** (J - 1)] * n_workers
    for j in range(1, J + 1):
        w += [dyn_permille * 2 ** (J - 1 - j) if j < J else dyn_permille] * n_workers
    return w


def default_dynamic_tail(kv_len, n_workers: int, granule: int, overhead_granules: int) -> Tuple[int, int]:
    """Default (dyn_permille, dyn_rounds) of the BALANCED plan (reading A32, a measured tuning rule, not
    from the paper), by the cost units (granules + per-sequence overhead) a worker gets: fewer than 48 -- the purely
    static plan (0, 0) (no claims, fewer parts to merge); 48 to 383 -- half of the cost axis handed out in 4 rounds;
    384 and more -- in 6 rounds (the longer a CTA streams, the finer the last lists may be)."""
    total = 0
    for n in np.asarray(kv_len, dtype=np.int64).reshape(-1):
        u = -(-int(n) // granule)
        total += u + (overhead_granules if u > 0 else 0)
    if total < 48 * n_workers:
        return (0, 0)
    if total < 384 * n_workers:
        return (500, 4)
    return (500, 6)


def plan_partitions(t: Tables, B, kv_len, n_workers: int, granule: int, overhead_granules: int,
                    mode: int, static_splits: int = 0, dyn_permille: int = 0, dyn_rounds: int = 0) -> Plan:
    """Offline deterministic planner (§4.3).  Sequences are visited r-major, then in `perm`
    order, so neighbours share a page table."""
    kv_len = np.asarray(kv_len)
    R, H, W, g, c0 = t.R, t.H, int(n_workers), int(granule), int(overhead_granules)
    if W < 1 or g < 1 or g % t.P != 0 or c0 < 0:
        raise ValueError("bad planner arguments (granule must be a positive multiple of P)")
    if not (0 <= dyn_permille < 1000 and 0 <= dyn_rounds <= 16 and (dyn_permille > 0) == (dyn_rounds > 0)):
        raise ValueError("bad dynamic-tail arguments")
    S_alg1 = split_map(B, t.perm, t.Hp, W)
    seqs = [(r, int(t.perm[j])) for r in range(R) for j in range(H)]
    raw: List[Tuple[int, int, int, int, int]] = []

    if mode == MODE_BALANCED:
        # north_star: "splits every (request, KV head) sequence into chunks of near-equal KV
        # bytes per CTA".  Cost of a sequence = its granules + c0 granules of fixed overhead.
        u = [-(-int(kv_len[r, h]) // g) for (r, h) in seqs]
        w = [ui + (c0 if ui > 0 else 0) for ui in u]
        T = sum(w)
        lw = list_weights(W, dyn_permille, dyn_rounds)
        n_static, W = W, len(lw)
        cum = [0]
        for x in lw:
            cum.append(cum[-1] + x)
        b = [(T * cum[k]) // cum[W] for k in range(W + 1)]   # list k owns positions [b_k, b_{k+1})
        a = 0
        k = 0
        for i, (r, h) in enumerate(seqs):
            n = int(kv_len[r, h])
            run_start = None
            run_worker = None
            for j in range(u[i]):
                pos = a + c0 + j
                while b[k + 1] <= pos:      # worker k owns positions b_k <= pos < b_{k+1}
                    k += 1
                if run_worker != k:
                    if run_start is not None:
                        raw.append((run_worker, r, h, run_start * g, min(n, j * g)))
                    run_start, run_worker = j, k
            if run_start is not None:
                raw.append((run_worker, r, h, run_start * g, n))
            a += w[i]
        return _finish(raw, t, W, mode, S_alg1, n_static)

    if mode == MODE_SPLITMAP:
        S = S_alg1
    elif mode == MODE_STATIC_EVEN:
        s = int(static_splits)
        if s <= 0:                      # smallest S with R*H*S >= W
            s = max(1, -(-W // (R * H)))
        S = np.full(t.C, s, dtype=np.int32)
    else:
        raise ValueError("mode")
    kk = 0
    for (r, h) in seqs:
        n = int(kv_len[r, h])
        npg = -(-n // g)                # granules of this sequence
        Sc = int(S[int(t.cluster_of[h])])
        for j in range(Sc):
            lo = (j * npg) // Sc
            hi = ((j + 1) * npg) // Sc
            tb, te = lo * g, min(n, hi * g)
            if te <= tb:
                continue                # empty chunk dropped
            raw.append((kk % W, r, h, tb, te))
            kk += 1
    return _finish(raw, t, W, mode, S)


# --------------------------------------------------------------------------------------------
# O5  log-sum-exp merge  (textbook; implied by split-KV :91)
# --------------------------------------------------------------------------------------------
def merge(parts: Sequence[Tuple[np.ndarray, float]]):
    """parts: (o_i normalised within its chunk [d] f64, lse_i).  L = m* + ln sum e^{lse_i-m*};
    out = sum e^{lse_i - L} o_i.  Parts with lse = -inf contribute nothing."""
    live = [(np.asarray(o, dtype=np.float64), float(l)) for (o, l) in parts if l != -math.inf]
    if not live:
        d = len(parts[0][0]) if parts else 0
        return np.zeros(d, dtype=np.float64), -math.inf
    mstar = max(l for (_, l) in live)
    tot = 0.0
    for (_, l) in live:
        tot += math.exp(l - mstar)
    L = mstar + math.log(tot)
    out = np.zeros_like(live[0][0])
    for (o, l) in live:
        out = out + math.exp(l - L) * o
    return out, L


# --------------------------------------------------------------------------------------------
# O6  KV append of one decode step (NEXT-1; page layout :190, capacity bound :176)
# --------------------------------------------------------------------------------------------
def append_kv(pool_bits: np.ndarray, t: Tables, kv_len, k_new_bits: np.ndarray, v_new_bits: np.ndarray):
    """One decode step's new K/V row of every (request, KV head) written behind its retained tokens.

    pool_bits  uint16 [n_pages][Hp][2][P][d] (raw bf16 bits; a modified COPY is returned)
    k_new_bits, v_new_bits  uint16 [R][H][d]
    Rule (reading A29): the row goes to token index n = kv_len[r][h] of head h, i.e. to
    pool[tbl_pages[tbl_indptr[r*C + c] + n // P]][slot][kv][n % P]; kv_len[r][h] becomes n + 1.  If the
    (request, cluster) table holds no page for token n (n >= its assigned pages x P: a table without
    growth headroom that is full, or a row that extend_tables could not serve) the row is dropped and
    counted as an overflow.
    Returns (pool', kv_len', n_overflow)."""
    pool = np.array(pool_bits, dtype=np.uint16, copy=True)
    kv = np.array(kv_len, dtype=np.int32, copy=True)
    over = 0
    for r in range(t.R):
        for h in range(t.H):
            c, s = int(t.cluster_of[h]), int(t.slot_of[h])
            lo = int(t.tbl_indptr[r * t.C + c])
            n = int(kv[r, h])
            if n >= t.assigned(r * t.C + c) * t.P:
                over += 1
                continue
            page = int(t.tbl_pages[lo + n // t.P])
            pool[page, s, 0, n % t.P, :] = k_new_bits[r, h, :]
            pool[page, s, 1, n % t.P, :] = v_new_bits[r, h, :]
            kv[r, h] = n + 1
    return pool, kv, over


# --------------------------------------------------------------------------------------------
# O7  per-head Top-k selection + compaction into the ragged pages (NEXT-2; Eq. 4 :154, Eq. 1 :57)
# --------------------------------------------------------------------------------------------
def topk_indices(scores, k: int) -> np.ndarray:
    """I = Top(k, s) (Eq. 4): the k highest-scoring token indices, returned in ascending token order
    (storage order = logical order, reading A22).  Scores are compared as the fp32 values they are;
    among equal scores the lower token index wins (reading A30: the paper does not break ties)."""
    s = np.asarray(scores, dtype=np.float32)
    order = sorted(range(len(s)), key=lambda i: (-float(s[i]), i))
    return np.array(sorted(order[:k]), dtype=np.int64)


def compact_topk(pool_bits: np.ndarray, t: Tables, scores, k_dense_bits, v_dense_bits, ctx_len, keep):
    """K~ = K[I,:], V~ = V[I,:] (Eq. 1) with I = Top(keep[r][h], s_{r,h}[:N_r]) (Eq. 4) written into the
    ragged pages of head h in token order.

    pool_bits              uint16 [n_pages][Hp][2][P][d] (a modified COPY is returned)
    scores                 float32 [R][H][n_max]   (entries >= ctx_len[r] are ignored)
    k_dense_bits, v_dense_bits  uint16 [R][H][n_max][d]  the uncompressed cache
    keep                   int [R][H]  tokens to retain (= kv_len of a1; <= ctx_len and <= table capacity)
    Returns (pool', indices) with indices[r][h] the retained token indices."""
    pool = np.array(pool_bits, dtype=np.uint16, copy=True)
    out_idx = [[None] * t.H for _ in range(t.R)]
    for r in range(t.R):
        N = int(ctx_len[r])
        for h in range(t.H):
            k = int(keep[r][h])
            if k > N:
                raise ValueError("keep > ctx_len")
            c, sl = int(t.cluster_of[h]), int(t.slot_of[h])
            lo, hi = int(t.tbl_indptr[r * t.C + c]), int(t.tbl_indptr[r * t.C + c + 1])
            if k > t.assigned(r * t.C + c) * t.P:
                raise ValueError("keep exceeds the table capacity")
            idx = topk_indices(np.asarray(scores[r][h])[:N], k)
            out_idx[r][h] = idx
            for pos, tok in enumerate(idx):
                page = int(t.tbl_pages[lo + pos // t.P])
                pool[page, sl, 0, pos % t.P, :] = k_dense_bits[r, h, tok, :]
                pool[page, sl, 1, pos % t.P, :] = v_dense_bits[r, h, tok, :]
    return pool, out_idx


# --------------------------------------------------------------------------------------------
# O11  per-chunk Top-k + compaction appended behind the retained tokens (:152 "each prefill chunk is compressed
#      as soon as its KV cache is generated"; Eq. 4 applied to the chunk, Eq. 1 into the ragged pages)
# --------------------------------------------------------------------------------------------
def compact_topk_chunk(pool_bits: np.ndarray, t: Tables, scores, k_dense_bits, v_dense_bits, chunk_len, keep, kv_len):
    """One prefill chunk of chunk_len[r] tokens per request: I = Top(keep[r][h], s_{r,h}[:chunk_len[r]]) and the
    rows K[I,:], V[I,:] of the CHUNK written, in ascending token order, to token slots
    kv_len[r][h] .. kv_len[r][h] + keep[r][h] - 1 of head h's ragged pages; the length grows by keep.
    scores [R][H][n_max] f32, k/v_dense_bits uint16 [R][H][n_max][d] hold the chunk.  Raises if a head would
    exceed its table capacity (:176) or keep > chunk_len.
    Returns (pool', kv_len', indices) with indices[r][h] the retained token indices inside the chunk."""
    pool = np.array(pool_bits, dtype=np.uint16, copy=True)
    kv = np.array(kv_len, dtype=np.int32, copy=True)
    out_idx = [[None] * t.H for _ in range(t.R)]
    for r in range(t.R):
        N = int(chunk_len[r])
        for h in range(t.H):
            k = int(keep[r][h])
            if k > N:
                raise ValueError("keep > chunk_len")
            c, sl = int(t.cluster_of[h]), int(t.slot_of[h])
            lo, hi = int(t.tbl_indptr[r * t.C + c]), int(t.tbl_indptr[r * t.C + c + 1])
            base = int(kv[r, h])
            if base + k > t.assigned(r * t.C + c) * t.P:
                raise ValueError("chunk exceeds the table capacity")
            idx = topk_indices(np.asarray(scores[r][h])[:N], k)
            out_idx[r][h] = idx
            for j, tok in enumerate(idx):
                pos = base + j
                page = int(t.tbl_pages[lo + pos // t.P])
                pool[page, sl, 0, pos % t.P, :] = k_dense_bits[r, h, tok, :]
                pool[page, sl, 1, pos % t.P, :] = v_dense_bits[r, h, tok, :]
            kv[r, h] = base + k
    return pool, kv, out_idx


# --------------------------------------------------------------------------------------------
# O8  page accounting under a grouping policy (NEXT-3; Fig. 7 :168, :190, :235-242, Fig. 15 :316-320)
# --------------------------------------------------------------------------------------------
GROUP_CLUSTERED, GROUP_ADJACENT = 0, 1


def account_pages(B, reserved, ctx_len, Hp: int, page_size: int, policy: int) -> dict:
    """Memory a batch occupies when H_p heads share a page table sized by the group's largest reservation
    (:190).  policy CLUSTERED groups H_p consecutive heads of the budget-sorted order (:227-233), ADJACENT
    groups heads in index order ("naively grouping adjacent heads", :192); H_p = H is the monolithic page of
    one layer (Fig. 7(a)).  Unit = token-head slot (one token of one head, K and V).
      pages_alloc  = sum_r sum_groups ceil(max_{h in g} reserved[r][h] / P)   (pages of H_p x 2 x P x d elements)
      slots_alloc  = H_p * P * pages_alloc
      slots_exact  = sum_r sum_h P * ceil(reserved[r][h] / P)                 (every head its own table)
      slots_full   = sum_r H * P * ceil(N_r / P)                              (uncompressed cache)
      slots_used   = sum_r sum_h reserved[r][h]
      tables       = R * H / H_p                                              (block tables to manage, :244)
      reclaimed_frac = 1 - slots_alloc / slots_full   ("memory reclaimed, fraction of the full KV cache", Fig. 15)
      fragmentation  = (slots_alloc - slots_used) / slots_alloc               (allocated slots holding no retained
                                                                               token; reading A31)"""
    B = np.asarray(B, dtype=np.float64)
    res = np.asarray(reserved, dtype=np.int64)
    R, H = res.shape
    P = int(page_size)
    if Hp < 1 or H % Hp != 0 or P < 1:
        raise ValueError("bad H_p / page size")
    if policy == GROUP_CLUSTERED:
        order = sorted(range(H), key=lambda h: (B[h], h))
    elif policy == GROUP_ADJACENT:
        order = list(range(H))
    else:
        raise ValueError("bad policy")
    pages = 0
    exact = 0
    full = 0
    used = 0
    for r in range(R):
        for g in range(H // Hp):
            longest = max(int(res[r, order[g * Hp + j]]) for j in range(Hp))
            pages += -(-longest // P)
        for h in range(H):
            exact += P * (-(-int(res[r, h]) // P))
            used += int(res[r, h])
        full += H * P * (-(-int(ctx_len[r]) // P))
    alloc = Hp * P * pages
    return dict(pages_alloc=pages, slots_alloc=alloc, slots_exact=exact, slots_full=full, slots_used=used,
                tables=R * (H // Hp), reclaimed_frac=1.0 - float(alloc) / float(full),
                fragmentation=float(alloc - used) / float(alloc))


# --------------------------------------------------------------------------------------------
# O9  Budget Calibration (NEXT-4; :156-158, Eq. 5)
# --------------------------------------------------------------------------------------------
def calibrate_budgets(ratios, alpha: float):
    """ratios[i][h] = implicit retention ratio head h received on calibration sample i (:156).  Returns
    (mu, sigma, B): mu_h = (sum_i x_ih) / n and sigma_h = sqrt((sum_i (x_ih - mu_h)^2) / n) -- the
    population standard deviation (reading A10: the paper says "standard deviation" only) -- both summed in
    sample order in fp64, and B_h = min(1, mu_h + alpha * sigma_h) (Eq. 5)."""
    x = np.asarray(ratios, dtype=np.float64)
    n, H = x.shape
    if n < 1:
        raise ValueError("no samples")
    mu = np.zeros(H)
    sigma = np.zeros(H)
    B = np.zeros(H)
    for h in range(H):
        acc = 0.0
        for i in range(n):
            acc = acc + float(x[i, h])
        m = acc / float(n)
        acc2 = 0.0
        for i in range(n):
            dlt = float(x[i, h]) - m
            acc2 = acc2 + dlt * dlt
        sd = math.sqrt(acc2 / float(n))
        mu[h], sigma[h] = m, sd
        B[h] = min(1.0, m + alpha * sd)
    return mu, sigma, B


# --------------------------------------------------------------------------------------------
# O10  implicit per-head retention ratios of the global flat Top-k (NEXT-4; Eq. 3 :68-77, :156)
# --------------------------------------------------------------------------------------------
def implicit_ratios(scores, ctx_len, rho: float):
    """I = Top(ceil(rho H N), s^flat) over the flattened scores of all H heads of a request (Eq. 3), and the
    ratio |{(h, t) in I}| / N each head receives from it -- the quantity Budget Calibration records on every
    sample context (:156).  s^flat is head-major (index h N + t); ties go to the lower flat index (reading
    A30 applied to the flat vector).  scores [R][H][n_max] f32 (entries >= ctx_len[r] ignored).
    Returns (counts [R][H] int64, ratios [R][H] f64 = counts / N_r)."""
    sc = np.asarray(scores, dtype=np.float32)
    R, H = sc.shape[0], sc.shape[1]
    counts = np.zeros((R, H), dtype=np.int64)
    ratios = np.zeros((R, H), dtype=np.float64)
    for r in range(R):
        N = int(ctx_len[r])
        flat = np.concatenate([sc[r, h, :N] for h in range(H)])
        k = int(math.ceil(rho * float(H * N)))
        k = max(0, min(k, H * N))
        for i in topk_indices(flat, k):
            counts[r, int(i) // N] += 1
        for h in range(H):
            ratios[r, h] = float(counts[r, h]) / float(N)
    return counts, ratios


# --------------------------------------------------------------------------------------------
# O1  attention through the page tables (plain C, fp64; attention_oracle.c)
# --------------------------------------------------------------------------------------------
_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_attention.so")
_lib = None


def build_c(force: bool = False) -> str:
    src = os.path.join(_HERE, "attention_oracle.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", _SO, src, "-lm"])
    return _SO


def _c():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build_c())
        _lib.tangram_oracle_attention_pairs.restype = ctypes.c_int
    return _lib


def _u16(x) -> np.ndarray:
    """bf16 torch tensor (or uint16 ndarray) -> contiguous uint16 ndarray of the raw bits."""
    if isinstance(x, np.ndarray):
        assert x.dtype == np.uint16
        return np.ascontiguousarray(x)
    import torch
    assert x.dtype == torch.bfloat16 and x.device.type == "cpu"
    return x.contiguous().view(torch.int16).numpy().view(np.uint16)


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def attention_pairs(q, pool, t: Tables, kv_len, Hq: int, d: int, pairs, n_threads: int = 0,
                    sm_scale: Optional[float] = None):
    """Attention for the listed (r, j) pairs.  Returns (out [n,d] f64, lse [n] f64, threads).
    sm_scale: softmax scale (the scores are (q . k) * sm_scale); None = 1/sqrt(d) (reading A19)."""
    qb, pb = _u16(q), _u16(pool)
    pairs = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    kv = np.ascontiguousarray(np.asarray(kv_len, dtype=np.int32))
    n = pairs.shape[0]
    out = np.zeros((n, d), dtype=np.float64)
    lse = np.zeros(n, dtype=np.float64)
    ip = np.ascontiguousarray(t.tbl_indptr, dtype=np.int64)
    pg = np.ascontiguousarray(t.tbl_pages, dtype=np.int32)
    co = np.ascontiguousarray(t.cluster_of, dtype=np.int32)
    so = np.ascontiguousarray(t.slot_of, dtype=np.int32)
    used = _c().tangram_oracle_attention_pairs(
        _p(qb), _p(pb), _p(ip), _p(pg), _p(co), _p(so), _p(kv),
        ctypes.c_int32(t.R), ctypes.c_int32(t.H), ctypes.c_int32(Hq), ctypes.c_int32(t.C),
        ctypes.c_int32(t.Hp), ctypes.c_int32(t.P), ctypes.c_int32(d), _p(pairs),
        ctypes.c_int64(n), ctypes.c_double(0.0 if sm_scale is None else float(sm_scale)), _p(out), _p(lse),
        ctypes.c_int32(n_threads))
    return out, lse, int(used)


def attention(q, pool, t: Tables, kv_len, Hq: int, d: int, n_threads: int = 0, sm_scale: Optional[float] = None):
    """Whole batch: out [R][Hq][d] f64, lse [R][Hq] f64."""
    pairs = [(r, j) for r in range(t.R) for j in range(Hq)]
    out, lse, used = attention_pairs(q, pool, t, kv_len, Hq, d, pairs, n_threads, sm_scale)
    return out.reshape(t.R, Hq, d), lse.reshape(t.R, Hq), used


def attend_range(q, pool, t: Tables, Hq: int, d: int, r: int, j: int, t0: int, t1: int,
                 sm_scale: Optional[float] = None):
    """Attention of (r, j) over tokens [t0, t1) only: (o [d] normalised in the range, lse)."""
    qb, pb = _u16(q), _u16(pool)
    out = np.zeros(d, dtype=np.float64)
    lse = ctypes.c_double(0.0)
    ip = np.ascontiguousarray(t.tbl_indptr, dtype=np.int64)
    pg = np.ascontiguousarray(t.tbl_pages, dtype=np.int32)
    co = np.ascontiguousarray(t.cluster_of, dtype=np.int32)
    so = np.ascontiguousarray(t.slot_of, dtype=np.int32)
    _c().tangram_oracle_attend_range(
        _p(qb), _p(pb), _p(ip), _p(pg), _p(co), _p(so),
        ctypes.c_int32(t.R), ctypes.c_int32(t.H), ctypes.c_int32(Hq), ctypes.c_int32(t.C),
        ctypes.c_int32(t.Hp), ctypes.c_int32(t.P), ctypes.c_int32(d), ctypes.c_int32(r),
        ctypes.c_int32(j), ctypes.c_int32(t0), ctypes.c_int32(t1),
        ctypes.c_double(0.0 if sm_scale is None else float(sm_scale)), _p(out), ctypes.byref(lse))
    return out, float(lse.value)
