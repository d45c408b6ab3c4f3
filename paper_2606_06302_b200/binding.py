"""Thin ctypes binding over libtangram.so (C ABI declared in include/tangram.h).

Argument marshalling only: every step of the path (Budget Reservation, Ragged Paging tables, the
AoT planner, the decode and merge kernels) runs inside the library.  Names mirror the C entry
points.  There is no CPU fallback: if the library is missing this module raises on import, and the
device calls raise TangramError on any CUDA problem.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# TANGRAM_LIB selects another build of the same library (the debug build with bounded spin loops,
# paper_2606_06302_b200/build.py --spin-limit); there is still no fallback: the named file must exist.
LIB_PATH = os.environ.get("TANGRAM_LIB") or os.path.join(_HERE, "libtangram.so")

OK, ERR_INVALID_ARG, ERR_OUT_OF_PAGES, ERR_BUFFER_TOO_SMALL, ERR_CUDA = 0, -1, -2, -3, -4
FILL_GROUP = 1
MODE_BALANCED, MODE_SPLITMAP, MODE_STATIC_EVEN = 0, 1, 2
# the finest dynamic tail tangram_default_dynamic_tail picks (large batches; tuned on B200)
DEFAULT_DYN_PERMILLE, DEFAULT_DYN_ROUNDS = 500, 6
GROUP_CLUSTERED, GROUP_ADJACENT = 0, 1
MODE_NAMES = {MODE_BALANCED: "balanced", MODE_SPLITMAP: "splitmap", MODE_STATIC_EVEN: "static_even"}

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_06302_b200.build` "
                      "(there is no fallback path)")
_lib = C.CDLL(LIB_PATH)


class TangramError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"tangram error {code}: {msg}")
        self.code = code


class _Tables(C.Structure):
    _fields_ = [("R", C.c_int32), ("H", C.c_int32), ("C", C.c_int32), ("Hp", C.c_int32), ("P", C.c_int32),
                ("perm", C.c_void_p), ("cluster_of", C.c_void_p), ("slot_of", C.c_void_p),
                ("tbl_indptr", C.c_void_p), ("tbl_pages", C.c_void_p), ("tbl_pages_cap", C.c_int64),
                ("n_pages_used", C.c_int64), ("headroom_pages", C.c_int32), ("reserved_", C.c_int32),
                ("row_pages", C.c_void_p), ("n_slots", C.c_int64)]


class _Plan(C.Structure):
    _fields_ = [("W", C.c_int32), ("n_static", C.c_int32), ("mode", C.c_int32), ("reserved_", C.c_int32),
                ("n_items", C.c_int64), ("n_part_slots", C.c_int64),
                ("split_map", C.c_void_p), ("items", C.c_void_p), ("items_cap", C.c_int64),
                ("worker_indptr", C.c_void_p), ("part_indptr", C.c_void_p)]


class _DevicePlan(C.Structure):
    _fields_ = [("R", C.c_int32), ("H", C.c_int32), ("C", C.c_int32), ("Hp", C.c_int32), ("P", C.c_int32),
                ("W", C.c_int32), ("mode", C.c_int32), ("n_static", C.c_int32), ("n_items", C.c_int64),
                ("n_part_slots", C.c_int64), ("n_merge_seqs", C.c_int64), ("n_empty_seqs", C.c_int64), ("n_big_merge_seqs", C.c_int64),
                ("merge_seqs", C.c_void_p),
                ("items", C.c_void_p), ("worker_indptr", C.c_void_p), ("list_heads", C.c_void_p),
                ("seq_info", C.c_void_p), ("part_indptr", C.c_void_p), ("tbl_pages", C.c_void_p), ("sched", C.c_void_p),
                ("max_merge_parts", C.c_int64), ("min_pool_pages", C.c_int64), ("n_slots", C.c_int64),
                ("row_ptr", C.c_void_p), ("row_pages", C.c_void_p), ("perm", C.c_void_p), ("seq_cap", C.c_void_p),
                ("plan_cover", C.c_void_p), ("grow_state", C.c_void_p), ("q_flags", C.c_void_p),
                ("seq_done", C.c_void_p)]


_lib.tangram_last_error.restype = C.c_char_p
_lib.tangram_blob_bytes.restype = C.c_size_t
_lib.tangram_workspace_bytes.restype = C.c_size_t
_lib.tangram_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32]
_lib.tangram_compact_workspace_bytes.restype = C.c_size_t
_lib.tangram_compact_workspace_bytes.argtypes = [C.c_int32, C.c_int32]
for _name in ("tangram_reserve_budgets", "tangram_build_ragged_tables", "tangram_plan_partitions",
              "tangram_query_max_ctas", "tangram_upload", "tangram_decode_attention", "tangram_decode_partials",
              "tangram_merge_partials", "tangram_append_kv", "tangram_compact_topk",
              "tangram_account_pages", "tangram_calibrate_budgets", "tangram_implicit_ratios",
              "tangram_compact_topk_chunk", "tangram_stage_from_host", "tangram_default_dynamic_tail",
              "tangram_extend_tables", "tangram_extend_tables_device", "tangram_sync_tables", "tangram_download_tables",
              "tangram_decode_step", "tangram_reset_plan", "tangram_read_stream", "tangram_overlap_state",
              "tangram_decode_attention_host", "tangram_decode_attention_static"):
    getattr(_lib, _name).restype = C.c_int

EXPORTS = ("tangram_last_error", "tangram_reserve_budgets", "tangram_build_ragged_tables",
           "tangram_plan_partitions", "tangram_query_max_ctas", "tangram_blob_bytes", "tangram_upload",
           "tangram_workspace_bytes", "tangram_decode_attention", "tangram_decode_partials", "tangram_merge_partials", "tangram_append_kv",
           "tangram_compact_workspace_bytes", "tangram_compact_topk", "tangram_account_pages",
           "tangram_calibrate_budgets", "tangram_implicit_ratios", "tangram_compact_topk_chunk",
           "tangram_stage_from_host", "tangram_default_dynamic_tail", "tangram_extend_tables",
           "tangram_extend_tables_device", "tangram_sync_tables", "tangram_download_tables", "tangram_decode_step",
           "tangram_reset_plan", "tangram_read_stream", "tangram_overlap_state", "tangram_decode_attention_host",
           "tangram_decode_attention_static")
STEP_OVERLAP = 1
STATIC_WORKSPACE_BYTES = 8 << 20     # TANGRAM_STATIC_WORKSPACE_BYTES of include/tangram.h


def _check(rc: int):
    if rc != OK:
        raise TangramError(rc, _lib.tangram_last_error().decode())


def _stream_ptr(stream):
    import torch
    return C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)


def _np(a, dtype) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=dtype))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# ------------------------------------------------------------------------------------------ a1
def tangram_reserve_budgets(mu, sigma, alpha: float, ctx_len, demand=None):
    """-> (B [H] f64, reserved [R,H] i32, kv_len [R,H] i32).  Eq. 5 / Eq. 4 / overflow rule."""
    mu, sigma, ctx = _np(mu, np.float64), _np(sigma, np.float64), _np(ctx_len, np.int32)
    H, R = mu.shape[0], ctx.shape[0]
    dem = None if demand is None else _np(demand, np.int32).reshape(R, H)
    B = np.zeros(H, np.float64)
    reserved = np.zeros((R, H), np.int32)
    kv_len = np.zeros((R, H), np.int32)
    _check(_lib.tangram_reserve_budgets(_ptr(mu), _ptr(sigma), C.c_double(alpha), C.c_int32(H), _ptr(ctx),
                                        C.c_int32(R), _ptr(dem), _ptr(B), _ptr(reserved), _ptr(kv_len)))
    return B, reserved, kv_len


# ------------------------------------------------------------------------------------------ a2
@dataclasses.dataclass
class Tables:
    R: int
    H: int
    C: int
    Hp: int
    P: int
    perm: np.ndarray
    cluster_of: np.ndarray
    slot_of: np.ndarray
    tbl_indptr: np.ndarray     # [R*C+1] i64: row r*C+c owns the page slots [indptr[row], indptr[row+1])
    tbl_pages: np.ndarray      # [n_slots] i32 page id per slot, -1 = no page yet (growth headroom)
    n_pages_used: int          # pages taken from the free list so far
    headroom_pages: int = 0
    row_pages: Optional[np.ndarray] = None   # [R*C] i32 pages each row holds (None: tight tables, every slot)

    def _c(self) -> _Tables:
        return _Tables(self.R, self.H, self.C, self.Hp, self.P, _ptr(self.perm), _ptr(self.cluster_of),
                       _ptr(self.slot_of), _ptr(self.tbl_indptr), _ptr(self.tbl_pages), len(self.tbl_pages),
                       self.n_pages_used, self.headroom_pages, 0, _ptr(self.row_pages), len(self.tbl_pages))


def tangram_pages_needed(B, reserved, n_clusters: int, page_size: int) -> int:
    """Query form of tangram_build_ragged_tables: pages the batch needs (no free list consumed)."""
    B, reserved = _np(B, np.float64), _np(reserved, np.int32)
    R, H = reserved.shape
    t = _Tables()
    rc = _lib.tangram_build_ragged_tables(_ptr(B), _ptr(reserved), C.c_int32(R), C.c_int32(H), C.c_int32(n_clusters),
                                          C.c_int32(page_size), None, C.c_int64(0), C.c_uint32(0), None, C.byref(t))
    if rc not in (OK, ERR_OUT_OF_PAGES):
        _check(rc)
    return int(t.n_pages_used)


def tangram_build_ragged_tables(B, reserved, n_clusters: int, page_size: int, free_pages, flags: int = 0,
                                kv_len=None, headroom_pages: int = 0):
    """-> (Tables, kv_len').  kv_len' is a copy of kv_len (raised to the cluster capacity with FILL_GROUP).
    headroom_pages > 0: growable tables (every row followed by that many empty page slots, row_pages filled)."""
    B, reserved = _np(B, np.float64), _np(reserved, np.int32)
    free = _np(free_pages, np.int32)
    R, H = reserved.shape
    kv = None if kv_len is None else _np(kv_len, np.int32).reshape(R, H).copy()
    need = tangram_pages_needed(B, reserved, n_clusters, page_size)
    n_rows = R * max(1, n_clusters)
    n_slots = need + n_rows * max(0, headroom_pages)
    t = Tables(R, H, n_clusters, H // max(1, n_clusters), page_size, np.zeros(H, np.int32), np.zeros(H, np.int32),
               np.zeros(H, np.int32), np.zeros(R * n_clusters + 1, np.int64), np.zeros(max(n_slots, 1), np.int32), 0,
               headroom_pages, np.zeros(n_rows, np.int32) if headroom_pages > 0 else None)
    ct = t._c()
    _check(_lib.tangram_build_ragged_tables(_ptr(B), _ptr(reserved), C.c_int32(R), C.c_int32(H),
                                            C.c_int32(n_clusters), C.c_int32(page_size), _ptr(free),
                                            C.c_int64(free.shape[0]), C.c_uint32(flags), _ptr(kv), C.byref(ct)))
    t.n_pages_used = int(ct.n_pages_used)
    t.tbl_pages = t.tbl_pages[:int(ct.n_slots)]
    t.Hp, t.C = int(ct.Hp), int(ct.C)
    return t, kv


def tangram_extend_tables(t: Tables, kv_len, free_pages, n_threads: int = 0):
    """NEXT-4 (host): one Vectorized Block Table update of `t` in place -> (rows extended, rows starved)."""
    kv, free = _np(kv_len, np.int32), _np(free_pages, np.int32)
    assert kv.shape == (t.R, t.H) and t.row_pages is not None
    ct = t._c()
    ext, starved = C.c_int64(0), C.c_int64(0)
    _check(_lib.tangram_extend_tables(C.byref(ct), _ptr(kv), _ptr(free), C.c_int64(free.shape[0]), C.c_int32(n_threads),
                                      C.byref(ext), C.byref(starved)))
    t.n_pages_used = int(ct.n_pages_used)
    return int(ext.value), int(starved.value)


# ------------------------------------------------------------------------------------------ a3
@dataclasses.dataclass
class Plan:
    W: int                     # work lists in total
    n_static: int              # launch grid: lists 0..n_static-1 are the CTAs' own
    mode: int
    split_map: np.ndarray      # [C]
    items: np.ndarray          # [n_items, 8] i32: req, kv_head, cluster, slot, tok_begin, tok_end, part_slot, n_parts
    worker_indptr: np.ndarray  # [W+1] i64
    part_indptr: np.ndarray    # [R*H+1] i64
    n_items: int
    n_part_slots: int

    def _c(self) -> _Plan:
        return _Plan(self.W, self.n_static, self.mode, 0, self.n_items, self.n_part_slots, _ptr(self.split_map),
                     _ptr(self.items),
                     self.items.shape[0], _ptr(self.worker_indptr), _ptr(self.part_indptr))


def tangram_plan_partitions(t: Tables, B, kv_len, n_workers: int, granule_tokens: int, overhead_granules: int,
                            mode: int, static_splits: int = 0, dyn_permille: int = 0, dyn_rounds: int = 0) -> Plan:
    B, kv = _np(B, np.float64), _np(kv_len, np.int32)
    ct = t._c()
    split_map = np.zeros(t.C, np.int32)
    q = _Plan(0, 0, 0, 0, 0, 0, _ptr(split_map), None, 0, None, None)
    args = (C.byref(ct), _ptr(B), _ptr(kv), C.c_int32(n_workers), C.c_int32(granule_tokens),
            C.c_int32(overhead_granules), C.c_int32(mode), C.c_int32(static_splits), C.c_int32(dyn_permille),
            C.c_int32(dyn_rounds))
    _check(_lib.tangram_plan_partitions(*args, C.byref(q)))
    pl = Plan(int(q.W), int(q.n_static), mode, split_map, np.zeros((max(int(q.n_items), 1), 8), np.int32),
              np.zeros(int(q.W) + 1, np.int64), np.zeros(t.R * t.H + 1, np.int64), int(q.n_items),
              int(q.n_part_slots))
    cp = pl._c()
    _check(_lib.tangram_plan_partitions(*args, C.byref(cp)))
    pl.items = pl.items[:pl.n_items]
    return pl


# ------------------------------------------------------------------------------------------ device side
def tangram_query_max_ctas(device: int, head_dim: int, gqa: int) -> int:
    n = C.c_int32(0)
    _check(_lib.tangram_query_max_ctas(C.c_int(device), C.c_int32(head_dim), C.c_int32(gqa), C.byref(n)))
    return int(n.value)


def tangram_blob_bytes(t: Tables, p: Plan) -> int:
    ct, cp = t._c(), p._c()
    return int(_lib.tangram_blob_bytes(C.byref(ct), C.byref(cp)))


def tangram_workspace_bytes(n_part_slots: int, gqa: int, head_dim: int) -> int:
    return int(_lib.tangram_workspace_bytes(n_part_slots, gqa, head_dim))


class DevicePlan:
    """Uploaded tables + plan.  Keeps the device blob (a torch uint8 tensor) alive."""

    def __init__(self, t: Tables, p: Plan, device="cuda", stream=None):
        import torch
        self.tables, self.plan = t, p
        nbytes = tangram_blob_bytes(t, p)
        self.blob = torch.empty(nbytes, dtype=torch.uint8, device=device)
        self.c = _DevicePlan()
        ct, cp = t._c(), p._c()
        sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
        _check(_lib.tangram_upload(C.byref(ct), C.byref(cp), C.c_void_p(self.blob.data_ptr()), C.c_size_t(nbytes), sp,
                                   C.byref(self.c)))


def tangram_upload(t: Tables, p: Plan, device="cuda", stream=None) -> DevicePlan:
    return DevicePlan(t, p, device, stream)


def tangram_decode_attention(dp: DevicePlan, q, kv_pool, out=None, lse=None, workspace=None, sm_scale: float = 0.0,
                             worker_ns=None, stream=None, kv_len=None, _entry="tangram_decode_attention"):
    """q [R,Hq,d] bf16 cuda, kv_pool [n_pages,Hp,2,P,d] bf16 cuda -> (out [R,Hq,d] bf16, lse [R,Hq] f32).
    Asynchronous on the current (or given) torch stream."""
    import torch
    # out / lse may also be PINNED host tensors: page-locked memory is mapped into the device's address space
    # (unified addressing) and the kernels write them in place over the bus; q must be on the device (host-resident
    # queries: tangram_decode_attention_host)
    assert q.is_cuda and kv_pool.is_cuda and q.dtype == torch.bfloat16 and kv_pool.dtype == torch.bfloat16
    assert q.is_contiguous() and kv_pool.is_contiguous()
    R, Hq, d = q.shape
    n_pages = kv_pool.shape[0]
    assert tuple(kv_pool.shape[1:]) == (dp.c.Hp, 2, dp.c.P, d) and R == dp.c.R
    G = Hq // dp.c.H
    if out is None:
        out = torch.empty(R, Hq, d, dtype=torch.bfloat16, device=kv_pool.device)
    if lse is None:
        lse = torch.empty(R, Hq, dtype=torch.float32, device=kv_pool.device)
    assert (out.is_cuda or out.is_pinned()) and (lse.is_cuda or lse.is_pinned())
    need = tangram_workspace_bytes(int(dp.c.n_part_slots), G, d)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=kv_pool.device)
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    wn = C.c_void_p(worker_ns.data_ptr()) if worker_ns is not None else None
    if kv_len is not None:
        assert kv_len.is_cuda and kv_len.dtype == torch.int32 and kv_len.is_contiguous() and kv_len.numel() == R * dp.c.H
    kvl = C.c_void_p(kv_len.data_ptr()) if kv_len is not None else None
    _check(getattr(_lib, _entry)(C.byref(dp.c), C.c_void_p(q.data_ptr()), C.c_void_p(kv_pool.data_ptr()),
                                         C.c_int64(n_pages), kvl, C.c_int32(Hq), C.c_int32(d), C.c_float(sm_scale),
                                         C.c_void_p(out.data_ptr()), C.c_void_p(lse.data_ptr()),
                                         C.c_void_p(workspace.data_ptr()), C.c_size_t(workspace.numel()), wn, sp))
    return out, lse


def tangram_decode_attention_host(dp: DevicePlan, q_host, q_stage, kv_pool, out, lse, workspace, sm_scale: float = 0.0,
                                  stream=None, kv_len=None):
    """End to end with host buffers: q_host (pinned) -> q_stage (cuda) by the staging kernel, decode kernel overlapped
    behind it; out / lse may be pinned host tensors."""
    import torch
    assert q_host.is_pinned() and q_stage.is_cuda and kv_pool.is_cuda and q_host.dtype == torch.bfloat16
    assert q_host.is_contiguous() and q_stage.is_contiguous() and q_stage.shape == q_host.shape and q_stage.dtype == q_host.dtype
    R, Hq, d = q_host.shape
    assert tuple(kv_pool.shape[1:]) == (dp.c.Hp, 2, dp.c.P, d) and R == dp.c.R
    assert (out.is_cuda or out.is_pinned()) and (lse.is_cuda or lse.is_pinned())
    kvl = C.c_void_p(kv_len.data_ptr()) if kv_len is not None else None
    _check(_lib.tangram_decode_attention_host(C.byref(dp.c), C.c_void_p(q_host.data_ptr()), C.c_void_p(q_stage.data_ptr()),
                                              C.c_void_p(kv_pool.data_ptr()), C.c_int64(kv_pool.shape[0]), kvl, C.c_int32(Hq),
                                              C.c_int32(d), C.c_float(sm_scale), C.c_void_p(out.data_ptr()),
                                              C.c_void_p(lse.data_ptr()), C.c_void_p(workspace.data_ptr()),
                                              C.c_size_t(workspace.numel()), None, _stream_ptr(stream)))
    return out, lse


def tangram_decode_attention_static(dp: DevicePlan, q, kv_pool, out=None, lse=None, sm_scale: float = 0.0, worker_ns=None,
                                    stream=None, kv_len=None):
    """tangram_decode_attention for a caller that cannot allocate the split-KV workspace (a serving engine whose HBM
    all went to the page pool, code running under somebody else's allocator): the library's fixed 8 MiB array is the
    workspace and the C call allocates nothing.  Pass `out` and `lse` if this wrapper must not allocate either (when
    they are None it makes them with torch.empty, like the other wrappers).  Raises TangramError (BUFFER_TOO_SMALL)
    for a plan whose partials exceed STATIC_WORKSPACE_BYTES.  Every call on a GPU shares the one array: calls that
    overlap on the GPU race (include/tangram.h)."""
    import torch
    assert q.is_cuda and kv_pool.is_cuda and q.dtype == torch.bfloat16 and kv_pool.dtype == torch.bfloat16
    assert q.is_contiguous() and kv_pool.is_contiguous()
    R, Hq, d = q.shape
    assert tuple(kv_pool.shape[1:]) == (dp.c.Hp, 2, dp.c.P, d) and R == dp.c.R
    if out is None:
        out = torch.empty(R, Hq, d, dtype=torch.bfloat16, device=kv_pool.device)
    if lse is None:
        lse = torch.empty(R, Hq, dtype=torch.float32, device=kv_pool.device)
    wn = C.c_void_p(worker_ns.data_ptr()) if worker_ns is not None else None
    if kv_len is not None:
        assert kv_len.is_cuda and kv_len.dtype == torch.int32 and kv_len.is_contiguous() and kv_len.numel() == R * dp.c.H
    kvl = C.c_void_p(kv_len.data_ptr()) if kv_len is not None else None
    _check(_lib.tangram_decode_attention_static(C.byref(dp.c), C.c_void_p(q.data_ptr()), C.c_void_p(kv_pool.data_ptr()),
                                                C.c_int64(kv_pool.shape[0]), kvl, C.c_int32(Hq), C.c_int32(d),
                                                C.c_float(sm_scale), C.c_void_p(out.data_ptr()), C.c_void_p(lse.data_ptr()),
                                                wn, _stream_ptr(stream)))
    return out, lse


def tangram_decode_partials(dp: DevicePlan, q, kv_pool, out=None, lse=None, workspace=None, sm_scale: float = 0.0,
                            worker_ns=None, stream=None, kv_len=None):
    """a4 alone: the split-KV decode kernel (see include/tangram.h)."""
    return tangram_decode_attention(dp, q, kv_pool, out, lse, workspace, sm_scale, worker_ns, stream, kv_len,
                                    _entry="tangram_decode_partials")


def tangram_merge_partials(dp: DevicePlan, out, lse, workspace, stream=None):
    """a5 alone: the LSE merge kernel over the partials in `workspace`."""
    import torch
    R, Hq, d = out.shape
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    _check(_lib.tangram_merge_partials(C.byref(dp.c), C.c_int32(Hq), C.c_int32(d), C.c_void_p(out.data_ptr()),
                                       C.c_void_p(lse.data_ptr()), C.c_void_p(workspace.data_ptr()),
                                       C.c_size_t(workspace.numel()), sp))
    return out, lse


def tangram_extend_tables_device(dp: DevicePlan, kv_len, free_pages, stream=None):
    """NEXT-4 (device): the same update on the uploaded tables; kv_len [R,H] / free_pages [n_free] int32 cuda."""
    import torch
    assert kv_len.is_cuda and kv_len.dtype == torch.int32 and kv_len.is_contiguous() and kv_len.numel() == dp.c.R * dp.c.H
    assert free_pages.is_cuda and free_pages.dtype == torch.int32 and free_pages.is_contiguous()
    _check(_lib.tangram_extend_tables_device(C.byref(dp.c), C.c_void_p(kv_len.data_ptr()), C.c_void_p(free_pages.data_ptr()),
                                             C.c_int64(free_pages.numel()), _stream_ptr(stream)))


def tangram_sync_tables(t: Tables, dp: DevicePlan, stream=None):
    """Host tables -> device copy of an uploaded plan (after tangram_extend_tables on the host)."""
    ct = t._c()
    _check(_lib.tangram_sync_tables(C.byref(ct), C.byref(dp.c), _stream_ptr(stream)))


def tangram_download_tables(dp: DevicePlan, t: Tables, stream=None) -> int:
    """Device state (tbl_pages, row_pages, free-list cursor) -> `t` in place; returns the rows starved so far."""
    assert t.row_pages is not None
    ct = t._c()
    starved = C.c_int64(0)
    _check(_lib.tangram_download_tables(C.byref(dp.c), C.byref(ct), C.byref(starved), _stream_ptr(stream)))
    t.n_pages_used = int(ct.n_pages_used)
    return int(starved.value)


def tangram_read_stream(src, sink, nbytes=None, stream=None):
    """Measurement aid: one read-only pass over `src` (cuda tensor) with 16-byte loads; sink = uint32/int32[1] cuda."""
    n = src.numel() * src.element_size() if nbytes is None else nbytes
    _check(_lib.tangram_read_stream(C.c_void_p(src.data_ptr()), C.c_size_t(n), C.c_void_p(sink.data_ptr()), _stream_ptr(stream)))


def tangram_overlap_state() -> int:
    return int(_lib.tangram_overlap_state())


def tangram_reset_plan(dp: DevicePlan, stream=None):
    _check(_lib.tangram_reset_plan(C.byref(dp.c), _stream_ptr(stream)))


def tangram_decode_step(dp: DevicePlan, q, k_new, v_new, kv_pool, kv_len, free_pages=None, out=None, lse=None,
                        workspace=None, sm_scale: float = 0.0, overflow=None, flags: int = 0, worker_ns=None, stream=None):
    """One decode step of one layer in one launch: KV append + attention + merge + length update + table growth
    for the next step (include/tangram.h).  kv_len [R,H] int32 cuda is incremented in place."""
    import torch
    assert q.is_cuda and kv_pool.is_cuda and q.dtype == torch.bfloat16 and kv_pool.dtype == torch.bfloat16
    assert q.is_contiguous() and kv_pool.is_contiguous()
    R, Hq, d = q.shape
    H = dp.c.H
    assert tuple(kv_pool.shape[1:]) == (dp.c.Hp, 2, dp.c.P, d) and R == dp.c.R
    for x in (k_new, v_new):
        assert x.is_cuda and x.dtype == torch.bfloat16 and x.is_contiguous() and tuple(x.shape) == (R, H, d)
    assert kv_len.is_cuda and kv_len.dtype == torch.int32 and kv_len.is_contiguous() and kv_len.numel() == R * H
    G = Hq // H
    if out is None:
        out = torch.empty(R, Hq, d, dtype=torch.bfloat16, device=kv_pool.device)
    if lse is None:
        lse = torch.empty(R, Hq, dtype=torch.float32, device=kv_pool.device)
    if workspace is None:
        workspace = torch.empty(tangram_workspace_bytes(int(dp.c.n_part_slots), G, d), dtype=torch.uint8, device=kv_pool.device)
    fp, nf = None, 0
    if free_pages is not None:
        assert free_pages.is_cuda and free_pages.dtype == torch.int32 and free_pages.is_contiguous()
        fp, nf = C.c_void_p(free_pages.data_ptr()), free_pages.numel()
    ov = C.c_void_p(overflow.data_ptr()) if overflow is not None else None
    wn = C.c_void_p(worker_ns.data_ptr()) if worker_ns is not None else None
    _check(_lib.tangram_decode_step(C.byref(dp.c), C.c_void_p(q.data_ptr()), C.c_void_p(k_new.data_ptr()),
                                    C.c_void_p(v_new.data_ptr()), C.c_void_p(kv_pool.data_ptr()), C.c_int64(kv_pool.shape[0]),
                                    C.c_void_p(kv_len.data_ptr()), fp, C.c_int64(nf), C.c_int32(Hq), C.c_int32(d),
                                    C.c_float(sm_scale), C.c_void_p(out.data_ptr()), C.c_void_p(lse.data_ptr()),
                                    C.c_void_p(workspace.data_ptr()), C.c_size_t(workspace.numel()), ov, C.c_uint32(flags),
                                    wn, _stream_ptr(stream)))
    return out, lse


def tangram_append_kv(dp: DevicePlan, k_new, v_new, kv_pool, kv_len, overflow=None, stream=None):
    """NEXT-1: append one decode step's K/V rows ([R,H,d] bf16 each) into the ragged pages; kv_len
    ([R,H] int32, cuda) is incremented in place; `overflow` (int32[1], cuda) counts dropped rows."""
    import torch
    R, H, d = k_new.shape
    assert k_new.is_cuda and v_new.is_cuda and kv_pool.is_cuda and kv_len.is_cuda
    assert k_new.dtype == torch.bfloat16 and v_new.dtype == torch.bfloat16 and kv_len.dtype == torch.int32
    assert k_new.is_contiguous() and v_new.is_contiguous() and kv_len.is_contiguous()
    assert (R, H) == (dp.c.R, dp.c.H) and tuple(kv_pool.shape[1:]) == (dp.c.Hp, 2, dp.c.P, d)
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    ov = C.c_void_p(overflow.data_ptr()) if overflow is not None else None
    _check(_lib.tangram_append_kv(C.byref(dp.c), C.c_void_p(k_new.data_ptr()), C.c_void_p(v_new.data_ptr()),
                                  C.c_void_p(kv_pool.data_ptr()), C.c_int64(kv_pool.shape[0]), C.c_int32(d),
                                  C.c_void_p(kv_len.data_ptr()), ov, sp))
    return kv_len


def tangram_compact_workspace_bytes(R: int, H: int) -> int:
    return int(_lib.tangram_compact_workspace_bytes(R, H))


def tangram_compact_topk(dp: DevicePlan, scores, k_dense, v_dense, ctx_len, keep, kv_pool, idx_out=None,
                         clamped=None, workspace=None, stream=None, kv_len=None):
    """NEXT-2: per-head Top-keep[r][h] selection on `scores` ([R,H,n_max] f32) and compaction of the selected
    K/V rows ([R,H,n_max,d] bf16 each) into the ragged pages.  ctx_len [R] / keep [R,H] int32 cuda.
    -> idx_out [R,H,n_max] int32 (first keep[r][h] entries of each row = retained token indices, ascending).
    With kv_len ([R,H] int32 cuda, updated in place) the call is tangram_compact_topk_chunk: the tensors hold one
    prefill chunk (ctx_len = chunk lengths) and the rows are appended behind the kv_len tokens already held."""
    import torch
    R, H, n_max, d = k_dense.shape
    assert scores.is_cuda and k_dense.is_cuda and v_dense.is_cuda and kv_pool.is_cuda and ctx_len.is_cuda and keep.is_cuda
    assert scores.dtype == torch.float32 and tuple(scores.shape) == (R, H, n_max) and scores.is_contiguous()
    assert k_dense.dtype == torch.bfloat16 and v_dense.dtype == torch.bfloat16 and v_dense.shape == k_dense.shape
    assert k_dense.is_contiguous() and v_dense.is_contiguous() and kv_pool.is_contiguous()
    assert ctx_len.dtype == torch.int32 and keep.dtype == torch.int32 and ctx_len.numel() == R and keep.numel() == R * H
    assert ctx_len.is_contiguous() and keep.is_contiguous()
    assert (R, H) == (dp.c.R, dp.c.H) and tuple(kv_pool.shape[1:]) == (dp.c.Hp, 2, dp.c.P, d)
    if idx_out is None:
        idx_out = torch.empty(R, H, n_max, dtype=torch.int32, device=scores.device)
    need = tangram_compact_workspace_bytes(R, H)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=scores.device)
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    cl = C.c_void_p(clamped.data_ptr()) if clamped is not None else None
    tail = (C.c_void_p(kv_pool.data_ptr()), C.c_int64(kv_pool.shape[0]), C.c_int32(d), C.c_void_p(idx_out.data_ptr()), cl,
            C.c_void_p(workspace.data_ptr()), C.c_size_t(workspace.numel()), sp)
    head = (C.byref(dp.c), C.c_void_p(scores.data_ptr()), C.c_void_p(k_dense.data_ptr()), C.c_void_p(v_dense.data_ptr()),
            C.c_int64(n_max), C.c_void_p(ctx_len.data_ptr()), C.c_void_p(keep.data_ptr()))
    if kv_len is None:
        _check(_lib.tangram_compact_topk(*head, *tail))
    else:
        assert kv_len.is_cuda and kv_len.dtype == torch.int32 and kv_len.is_contiguous() and kv_len.numel() == R * H
        _check(_lib.tangram_compact_topk_chunk(*head, C.c_void_p(kv_len.data_ptr()), *tail))
    return idx_out


def tangram_compact_topk_chunk(dp: DevicePlan, scores, k_dense, v_dense, chunk_len, keep, kv_len, kv_pool, **kw):
    """One prefill chunk compressed and appended behind the kv_len tokens every head already holds."""
    return tangram_compact_topk(dp, scores, k_dense, v_dense, chunk_len, keep, kv_pool, kv_len=kv_len, **kw)


class _PageAccount(C.Structure):
    _fields_ = [("pages_alloc", C.c_int64), ("slots_alloc", C.c_int64), ("slots_exact", C.c_int64),
                ("slots_full", C.c_int64), ("slots_used", C.c_int64), ("tables", C.c_int64),
                ("reclaimed_frac", C.c_double), ("fragmentation", C.c_double)]


def tangram_account_pages(B, reserved, ctx_len, heads_per_page: int, page_size: int, policy: int) -> dict:
    """NEXT-3: pages / token-head slots the batch occupies when heads_per_page heads share a page table."""
    B, reserved, ctx = _np(B, np.float64), _np(reserved, np.int32), _np(ctx_len, np.int32)
    R, H = reserved.shape
    acc = _PageAccount()
    _check(_lib.tangram_account_pages(_ptr(B), _ptr(reserved), _ptr(ctx), C.c_int32(R), C.c_int32(H),
                                      C.c_int32(heads_per_page), C.c_int32(page_size), C.c_int32(policy), C.byref(acc)))
    return {k: getattr(acc, k) for k, _ in _PageAccount._fields_}


def tangram_calibrate_budgets(ratios, alpha: float):
    """NEXT-4: (mu, sigma, B) from the recorded per-head implicit retention ratios [n_samples, H] (Eq. 5)."""
    x = _np(ratios, np.float64)
    n, H = x.shape
    mu, sigma, B = np.zeros(H), np.zeros(H), np.zeros(H)
    _check(_lib.tangram_calibrate_budgets(_ptr(x), C.c_int32(n), C.c_int32(H), C.c_double(alpha), _ptr(mu), _ptr(sigma),
                                          _ptr(B)))
    return mu, sigma, B


def tangram_implicit_ratios(scores, ctx_len, rho: float, stream=None):
    """NEXT-4 (device): per-head (counts [R,H] int32, ratios [R,H] f64) of the global flat Top-ceil(rho H N)
    selection (Eq. 3) on scores [R,H,n_max] f32 cuda; ctx_len [R] int32 cuda."""
    import torch
    R, H, n_max = scores.shape
    assert scores.is_cuda and scores.dtype == torch.float32 and scores.is_contiguous()
    assert ctx_len.is_cuda and ctx_len.dtype == torch.int32 and ctx_len.numel() == R and ctx_len.is_contiguous()
    counts = torch.empty(R, H, dtype=torch.int32, device=scores.device)
    ratios = torch.empty(R, H, dtype=torch.float64, device=scores.device)
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    _check(_lib.tangram_implicit_ratios(C.c_void_p(scores.data_ptr()), C.c_int32(R), C.c_int32(H), C.c_int64(n_max),
                                        C.c_void_p(ctx_len.data_ptr()), C.c_double(rho), C.c_void_p(counts.data_ptr()),
                                        C.c_void_p(ratios.data_ptr()), sp))
    return counts, ratios


def tangram_stage_from_host(dst, src, stream=None):
    """dst (cuda tensor) <- src (pinned host tensor of the same size), copied by a kernel on the stream."""
    import torch
    assert dst.is_cuda and src.is_pinned() and dst.is_contiguous() and src.is_contiguous()
    nbytes = dst.numel() * dst.element_size()
    assert nbytes == src.numel() * src.element_size()
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    _check(_lib.tangram_stage_from_host(C.c_void_p(dst.data_ptr()), C.c_void_p(src.data_ptr()), C.c_size_t(nbytes), sp))
    return dst


def tangram_default_dynamic_tail(kv_len, n_workers: int, granule_tokens: int, overhead_granules: int = 1):
    """-> (dyn_permille, dyn_rounds): the library's default dynamic tail for this batch (static plan for small ones)."""
    kv = _np(kv_len, np.int32)
    R, H = kv.shape
    a, b = C.c_int32(0), C.c_int32(0)
    _check(_lib.tangram_default_dynamic_tail(_ptr(kv), C.c_int32(R), C.c_int32(H), C.c_int32(n_workers),
                                             C.c_int32(granule_tokens), C.c_int32(overhead_granules), C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)
