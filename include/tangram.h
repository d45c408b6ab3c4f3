/*
 * tangram.h -- C ABI of the B200-native Tangram hot path (arxiv/paper_2606_06302; citations are
 * lines of the paper text, PAPER.md, with the section / equation / algorithm they fall in).
 *
 * The path: decode-step attention over a KV cache that was compressed non-uniformly (every KV
 * head keeps its own token budget), stored through Ragged Paging (§4.2) and
 * executed from an Ahead-of-Time work list (§4.3), followed by a log-sum-exp
 * merge of the split-KV partials.
 *
 * Conventions
 *  - Every call returns TANGRAM_OK (0) or a negative TANGRAM_ERR_* code; a description of the last
 *    error of the calling thread is returned by tangram_last_error().  Nothing throws across the ABI.
 *  - The CALLER owns every buffer, host and device.  The library allocates no device memory.
 *  - "host" / "device" is stated per pointer.  Host calls (reserve, build tables, plan) are pure,
 *    deterministic functions of their arguments, thread-safe, and need no CUDA context.
 *  - Variable-size outputs use query-then-fill: call with the output array NULL to get the counts
 *    in the struct, allocate, call again.
 *  - fp64 expressions are evaluated exactly as written (no FMA contraction); integer results are
 *    bit-exact against the CPU oracle (oracle/tangram_oracle.py).
 */
#ifndef TANGRAM_H_
#define TANGRAM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TANGRAM_OK 0
#define TANGRAM_ERR_INVALID_ARG (-1)
#define TANGRAM_ERR_OUT_OF_PAGES (-2)
#define TANGRAM_ERR_BUFFER_TOO_SMALL (-3)
#define TANGRAM_ERR_CUDA (-4)

/* Thread-local, never NULL; valid until the next failing call on the same thread. */
const char* tangram_last_error(void);

/* ------------------------------------------------------------------------------------------------
 * a1  Budget Reservation -- PAPER.md:156-158 (Eq. 5: B = min(1, mu + alpha*sigma)), :152-154
 *     (Eq. 4: per-head top-ceil(B N)), :172-174 (Precise Page Allocation: the scheduler reserves
 *     exactly the post-compression footprint at admission), :176 (overflow: a head that demands
 *     more than its budget keeps the top entries within capacity).
 *
 *   mu, sigma    host [H] f64   calibrated mean / std of each KV head's implicit retention ratio
 *   alpha        safety-margin coefficient (the paper uses 2, :262)
 *   ctx_len      host [R] i32   pre-compression context length N_r >= 1
 *   demand       host [R][H] i32 or NULL: tokens the compressor would retain for this input (>= 0)
 *   B_out        host [H] f64   B_h = min(1.0, mu_h + alpha*sigma_h), one multiply then one add
 *   reserved_out host [R][H] i32  ceil(B_h * N_r) clamped to [1, N_r]
 *   kv_len_out   host [R][H] i32  min(demand, reserved), or reserved if demand == NULL
 * Errors: INVALID_ARG if H < 1, R < 1, ctx_len < 1, demand < 0, or mu + alpha*sigma <= 0 (B must
 * be in (0,1], :152); nothing is written then. */
int tangram_reserve_budgets(const double* mu, const double* sigma, double alpha, int32_t H,
                            const int32_t* ctx_len, int32_t R, const int32_t* demand,
                            double* B_out, int32_t* reserved_out, int32_t* kv_len_out);

/* ------------------------------------------------------------------------------------------------
 * a2  Ragged Paging -- PAPER.md:190 (a page holds H_p x 2 x P x d elements of one head group in
 *     one layer; each group owns a page table sized by its max budget), :192-194 and :227-233
 *     (Budget-Aware Clustering: sort heads by budget ascending, H_p consecutive heads = group),
 *     :235 (slack: smaller-budget heads may keep extra KV up to the group's budget).
 *
 * Heads are stably sorted by B (ties keep head order); cluster c = sorted positions
 * [c*H_p, (c+1)*H_p); row (r, c) of the tables has ceil(max_{h in c} reserved[r][h] / P) pages and
 * takes the next entries of free_pages in order, rows visited r-major then c.  Page layout in the
 * pool (bf16): pool[page][slot][kv][token][d], kv 0 = K, 1 = V, slot = slot_of[head].
 *
 * Growth during decode (NEXT-4, "a scheduling step requests the pages required for the
 * next pass", :244 Vectorized Block Table): with out->headroom_pages = h > 0 every row is followed by
 * h page SLOTS that hold no page yet (tbl_pages = -1), so that tangram_extend_tables /
 * tangram_extend_tables_device can hand a row its next page without moving any row; out->row_pages
 * (required then) receives the pages each row holds.  With headroom_pages = 0 and row_pages = NULL
 * the tables are tight (every slot holds a page), as :172 reserves them at admission.
 *
 *   B            host [H] f64 (from a1)            reserved  host [R][H] i32 (from a1)
 *   free_pages   host [n_free] i32 page ids the caller's allocator hands out (not modified)
 *   flags        TANGRAM_FILL_GROUP: kv_len_inout[r][h] := max reserved of h's cluster (:235)
 *   kv_len_inout host [R][H] i32 or NULL (only touched with TANGRAM_FILL_GROUP)
 *   out          ZERO-INITIALISE the struct first (memset / = {0}): it carries inputs (headroom_pages, row_pages,
 *                tbl_pages_cap) next to outputs and has no version field, so a field a caller does not know about
 *                must read as 0.  Then caller-filled: perm/cluster_of/slot_of [H], tbl_indptr [R*C+1], tbl_pages
 *                [tbl_pages_cap] (or tbl_pages == NULL to query: only n_pages_used / n_slots are
 *                written), headroom_pages (in), row_pages [R*C] (or NULL if headroom_pages == 0).
 *                On success R,H,C,Hp,P, the arrays, n_pages_used and n_slots are written.
 * Errors: INVALID_ARG (H % n_clusters != 0, page_size <= 0, headroom_pages < 0 or > 0 without
 * row_pages, ...); OUT_OF_PAGES if the free list is too short (n_pages_used = pages needed; arrays
 * untouched); BUFFER_TOO_SMALL if tbl_pages_cap < n_slots (n_pages_used / n_slots = needed). */
#define TANGRAM_FILL_GROUP 1u
typedef struct tangram_tables {
    int32_t R, H, C, Hp, P;
    int32_t* perm;        /* host [H]  sorted position -> head (pi of :229) */
    int32_t* cluster_of;  /* host [H]  head -> cluster */
    int32_t* slot_of;     /* host [H]  head -> slot inside the cluster's pages */
    int64_t* tbl_indptr;  /* host [R*C+1]  CSR row pointer, row = r*C + c: the row owns page slots
                             [tbl_indptr[row], tbl_indptr[row+1]) */
    int32_t* tbl_pages;   /* host [tbl_pages_cap]  page id of every slot, row after row; -1 = no page yet */
    int64_t tbl_pages_cap;
    int64_t n_pages_used; /* pages taken from the free list so far (the free list's cursor) */
    int32_t headroom_pages; /* in: unassigned slots kept behind every row for growth (0 = tight tables) */
    int32_t reserved_;
    int32_t* row_pages;   /* host [R*C] pages each row holds (its first row_pages slots), or NULL: all slots */
    int64_t n_slots;      /* out: tbl_indptr[R*C] = entries of tbl_pages = n_pages_used + R*C*headroom at build */
} tangram_tables;
int tangram_build_ragged_tables(const double* B, const int32_t* reserved, int32_t R, int32_t H,
                                int32_t n_clusters, int32_t page_size, const int32_t* free_pages,
                                int64_t n_free, uint32_t flags, int32_t* kv_len_inout,
                                tangram_tables* out);

/* ------------------------------------------------------------------------------------------------
 * a3  AoT Load Balancing -- PAPER.md:196-225 (Algorithm 1: S_i = max(1, round(Phi_i / tau)),
 *     tau = Omega / N_CTA), :250-256 (the split map is computed offline from budget ratios; zero
 *     runtime planning), :120 (static uniform num_splits is the straggler baseline).
 *
 * Offline, host-side, deterministic work-list builder.  Sequences (r, h) are visited r-major then
 * in perm order.  A sequence of n = kv_len[r][h] tokens has ceil(n / g) granules.
 *   TANGRAM_MODE_BALANCED   (primary; BASELINE.json north_star "chunks of near-equal KV bytes per
 *       CTA"): the sequences are laid end to end, each preceded by `overhead_granules` cost units;
 *       worker k owns positions [floor(k T / W), floor((k+1) T / W)); every maximal run of one
 *       sequence's granules inside one worker is one item.
 *   TANGRAM_MODE_SPLITMAP   (Algorithm 1, literal): every sequence of cluster c is cut into
 *       split_map[c] granule-aligned chunks; item k (global order) goes to worker k mod W.
 *   TANGRAM_MODE_STATIC_EVEN (baseline of :120): as SPLITMAP with the same split count for every
 *       head: static_splits, or if <= 0 the smallest S with R*H*S >= W.
 * Items of a worker are stored contiguously (worker_indptr), plan order kept.  part_slot numbers
 * the items of a sequence in token order from part_indptr[r*H + h]; n_parts = their count
 * (n_parts == 1: the decode kernel writes the final output directly, no merge).
 *
 *   t        tables from a2 (host)      B host [H]      kv_len host [R][H] i32 (<= cluster capacity)
 *   n_workers >= 1 (persistent CTAs = launch grid, from tangram_query_max_ctas)
 *   granule_tokens g: positive multiple of t->P;  overhead_granules c0 >= 0
 *   dyn_permille, dyn_rounds (BALANCED only; both 0 = every CTA owns exactly one list, the purely
 *       static plan): the last dyn_permille/1000 of the cost axis is not pre-assigned to a CTA but
 *       cut into dyn_rounds rounds of n_workers lists each -- round j < dyn_rounds takes 2^-j of
 *       that share, the last round the rest -- which the CTAs claim in list order when they run
 *       out of work.  Everything is still computed offline; the claim only decides WHICH CTA runs
 *       a precomputed list, which is what absorbs the stable +-15 % per-SM bandwidth differences
 *       measured on B200.  List k covers cost positions [b_k, b_{k+1}),
 *       b_k = floor(T * cumw_k / cumw_W) with the integer list weights of DESIGN.md §Planner.
 *   out      caller-filled: split_map [C], worker_indptr [W+1], part_indptr [R*H+1], items
 *            [items_cap] (or items == NULL to query: n_items / n_part_slots only).
 *            split_map always receives Algorithm 1's S (the constant S for STATIC_EVEN).
 * Errors: INVALID_ARG; BUFFER_TOO_SMALL (n_items = needed). */
#define TANGRAM_MODE_BALANCED 0
#define TANGRAM_MODE_SPLITMAP 1
#define TANGRAM_MODE_STATIC_EVEN 2
typedef struct tangram_item { /* 32 bytes */
    int32_t req, kv_head, cluster, slot, tok_begin, tok_end, part_slot, n_parts;
} tangram_item;
typedef struct tangram_plan {
    int32_t W;        /* work lists in total = n_static * (1 + dyn_rounds) */
    int32_t n_static; /* = n_workers: lists 0..n_static-1 belong to CTA 0..n_static-1 (the launch grid) */
    int32_t mode, reserved_;
    int64_t n_items, n_part_slots;
    int32_t* split_map;     /* host [C] */
    tangram_item* items;    /* host [items_cap], worker-major */
    int64_t items_cap;
    int64_t* worker_indptr; /* host [W+1] */
    int64_t* part_indptr;   /* host [R*H+1], seq = r*H + h */
} tangram_plan;
int tangram_plan_partitions(const tangram_tables* t, const double* B, const int32_t* kv_len,
                            int32_t n_workers, int32_t granule_tokens, int32_t overhead_granules,
                            int32_t mode, int32_t static_splits, int32_t dyn_permille, int32_t dyn_rounds,
                            tangram_plan* out);

/* Default dynamic tail for tangram_plan_partitions (a measured tuning rule, not from the paper), by the cost units
 * (granules of granule_tokens + overhead_granules per non-empty sequence) a worker gets: fewer than 48 -> (0, 0), the
 * purely static plan (with little work per CTA the claims and the extra parts to merge cost more than the balance
 * brings: 8b shape, 4 requests: 30.7 us static against 34.8 us with a tail); 48 .. 383 -> (500, 4); 384 and more ->
 * (500, 6) (round-2 sweep on B200, reading A32: e.g. 32b shape with 16 requests 113 us with (500, 4), 119 us
 * with (500, 6), 127 us static).
 * kv_len host [R][H] i32.  Errors: INVALID_ARG. */
int tangram_default_dynamic_tail(const int32_t* kv_len, int32_t R, int32_t H, int32_t n_workers, int32_t granule_tokens,
                                 int32_t overhead_granules, int32_t* dyn_permille_out, int32_t* dyn_rounds_out);

/* ------------------------------------------------------------------------------------------------
 * Device side.  One upload of tables + plan per (batch, layer); then one
 * tangram_decode_attention per decode step with no host planning (:254 "zero runtime planning").
 */

/* N_CTA of :252 ("CUDAMaxOccupancy API ... CTAs the GPU can execute concurrently for the attention
 * kernel") = SM count x resident CTAs per SM of the decode kernel for this head_dim / GQA group.
 * Needs a CUDA device.  head_dim in {64, 128, 256}, 1 <= gqa <= 16 (<= 8 at head_dim 256). */
int tangram_query_max_ctas(int device, int32_t head_dim, int32_t gqa, int32_t* n_cta_out);

/* Bytes of the device blob that tangram_upload fills for these tables + plan. */
size_t tangram_blob_bytes(const tangram_tables* t, const tangram_plan* p);

/* Host-side view of an uploaded plan: sizes plus DEVICE pointers into the blob.  Plain data; valid
 * as long as the blob is. */
typedef struct tangram_device_plan {
    int32_t R, H, C, Hp, P, W /* work lists on the device: the plan's, minus empty dynamic-tail lists */, mode,
        n_static /* launch grid */;
    int64_t n_items, n_part_slots;
    int64_t n_merge_seqs;       /* sequences whose part count is not 1 */
    int64_t n_empty_seqs;       /* of these, the first n_empty_seqs have no part at all (kv_len 0) */
    int64_t n_big_merge_seqs;   /* ... and the last n_big_merge_seqs have more than 16 parts */
    const int32_t* merge_seqs;  /* device [n_merge_seqs][4]: {r * H + h, first part slot, parts, 0}, empty
                                   sequences first, then by part count <= 16 / > 16 */
    const void* items;          /* device: 32-byte device items (cluster replaced by the table row offset) */
    const int64_t* worker_indptr; /* device [W+1] */
    const void* list_heads;       /* device [W] 128-byte list heads: item range, first item, its first 16 page ids */
    const int32_t* seq_info;      /* device [R*H][4]: {first slot of the head's row, slot capacity in tokens, slot in
                                     the page, row index r*C + c} */
    const int64_t* part_indptr;   /* device [R*H+1] */
    const int32_t* tbl_pages;     /* device page ids */
    int32_t* sched;               /* device [8]: list-claim / CTAs-done counters of the dynamic tail, the ticket and
                                     exit counters of the in-kernel merge (zero between launches; the kernel re-arms
                                     them itself), the launch number of the host-query staging and the number of
                                     launches that merged in-grid on this plan (the epoch of seq_done) */
    int64_t max_merge_parts;      /* most parts any sequence has (sizes the column split of the big-record merge) */
    int64_t min_pool_pages;       /* largest page id in the tables at upload + 1: the device calls return INVALID_ARG
                                     for a kv_pool with fewer pages */
    /* block-table state on the device (NEXT-4); all arrays live in the blob */
    int64_t n_slots;              /* entries of tbl_pages (assigned pages + growth slots) */
    const int32_t* row_ptr;       /* device [R*C+1]: first slot of every (request, cluster) row */
    int32_t* row_pages;           /* device [R*C]: pages each row holds */
    const int32_t* perm;          /* device [H]: sorted position -> head (cluster c = perm[c*Hp .. (c+1)*Hp)) */
    int32_t* seq_cap;             /* device [R*H]: tokens the pages of head h's row hold (row_pages x P) */
    const int32_t* plan_cover;    /* device [R*H]: largest tok_end any item of the plan has for the sequence */
    int32_t* grow_state;          /* device [4]: {free-list cursor, rows starved so far, 0, 0} */
    int32_t* q_flags;             /* device [R*H]: staging flags of tangram_decode_attention_host (launch numbers) */
    uint32_t* seq_done;           /* device [R*H]: parts of each sequence written so far, summed over the launches that
                                     merged in-grid on this plan (the in-grid merge waits for launches x parts) */
} tangram_device_plan;

/* Packs tables + plan and copies them into dev_blob (device, >= tangram_blob_bytes, 256-byte
 * aligned) with cudaMemcpyAsync on `stream` (a cudaStream_t, may be NULL); fills *dp.  The host
 * arrays may be freed when the call returns. */
int tangram_upload(const tangram_tables* t, const tangram_plan* p, void* dev_blob, size_t bytes,
                   void* stream, tangram_device_plan* dp);

/* Zeroes the launch-state counters of an uploaded plan (dp->sched, dp->q_flags, dp->seq_done) on `stream`.  The kernels re-arm the counters
 * themselves at the end of every launch that runs to completion; this call is for recovery after a launch that
 * did not (an aborted process, a fault), or after two launches on one plan were wrongly overlapped. */
int tangram_reset_plan(const tangram_device_plan* dp, void* stream);

/* Workspace for the split-KV partials: n_part_slots x G x (d + 1) fp32, rounded up. */
size_t tangram_workspace_bytes(int64_t n_part_slots, int32_t gqa, int32_t head_dim);

/* a4 + a5  One layer, whole batch: split-KV decode kernel over the work lists, then the LSE merge -- inside the
 * same persistent grid and without a grid barrier: every part of a multi-part sequence is published by a release add
 * on the sequence's counter (dp->seq_done), and a CTA that is out of work lists merges its share of the sequences,
 * each as soon as the counter shows all parts of this launch (ONE cooperative launch whenever the grid fits on the
 * device: n_static <= tangram_query_max_ctas); the stand-alone merge kernel follows as a second launch when the grid
 * is larger than that (CTAs that wait for one another must be gang-scheduled), at d = 256, or when a merge record is
 * wider than the CTA (G x d/4 > consumer threads: d = 128 with G > 8, or G > 4 on 32-token pages).
 * Asynchronous on `stream`; CUDA-graph capturable; no host work besides the launch.
 *
 *   dp        from tangram_upload (host struct holding device pointers)
 *   q         device [R][Hq][d] bf16, 16-byte aligned (host memory is refused, see "Host buffers" below)
 *   kv_pool   device [n_pool_pages][Hp][2][P][d] bf16, 128-byte aligned (Ragged page, :190)
 *   kv_len_dev device [R][H] i32 or NULL.  NULL: the items are executed exactly as planned.  Otherwise the
 *             plan is OPEN-ENDED: every item covers tokens [tok_begin, min(tok_end, kv_len_dev[r][h])), so a
 *             plan built once for lengths >= the run-time ones (e.g. the tables' capacity) serves every
 *             decode step while tangram_append_kv grows the cache; items beyond the current length are
 *             empty and a head with length 0 yields out = 0, lse = -inf.
 *   Hq        query heads, Hq % H == 0, G = Hq / H <= 16 (<= 8 at d = 256; query head j uses KV head floor(j / G))
 *   d         64, 128 or 256;  page size P 16, or 32 at d <= 128 (tangram_upload refuses any other P)
 *   sm_scale  softmax scale; 0 means 1/sqrt(d)
 *   out       device [R][Hq][d] bf16;  lse device [R][Hq] f32 (natural log of sum exp(scaled score);
 *             -inf and out = 0 for a head with kv_len 0)
 *   workspace device, >= tangram_workspace_bytes(dp->n_part_slots, G, d), 16-byte aligned
 *   worker_ns device [n_static][4] u64 or NULL: if given, every CTA stores its globaltimer stamps
 *             {start, end of its work lists, its last wait for a sequence's parts ended, merges done} (the last two only when
 *             the merge runs inside the decode grid; without it -- tangram_decode_partials -- the third slot
 *             holds the id of the SM the CTA ran on, %smid); the per-CTA elapsed-time spread of BASELINE.json
 *             is measured from the first two.
 * A device plan carries the launch's scheduler counters: launches on the SAME plan must be ordered (one stream, or
 * events between streams); different plans (e.g. one per layer) may run concurrently.  A grid that fits the device
 * (n_static <= SMs x occupancy: tangram_query_max_ctas) is launched cooperatively, so its in-grid waits are safe next
 * to any other work; a larger grid is a plain launch with no wait inside (merge, lengths and table growth run in
 * follow-up kernels), safe next to other work as well, just slower -- not a serving configuration.
 * Computes, for every (r, j): softmax(q_j K~^T * sm_scale) V~ over exactly the kv_len retained
 * tokens of its KV head (Eq. 1, :57), fp32 accumulation, bf16 output.
 * Errors: INVALID_ARG (shape / alignment / unsupported P / d / G / n_pool_pages <= a page id of the tables),
 * BUFFER_TOO_SMALL (workspace), CUDA. */
int tangram_decode_attention(const tangram_device_plan* dp, const void* q, const void* kv_pool,
                             int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq, int32_t d,
                             float sm_scale, void* out,
                             float* lse, void* workspace, size_t workspace_bytes,
                             uint64_t* worker_ns, void* stream);

/* Host buffers.  out and lse of tangram_decode_attention may be PINNED host memory (page-locked memory is mapped
 * into the device's address space under unified addressing): the kernel's stores then go over the bus as posted
 * writes and the result never waits for a copy engine.  q must be DEVICE memory: the kernel fetches query groups with
 * bulk asynchronous copies, and those hang now and then when pointed at mapped host memory (measured on B200), so a
 * host q is refused with INVALID_ARG.  Host-resident queries go through tangram_decode_attention_host below, or are
 * staged by this helper: it copies `bytes` (a multiple of 16) from pinned host memory `src_host` to device memory
 * `dst_dev` with a kernel on `stream` -- for the few hundred KB of a decode step ~10 us sooner than a copy-engine
 * transfer plus its stream hand-off.  Errors: INVALID_ARG (NULL, alignment, source not page-locked), CUDA. */
int tangram_stage_from_host(void* dst_dev, const void* src_host, size_t bytes, void* stream);

/* tangram_decode_attention with HOST buffers, end to end in ONE launch: the consumer warps of CTA b copy the query
 * blocks b, b + grid, ... (G x d bf16 per (request, KV head)) from q_host (pinned) to q_stage_dev (device, R x Hq x d
 * bf16, 16-byte aligned) when the CTA starts -- every block crosses the bus once, while the producer warps already
 * stream KV tiles -- and publish a per-block flag (dp->q_flags); a producer waits for the flag of the block its item
 * needs.  out and lse may be pinned host pointers (the kernel's stores go over the bus).  When the grid cannot be
 * launched cooperatively (or d = 256) the staging kernel of tangram_stage_from_host runs first and the decode kernel
 * is launched behind it with programmatic stream serialization.  All other arguments and errors as for
 * tangram_decode_attention and tangram_stage_from_host. */
int tangram_decode_attention_host(const tangram_device_plan* dp, const void* q_host, void* q_stage_dev,
                                  const void* kv_pool, int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq,
                                  int32_t d, float sm_scale, void* out, float* lse, void* workspace,
                                  size_t workspace_bytes, uint64_t* worker_ns, void* stream);

/* Measurement aid: reads `bytes` (a multiple of 16) of device memory once with 16-byte streaming loads on all SMs
 * and discards them -- a read-only HBM stream, the ceiling a4 can be held against (bench.py `roofline.read_peak_gbs`).
 * sink_dev: device u32 scratch.  Errors: INVALID_ARG, CUDA. */
int tangram_read_stream(const void* src_dev, size_t bytes, uint32_t* sink_dev, void* stream);

/* The two kernels of tangram_decode_attention as separate calls (same arguments, same checks):
 * a4 alone (split-KV decode kernel: final outputs of single-part sequences, fp32 partials of the
 * others into `workspace`) and a5 alone (LSE merge of the partials in `workspace` into out / lse;
 * zero-length sequences get out = 0, lse = -inf).  decode_partials followed by merge_partials on the
 * same stream is exactly tangram_decode_attention; they exist so that each kernel can be timed and
 * profiled on its own. */
int tangram_decode_partials(const tangram_device_plan* dp, const void* q, const void* kv_pool,
                            int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq, int32_t d,
                            float sm_scale, void* out,
                            float* lse, void* workspace, size_t workspace_bytes, uint64_t* worker_ns,
                            void* stream);
int tangram_merge_partials(const tangram_device_plan* dp, int32_t Hq, int32_t d, void* out, float* lse,
                           void* workspace, size_t workspace_bytes, void* stream);

/* ------------------------------------------------------------------------------------------------
 * tangram_decode_attention for callers that have no device memory to give and must not allocate any.
 *
 * Who that is.  The decode attention of a serving engine runs in the engine's steady state: at start-up the engine
 * measures the model and hands ALL the HBM that is left to its KV page pool (the Block Pool of PAPER.md:89), so when
 * the per-layer attention call comes there is nothing left for cudaMalloc to return; and a cudaMalloc / cudaFree issued
 * from the decode loop would in any case synchronise the whole device in the middle of the step and can stall against
 * a collective that is in flight on another stream.  The same holds for an attention plug-in loaded into a process
 * whose device memory belongs to somebody else's allocator (a framework's caching allocator, a memory-budgeted
 * container): it is not the plug-in's place to take memory behind that allocator's back.  Such callers still own q,
 * the pool, out and lse -- what they do not have is the split-KV WORKSPACE (the fp32 partial outputs and partial LSEs
 * of every multi-part sequence), which is pure scratch between the decode kernel and the merge.
 *
 * What this call does about it.  It is tangram_decode_attention, same kernels and same results, with the workspace
 * taken from a fixed array of TANGRAM_STATIC_WORKSPACE_BYTES (8 MiB) that is part of the library image: every GPU
 * that loads libtangram.so holds those 8 MiB from module load until the process exits, whether or not this call is
 * ever made.  The call itself performs no cudaMalloc, cudaFree or any other allocating CUDA / library routine, on the
 * first call or on any later one.
 *
 *   - Limit: tangram_workspace_bytes(dp->n_part_slots, Hq / H, d) must be <= TANGRAM_STATIC_WORKSPACE_BYTES, else
 *     TANGRAM_ERR_BUFFER_TOO_SMALL ("... static workspace ...") and nothing is launched.  8 MiB holds about 4 000
 *     part slots at G = 4, d = 128; on a 148-CTA grid the five configurations of BASELINE.json need 11 KB (tiny),
 *     2.0 MB (8b), 4.0 MB (32b), 1.8 MB (skew) and 6.3 MB (uniform, 256 requests).  Plans with more parts need the
 *     caller-workspace call.
 *   - First call on a device: the array's device address is looked up once per device (with that device current,
 *     as it is for the launch) and kept; this first call should be made before any stream capture is begun.
 *   - One array per GPU, shared by EVERY call of this entry point on that GPU, whatever the plan, stream or host
 *     thread: two such calls that overlap on the GPU (two streams, or two processes' worth of plans in one process)
 *     write each other's partials -- a race, silently wrong results.  Order them (one stream, or events), or give
 *     all but one of them a workspace of their own through tangram_decode_attention.
 *   - The array keeps whatever the last call left in it.  Nothing in it has to start at zero: every partial a merge
 *     reads was written earlier in the same call (the counters that order the two live in the plan's blob, not
 *     here), so no clearing is done or needed.
 * Arguments, results, asynchrony on `stream` and errors otherwise exactly as tangram_decode_attention. */
#define TANGRAM_STATIC_WORKSPACE_BYTES (8u << 20)
int tangram_decode_attention_static(const tangram_device_plan* dp, const void* q, const void* kv_pool,
                                    int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq, int32_t d,
                                    float sm_scale, void* out, float* lse, uint64_t* worker_ns, void* stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-1  KV append of one decode step.  The new K row and V row of every (request,
 * KV head) are written behind its retained tokens in the ragged pages (:190 page layout), and its length
 * grows by one.  A head whose (request, cluster) row holds no page for the new token (row_pages x P tokens
 * are full: tight tables, or a row the table growth above could not serve) keeps its length; its row is
 * dropped and counted.
 *
 *   dp            from tangram_upload (uses the tables only)
 *   k_new, v_new  device [R][H][d] bf16, 16-byte aligned
 *   kv_pool       device [n_pool_pages][Hp][2][P][d] bf16 (written)
 *   kv_len_dev    device [R][H] i32, read and incremented
 *   overflow_dev  device i32 or NULL: incremented once per dropped row
 * Asynchronous on `stream`; graph capturable.  Errors: INVALID_ARG, CUDA. */
int tangram_append_kv(const tangram_device_plan* dp, const void* k_new, const void* v_new, void* kv_pool,
                      int64_t n_pool_pages, int32_t d, int32_t* kv_len_dev, int32_t* overflow_dev,
                      void* stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-4 (second half)  Vectorized Block Table: growing the page tables during decode.
 * PAPER.md:89 ("between consecutive forward passes, a scheduling step requests the pages required for the next
 * pass from the Block Pool"), :244 (the per-group block mappings of all groups are aggregated into a Vectorized
 * Block Table and updated together -- OpenMP across head groups, SIMD inside a group -- because the cost grows with
 * the number of groups, O(N_req x H / H_p)), :176 (what overflow means: truncation of the compressor's selection,
 * not the loss of decode tokens).
 *
 * One update visits every (request, cluster) row, r-major then by cluster.  A row whose LONGEST head has filled
 * the row's pages (max_{h in c} kv_len[r][h] >= row_pages x P) takes the next page of the free list -- the list
 * the tables were built from, whose first n_pages_used entries are taken -- into its first unassigned slot.  A row
 * with no unassigned slot left (headroom used up), or reached after the free list ran out, stays as it is and is
 * counted as starved; only then does tangram_append_kv / tangram_decode_step drop that row's next token.  At most
 * one page per row and call (a decode step appends one token per head).  Results are bit-exact against the oracle
 * (O12) on either path.
 *
 * Host path (a scheduler that owns the tables): tangram_extend_tables updates *t in place; the rows that need a
 * page are found for all groups at once (OpenMP across (cluster, block of requests), AVX-512 gathers / max /
 * compare inside a block when the CPU has it, else the same loop in scalar code), then the pages are handed out
 * in row order.  tangram_sync_tables copies the tables' current state over the device copy of an uploaded plan.
 *   t           tables built with headroom_pages > 0 (row_pages present); updated in place
 *   kv_len      host [R][H] i32 current lengths          free_pages host [n_free] i32, the build's free list
 *   n_threads   OpenMP threads for the row scan; <= 0: one thread per 2048 rows, at most the OpenMP default
 *   n_extended_out / n_starved_out  host, may be NULL: rows that took a page / rows that needed one and got none
 * Errors: INVALID_ARG.
 *
 * Device path (zero host work per step, CUDA-graph capturable): tangram_extend_tables_device runs the same update
 * on the device copy (one small kernel: a block-wide ordered scan over the rows); the free-list cursor and the
 * starved count live in dp->grow_state.  tangram_decode_step below runs it inside the decode kernel.
 *   free_pages_dev  device [n_free] i32: the free list the tables were built from.  Every entry must be a page of
 *                   the pool the attention calls are given.  tangram_decode_step knows the pool's size and hands out
 *                   no entry outside [0, n_pool_pages) (the row counts as starved instead);
 *                   tangram_extend_tables_device and tangram_sync_tables do not know it and cannot check, so as the
 *                   last line of defence tangram_append_kv and the fused append never STORE through a page id outside
 *                   the pool they are given (tangram_append_kv keeps the length and counts the row in overflow_dev;
 *                   reads of such a page are clamped by the hardware).
 * tangram_download_tables copies the device state (tbl_pages, row_pages, n_pages_used) back into *t (host arrays
 * sized as at build time) and synchronises the stream. */
int tangram_extend_tables(tangram_tables* t, const int32_t* kv_len, const int32_t* free_pages, int64_t n_free,
                          int32_t n_threads, int64_t* n_extended_out, int64_t* n_starved_out);
int tangram_extend_tables_device(const tangram_device_plan* dp, const int32_t* kv_len_dev, const int32_t* free_pages_dev,
                                 int64_t n_free, void* stream);
int tangram_sync_tables(const tangram_tables* t, const tangram_device_plan* dp, void* stream);
int tangram_download_tables(const tangram_device_plan* dp, tangram_tables* t, int64_t* n_starved_out, void* stream);

/* ------------------------------------------------------------------------------------------------
 * One decode step of one layer in ONE launch: KV append (NEXT-1) + split-KV attention (a4) + LSE merge (a5) +
 * block-table update for the next step (NEXT-4), on an OPEN-ENDED plan (built for the tables' slot capacity).
 *
 *   1. append   the new K / V row of every (request, KV head) goes to token index n = kv_len[r][h] of its ragged
 *               pages if its row holds a page for that token (n < row_pages x P), else it is dropped and counted
 *               in *overflow_dev.  The row is written by the CTA whose work item covers token n, just before it
 *               streams that item -- no extra launch, no grid-wide dependency.
 *   2. attend   exactly as tangram_decode_attention over the n + 1 tokens (the new one included).
 *   3. lengths  kv_len_dev[r][h] becomes n + 1 (unchanged for a dropped row).
 *   4. grow     if free_pages_dev != NULL: the block-table update described above, with the new lengths, so that
 *               the NEXT step's token has a page.  (Run tangram_extend_tables_device once before the first step.)
 * Steps 3 and 4 run on the CTA that is the last to run out of work lists (every append has happened then), while the
 * others merge; when the in-kernel merge is not available (d = 256, wide merge records) they run in a small
 * follow-up kernel.
 * The composition is bit-exact against the oracle's extend_tables -> append_kv -> attention for the pool, the
 * lengths, the tables and the counters; the attention output is within the a4 tolerances.
 *
 *   k_new, v_new  device [R][H][d] bf16, 16-byte aligned          kv_pool  device, read and written
 *   kv_len_dev    device [R][H] i32 (required), read, then incremented
 *   flags         TANGRAM_STEP_OVERLAP: the caller guarantees that the work preceding this call on the stream
 *                 writes nothing this call reads except q, k_new and v_new (true for the layers of one decode
 *                 step, each with its own plan, pool and lengths; NOT true when the preceding launch is a step
 *                 on the same plan -- it writes this call's lengths, tables and pool).  The kernel is then launched with programmatic stream serialization and fetches its
 *                 work lists, page ids and first KV tiles while its predecessor drains; it waits for the
 *                 predecessor (griddepcontrol.wait) before touching q / k_new / v_new.
 *   all other arguments as for tangram_decode_attention.
 * Errors: as tangram_decode_attention, plus INVALID_ARG for kv_len_dev == NULL. */
#define TANGRAM_STEP_OVERLAP 1u
/* 1 once a launch with TANGRAM_STEP_OVERLAP was accepted by the driver, 0 if it was refused (the flag is then
 * ignored and the steps run back to back), -1 before the first such launch. */
int tangram_overlap_state(void);
int tangram_decode_step(const tangram_device_plan* dp, const void* q, const void* k_new, const void* v_new,
                        void* kv_pool, int64_t n_pool_pages, int32_t* kv_len_dev, const int32_t* free_pages_dev,
                        int64_t n_free, int32_t Hq, int32_t d, float sm_scale, void* out, float* lse, void* workspace,
                        size_t workspace_bytes, int32_t* overflow_dev, uint32_t flags, uint64_t* worker_ns, void* stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-2  Per-head Top-k selection + compaction into the ragged pages.
 * PAPER.md:152-154 (Eq. 4: I_{l,h} = Top(ceil(B_{l,h} N), s_{l,h}) -- every head selects on its own scores
 * with its own static budget), :57-58 (Eq. 1: K~ = K[I,:], V~ = V[I,:]), :190 (the retained rows live in
 * the ragged pages of the head's group), :176 (the reserved budget is a hard capacity bound).
 *
 * For every (request r, KV head h): the keep[r][h] highest-scoring tokens among the first ctx_len[r] are
 * selected -- scores compared as the fp32 values they are (-0 == +0), among equal scores the lower token
 * index wins -- and their K rows and V rows are written, in ascending token order, to token slots
 * 0 .. keep-1 of head h's pages: pool[tbl_pages[row(r, cluster_of[h]) + pos / P]][slot_of[h]][kv][pos % P][:].
 * Nothing else in the pool is written.  Scores must not be NaN (their order is then unspecified).
 *
 *   dp            from tangram_upload (uses the tables only)
 *   scores        device [R][H][n_max] f32   importance of every token (entries >= ctx_len[r] are ignored)
 *   k_dense, v_dense  device [R][H][n_max][d] bf16, 16-byte aligned: the uncompressed cache
 *   ctx_len_dev   device [R] i32, 1 <= ctx_len[r] <= n_max <= 2^30
 *   keep_dev      device [R][H] i32  tokens to retain (= kv_len of a1).  A value outside
 *                 [0, min(ctx_len[r], pages(r, cluster) x P)] is clamped into it and the head is counted
 *   kv_pool       device [n_pool_pages][Hp][2][P][d] bf16 (written)
 *   idx_out       device [R][H][n_max] i32: the first keep[r][h] entries of row (r, h) receive the retained
 *                 token indices in ascending order (the set I of Eq. 4); the rest is not touched
 *   clamped_dev   device i32 or NULL: incremented by the number of clamped heads
 *   workspace     device, >= tangram_compact_workspace_bytes(R, H), 16-byte aligned
 * Asynchronous on `stream`; graph capturable.  Three launches (prepare, select, gather), each behind its predecessor
 * programmatically: the select is set up while the prepare kernel runs and waits for its results; the gather moves a
 * row as soon as that row's selection is written (per-row ready flags), so select and gather overlap; the call is
 * complete when the gather grid is.  TANGRAM_COMPACT_OVERLAP = 0 / 1 in the
 * environment forces the gather-heavy decision (whether the select leaves half of every SM to the gather), a
 * measurement aid; by default it is taken from the batch.  Errors: INVALID_ARG, BUFFER_TOO_SMALL, CUDA. */
size_t tangram_compact_workspace_bytes(int32_t R, int32_t H);
int tangram_compact_topk(const tangram_device_plan* dp, const float* scores, const void* k_dense,
                         const void* v_dense, int64_t n_max, const int32_t* ctx_len_dev, const int32_t* keep_dev,
                         void* kv_pool, int64_t n_pool_pages, int32_t d, int32_t* idx_out, int32_t* clamped_dev,
                         void* workspace, size_t workspace_bytes, void* stream);

/* The same for ONE PREFILL CHUNK -- PAPER.md:152 ("each prefill chunk is compressed as soon as its KV cache is
 * generated, fully fusing compression into chunked prefill"): scores / k_dense / v_dense hold the chunk
 * (chunk_len_dev[r] tokens of request r), the keep[r][h] highest-scoring tokens of the chunk are selected as above
 * and their rows are written to token slots kv_len[r][h] .. kv_len[r][h] + keep - 1 of head h -- behind what the
 * head already holds -- and kv_len_dev[r][h] (device [R][H] i32, read and updated) grows by keep.  keep is clamped
 * into [0, min(chunk_len[r], pages(r, cluster) x P - kv_len[r][h])] and clamped heads are counted (:176).
 * idx_out receives token indices inside the chunk.  All other arguments as for tangram_compact_topk, which is this
 * call with every kv_len = 0 and no update. */
int tangram_compact_topk_chunk(const tangram_device_plan* dp, const float* scores, const void* k_dense,
                               const void* v_dense, int64_t n_max, const int32_t* chunk_len_dev, const int32_t* keep_dev,
                               int32_t* kv_len_dev, void* kv_pool, int64_t n_pool_pages, int32_t d, int32_t* idx_out,
                               int32_t* clamped_dev, void* workspace, size_t workspace_bytes, void* stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-3  Page accounting under a grouping policy (host, pure).  PAPER.md:168 (Fig. 7: a page is freed only when
 * all heads sharing it are evicted; monolithic / ragged / clustered), :190 (a group's page table is sized by its
 * largest budget), :192 ("naively grouping adjacent heads mixes dissimilar budgets"), :235-242 (H_p trade-off),
 * :244 (block-table cost O(N_req x H / H_p)), :316-320 (Fig. 15: memory reclaimed as a fraction of the full KV cache).
 *
 *   B         host [H] f64   calibrated budgets (only their order is used: TANGRAM_GROUP_CLUSTERED sorts by them
 *                            exactly as tangram_build_ragged_tables does)
 *   reserved  host [R][H] i32 (from a1)      ctx_len  host [R] i32
 *   heads_per_page  H_p, must divide H (H_p = H: the monolithic page of one layer)
 *   policy    TANGRAM_GROUP_CLUSTERED (H_p consecutive heads of the budget-sorted order, :227-233) or
 *             TANGRAM_GROUP_ADJACENT (H_p consecutive heads in index order)
 *   out       unit = token-head slot (one token of one head, K and V):
 *               pages_alloc = sum_r sum_groups ceil(max_{h in g} reserved[r][h] / P)
 *               slots_alloc = H_p * P * pages_alloc;   slots_exact = sum_r sum_h P * ceil(reserved[r][h] / P)
 *               slots_full  = sum_r H * P * ceil(N_r / P);   slots_used = sum reserved;   tables = R * H / H_p
 *               reclaimed_frac = 1 - slots_alloc / slots_full;  fragmentation = (slots_alloc - slots_used) / slots_alloc
 * Errors: INVALID_ARG (NULL, R/H < 1, H % H_p != 0, page_size < 1, reserved < 0, ctx_len < 1, unknown policy). */
#define TANGRAM_GROUP_CLUSTERED 0
#define TANGRAM_GROUP_ADJACENT 1
typedef struct tangram_page_account {
    int64_t pages_alloc, slots_alloc, slots_exact, slots_full, slots_used, tables;
    double reclaimed_frac, fragmentation;
} tangram_page_account;
int tangram_account_pages(const double* B, const int32_t* reserved, const int32_t* ctx_len, int32_t R, int32_t H,
                          int32_t heads_per_page, int32_t page_size, int32_t policy, tangram_page_account* out);

/* ------------------------------------------------------------------------------------------------
 * NEXT-4  Budget Calibration (host, pure).  PAPER.md:156-158: on a small set of sample contexts the implicit
 * per-head retention ratio of the global top-k selection is recorded and summarised by its mean and standard
 * deviation; Eq. 5 fixes B = min(1, mu + alpha sigma) (50 samples, alpha = 2 in the paper, :262).
 *
 *   ratios    host [n_samples][H] f64   ratio head h received on sample i
 *   mu_out, sigma_out, B_out   host [H] f64:  mu = (sum_i x_i) / n,  sigma = sqrt((sum_i (x_i - mu)^2) / n) -- the
 *             POPULATION standard deviation (the paper does not say which) -- sums in sample order, fp64, no FMA;
 *             B as in tangram_reserve_budgets (B_out may be NULL)
 * Errors: INVALID_ARG (NULL, n_samples < 1, H < 1, a ratio that is not finite). */
int tangram_calibrate_budgets(const double* ratios, int32_t n_samples, int32_t H, double alpha, double* mu_out,
                              double* sigma_out, double* B_out);

/* NEXT-4 (device)  Implicit per-head retention ratios of the global flat Top-k -- PAPER.md:68-77 (Eq. 3:
 * I_l = Top(ceil(rho H N), s^flat) over the scores of all H heads of a layer flattened together), :156 (Budget
 * Calibration records the ratio each head receives from that selection on every sample context; the rows of
 * tangram_calibrate_budgets' `ratios` input).
 *
 *   scores       device [R][H][n_max] f32 (entries >= ctx_len[r] ignored); H * n_max < 2^31
 *   ctx_len_dev  device [R] i32, 1 <= ctx_len[r] <= n_max        rho in [0, 1]
 *   counts_out   device [R][H] i32: entries of head h among the ceil(rho * H * N_r) highest-scoring ones of request
 *                r; s^flat is head-major, scores compared as fp32 values (-0 == +0), ties to the lower flat index
 *   ratios_out   device [R][H] f64 = counts / N_r
 * Asynchronous on `stream` (one launch, one CTA per request).  Errors: INVALID_ARG, CUDA. */
int tangram_implicit_ratios(const float* scores, int32_t R, int32_t H, int64_t n_max, const int32_t* ctx_len_dev,
                            double rho, int32_t* counts_out, double* ratios_out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* TANGRAM_H_ */
