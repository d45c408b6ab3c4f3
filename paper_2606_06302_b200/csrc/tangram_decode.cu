// Tangram decode attention for B200 (sm_100a): split-KV decode kernel driven by the Ahead-of-Time
// work list (a4) and the log-sum-exp merge kernel (a5).  Contract: include/tangram.h.
//
// Decode kernel, one persistent CTA per worker (one per SM):
//   * warp 8 is the producer.  Lane 0 hands every item's descriptor and query group to the consumers
//     through a 2-slot ring (cp.async.bulk of the contiguous G x d bf16 block).  Lanes 0-7 each feed
//     the private tile ring of one consumer warp: one TMA tensor copy (cp.async.bulk.tensor, 128-byte
//     swizzle) per (page, head) brings the page's K rows and V rows -- one contiguous 2*P*d*2-byte run
//     of the ragged page pool[page][slot][kv][token][d] -- into shared memory and completes on that
//     stage's mbarrier.  Page ids are read one round ahead; the producer runs ahead across item
//     boundaries, so the HBM stream never drains between items.
//   * warps 0-7 are consumers.  Tile i of an item goes to warp (i + rot) % 8.  Per tile (16 tokens):
//     S = Q K^T with mma.sync m16n8k16 (bf16 in, fp32 accumulate; the GQA group sits in rows 0..G-1 of
//     the 16-row A operand), fp32 online softmax in the exp2 domain with a warp-uniform lazy rescale,
//     O += P V with V fragments from ldmatrix.trans.  At the end of an item the eight (m, l, O)
//     states are combined through shared memory and the CTA writes either the final bf16 output
//     (n_parts == 1) or an fp32 partial (o, lse).
// The path is HBM-bound (4*d bytes per token-head against 4*d*G flop); the tensor cores are used
// because at G = 4..5 the CUDA-core formulation would need ~50 warp instructions per 512 bytes and
// B200 has only ~7 bytes of HBM bandwidth per issue slot.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <type_traits>
#include <vector>

#include "tangram.h"
#include "tangram_internal.h"

namespace tangram {

// Page sizes (tokens per page) the kernels are instantiated for: 16 and 32.  One TMA box = the 2 P rows (K then V)
// of one (page, head): 8 KB at P = 16, d = 128; 16 KB at P = 32, d = 128 or P = 16, d = 256.
static bool page_supported(int P, int d) { return P == 16 || (P == 32 && d <= 128); }
// consumer warps of the decode kernel: 8, or 4 where one (page, head) tile is 16 KB and eight three-stage rings
// would not fit in shared memory
template <int D, int PAGE>
constexpr int consumer_warps() { return 2 * PAGE * D * 2 >= 16384 ? 4 : 8; }
constexpr int kMinQSlots = 2;      // item / query ring depth: as deep as shared memory allows, 2 .. 8 (runtime).  A deep
constexpr int kMaxQSlots = 8;      // ring lets the producer fetch query groups several items ahead
constexpr int kMaxStages = 8;      // per-consumer-warp tile ring depth (runtime <= this)
constexpr int kMaxG = 16;         // GQA groups above 8 use both halves of the 16-row A operand (d <= 128)
constexpr int kSmemLimit = 232448; // 227 KB opt-in limit per CTA
constexpr int kRunSplit = 1, kRunMerge = 2;
#ifndef TANGRAM_CLAIM_TILES
#define TANGRAM_CLAIM_TILES 16
#endif
constexpr int kClaimTiles = TANGRAM_CLAIM_TILES;  // how many tiles before the end of a list its successor is claimed

// Block-table state of an uploaded plan as the growth code sees it (NEXT-4).
struct GrowParams {
    const int32_t* row_ptr;      // [n_rows + 1] first slot of every (request, cluster) row
    int32_t* row_pages;          // [n_rows] pages a row holds
    const int32_t* perm;         // [H]
    int32_t* tbl_pages;          // page id per slot, -1 = none yet
    int32_t* seq_cap;            // [R*H] row_pages x P of the head's row
    const int32_t* plan_cover;   // [R*H] tokens the plan's items cover
    int32_t* kv_len;             // [R*H]
    int32_t* grow_state;         // {free-list cursor, rows starved so far}
    const int32_t* free_pages;   // [n_free] or nullptr: no growth
    int32_t* overflow;           // dropped rows, or nullptr
    int32_t n_free, n_rows, R, H, C, Hp;
    int32_t n_pool_pages;        // pages of the pool the caller passed (INT32_MAX: not known to this call): a free-list
                                 // entry outside [0, n_pool_pages) is not handed out -- the row counts as starved
};

struct DecodeParams {
    const DeviceItem* items;
    const int64_t* worker_indptr;
    const int32_t* tbl_pages;
    const __nv_bfloat16* q;
    __nv_bfloat16* out;
    float* lse;
    float* part_o;
    float* part_lse;
    unsigned long long* worker_ns;
    int* sched;  // [0] next list to claim (relative to gridDim.x), [1] CTAs done claiming, [2] tickets taken (CTAs
                 // out of work), [3] CTAs done merging; all 0 between launches (the kernel re-arms them);
                 // [4] launches that staged host queries on this plan (the epoch of q_flags); [5] launches that
                 // merged in-grid on this plan (the epoch of seq_done)
    unsigned* seq_done;  // [R*H] parts written so far, summed over the in-grid-merging launches on this plan
    const int32_t* merge_recs;  // merge records (see a5)
    const void* list_heads;     // [n_lists] 128-byte list heads
    const int32_t* kv_len;      // [R*H] run-time lengths (open-ended plan) or nullptr: items are taken as planned
    int32_t H, R;
    int32_t Hq, G, Hp, n_stages, n_qslots, n_lists;
    int32_t tail_merge, n_merge_units, n_merge_small, merge_split, merge_ctas;
    float scale_log2;
    // fused decode step (tangram_decode_step): KV append by the CTA that streams the sequence's last item, the
    // length update and the block-table growth for the next step after the grid barrier; all nullptr / 0 otherwise
    const uint4* k_new;          // [R*H][d/8] or nullptr: no append
    const uint4* v_new;
    uint4* pool_w;               // the page pool, writable view
    int32_t n_pool_pages;        // its pages: an appended row is only stored to a page id inside [0, n_pool_pages)
    const int32_t* seq_cap;      // [R*H] tokens the row's pages hold
    int32_t* kv_len_w;           // = kv_len, writable
    GrowParams grow;
    int32_t pdl;                 // launched with programmatic stream serialization: wait before reading q / k_new / v_new
    int32_t early_trigger;       // 1: dependents may be launched while this grid runs (griddepcontrol.launch_dependents)
    // host-resident queries (tangram_decode_attention_host, cooperative launch only): the consumer warps of CTA b
    // copy query blocks b, b + grid, ... from pinned host memory to `q` (device) when the CTA starts and publish each
    // block's flag; a producer waits for the flag of the block its item needs.  nullptr otherwise.
    const uint4* q_host;
    int32_t* q_flags;            // [R*H] launch number (epoch) in which the block was staged last
};

// ------------------------------------------------------------------ shared-memory carve-up
template <int D, int PAGE>
struct Smem {
    static constexpr int kNW = consumer_warps<D, PAGE>();
    static constexpr int kThreads = (kNW + 1) * 32;          // + the producer warp
    static constexpr int kTile = 2 * PAGE * D * 2;           // K rows + V rows of one (page, head)
    static constexpr int kHalf = 2 * PAGE * 128;             // one 64-element column block of the tile
    static constexpr int kRowF = D + 8;                      // padded fp32 row of the merge scratch
    __host__ __device__ static int q_slot(int G) { return (G * D * 2 + 127) & ~127; }
    __host__ __device__ static int off_q(int ns) { return kNW * ns * kTile; }
    __host__ __device__ static int off_desc(int ns, int G, int nq) { return off_q(ns) + nq * q_slot(G); }
    __host__ __device__ static int off_scratch(int ns, int G, int nq) { return off_desc(ns, G, nq) + nq * 32; }
    // merge scratch: 8 warp states of G padded rows; also reused by the tail merge (256 threads x 6 floats)
    __host__ __device__ static int scratch_bytes(int G) {
        return kNW * G * kRowF * 4 > kNW * 32 * 6 * 4 ? kNW * G * kRowF * 4 : kNW * 32 * 6 * 4;
    }
    __host__ __device__ static int off_ml(int ns, int G, int nq) { return off_scratch(ns, G, nq) + scratch_bytes(G); }
    __host__ __device__ static int off_bar(int ns, int G, int nq) { return (off_ml(ns, G, nq) + kNW * G * 8 + 15) & ~15; }
    __host__ __device__ static int off_flag(int ns, int G, int nq) {
        return off_bar(ns, G, nq) + (2 * kNW * kMaxStages + 2 * kMaxQSlots) * 8;
    }
    __host__ __device__ static int total(int ns, int G, int nq) {
        return off_flag(ns, G, nq) + 16 + 1024 /* base alignment slack */;
    }
    static int max_stages(int G) {
        int ns = kMaxStages;
        while (ns > 1 && total(ns, G, kMinQSlots) > kSmemLimit) --ns;
        return ns;
    }
    static int max_qslots(int ns, int G) {  // what is left after the tile rings goes to the query ring
        int nq = kMaxQSlots;
        while (nq > kMinQSlots && total(ns, G, nq) > kSmemLimit) --nq;
        return nq;
    }
};

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_tile(uint32_t dst, const CUtensorMap* map, uint32_t bar, int row,
                                              uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(dst),
        "l"(map), "r"(0), "r"(row), "r"(0), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr)
                 : "memory");
}
// D(16x8) += A(16x16) B(16x8), bf16 inputs, fp32 accumulate.  Only rows 0..7 of A are populated
// (the GQA group), so a1 = a3 = 0 and the row 8..15 halves of the accumulator are discarded.
__device__ __forceinline__ void mma_rows07(float& c0, float& c1, uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1) {
    [[maybe_unused]] float d2, d3;
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%10,%10};"
        : "+f"(c0), "+f"(c1), "=f"(d2), "=f"(d3)
        : "r"(a0), "r"(0u), "r"(a2), "r"(0u), "r"(b0), "r"(b1), "f"(0.f));
}
// The full 16-row form (GQA groups of 9..16 query heads): rows 0..7 accumulate into (c0, c1), rows 8..15 into (c2, c3).
__device__ __forceinline__ void mma_rows16(float& c0, float& c1, float& c2, float& c3, uint32_t a0, uint32_t a1, uint32_t a2,
                                           uint32_t a3, uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c0), "+f"(c1), "+f"(c2), "+f"(c3)
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ unsigned long long globaltimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// ------------------------------------------------------------------ a5: LSE merge
// The merge records list the sequences (r * H + h) whose part count is not 1 (built at upload time:
// empty sequences first, then sequences with at most kMergeBigParts parts, then the "big" ones).
// Sequences with one part were written by the decode kernel; sequences with no retained token get
// out = 0, lse = -inf.  A merge UNIT is a whole small record (all G query heads) or one query head of a
// big record; unit u of a launch is decoded by unit_of().  Within a unit a thread owns four adjacent
// output elements (one float4 of a partial row, so a row is read by D/4 adjacent threads) and one of
// PG part groups (parts k, k + PG, ...) with eight loads in flight and running-max accumulation (one
// pass); the group sums are then combined in group order.  The summation order is a function of
// (n, G, D, thread count) only, so the result is deterministic.
constexpr int kMergeThreads = 512;
#ifndef TANGRAM_MERGE_BIG_PARTS
#define TANGRAM_MERGE_BIG_PARTS 16
#endif
constexpr int kMergeBigParts = TANGRAM_MERGE_BIG_PARTS;  // records with more parts are merged by whole-CTA units
#ifndef TANGRAM_MERGE_BATCH
#define TANGRAM_MERGE_BATCH 8
#endif
constexpr int kMergeBatch = TANGRAM_MERGE_BATCH;  // partial rows a thread of the small-record merge keeps in flight
#ifndef TANGRAM_BARRIER_NANOSLEEP
#define TANGRAM_BARRIER_NANOSLEEP 32
#endif

struct MergeUnit {
    int seq, p0, n, g;  // g < 0: all query heads of the group (small record)
    int c0, cb;         // big record: the unit's block of float4 columns [c0, c0 + cb) of the D/4 of a row
};
// Units [0, n_small) are the small records; then every big record gives G * S units, S = column blocks per row.
__device__ __forceinline__ MergeUnit unit_of(const int32_t* __restrict__ recs, int n_small, int u, int G, int S, int D4) {
    const int v = u - n_small;
    const int r = u < n_small ? u : n_small + v / (G * S);
    const int4 rec = reinterpret_cast<const int4*>(recs)[r];  // {seq, first part slot, parts, -}
    if (u < n_small) return MergeUnit{rec.x, rec.y, rec.z, -1, 0, D4};
    return MergeUnit{rec.x, rec.y, rec.z, (v / S) % G, (v % S) * (D4 / S), D4 / S};
}

// One query head of a BIG record (a long sequence that the work lists dice into up to thousands of parts), one
// block of cb float4 columns: thread (grp, c) accumulates parts grp, grp + PG, ... of column c0 + c with eight
// loads in flight, PG = NT / cb part groups; the group states are then combined by a fixed binary tree through
// shared memory.  The narrower the column block, the more part groups work on the record at once: with cb = 1 a
// CTA covers 8 * NT parts per round trip, and a record's G * D/4 units spread over the whole grid -- a single
// 2^20-token sequence in 1036 parts merges in ~3 us instead of ~15 us with one CTA per query head.  The order
// of the additions is a function of (n, cb, NT) only: deterministic.
template <int D, int NT, bool NAMED_BAR>
__device__ __forceinline__ void merge_big_unit(const MergeUnit mu, int G, const float* __restrict__ part_o,
                                               const float* __restrict__ part_lse, __nv_bfloat16* __restrict__ out,
                                               float* __restrict__ lse, float (*s_part)[6], int tid) {
    auto sync = [] {
        if constexpr (NAMED_BAR) named_bar_sync(1, NT);
        else __syncthreads();
    };
    const int cb = mu.cb, PG = NT / cb;
    const int c = tid % cb, grp = tid / cb, c4 = mu.c0 + c, n = mu.n;
    const size_t row = static_cast<size_t>(mu.seq) * G + mu.g;  // (r*H + h)*G + g = r*Hq + h*G + g
    float m = -INFINITY, tot = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    {
        const float* pl = part_lse + static_cast<size_t>(mu.p0) * G + mu.g;  // [part][g]
        const float* po = part_o + (static_cast<size_t>(mu.p0) * G + mu.g) * D + c4 * 4;
        const size_t stride = static_cast<size_t>(G) * D;
        for (int i = grp; i < n; i += 8 * PG) {
            float4 v[8];
            float w[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int ii = i + u * PG;
                const int ic = ii < n ? ii : i;
                v[u] = __ldcg(reinterpret_cast<const float4*>(po + ic * stride));
                w[u] = ii < n ? __ldcg(pl + ic * G) : -INFINITY;
            }
            float m_new = m;
#pragma unroll
            for (int u = 0; u < 8; ++u) m_new = fmaxf(m_new, w[u]);
            const float resc = m_new == -INFINITY ? 1.f : __expf(m - m_new);  // m = -inf on the first batch -> 0
            tot *= resc, a0 *= resc, a1 *= resc, a2 *= resc, a3 *= resc;
            m = m_new;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float e = m == -INFINITY ? 0.f : __expf(w[u] - m);  // -inf -> 0; all parts empty so far -> 0
                tot += e, a0 += e * v[u].x, a1 += e * v[u].y, a2 += e * v[u].z, a3 += e * v[u].w;
            }
        }
    }
    float* mine = s_part[tid];
    mine[0] = m, mine[1] = tot, mine[2] = a0, mine[3] = a1, mine[4] = a2, mine[5] = a3;
    for (int half = PG >> 1; half >= 1; half >>= 1) {  // group grp takes in group grp + half
        sync();
        if (grp < half) {
            const float* o = s_part[(grp + half) * cb + c];
            const float M = fmaxf(m, o[0]);
            const float sa = M == -INFINITY ? 0.f : __expf(m - M), sb = M == -INFINITY ? 0.f : __expf(o[0] - M);
            tot = sa * tot + sb * o[1];
            a0 = sa * a0 + sb * o[2], a1 = sa * a1 + sb * o[3], a2 = sa * a2 + sb * o[4], a3 = sa * a3 + sb * o[5];
            m = M;
            mine[0] = m, mine[1] = tot, mine[2] = a0, mine[3] = a1, mine[4] = a2, mine[5] = a3;
        }
    }
    if (grp == 0) {
        const float inv = tot > 0.f ? 1.f / tot : 0.f;
        const __nv_bfloat162 lo = __floats2bfloat162_rn(a0 * inv, a1 * inv), hi = __floats2bfloat162_rn(a2 * inv, a3 * inv);
        reinterpret_cast<uint2*>(out + row * D)[c4] =
            make_uint2(*reinterpret_cast<const uint32_t*>(&lo), *reinterpret_cast<const uint32_t*>(&hi));
        if (c4 == 0) lse[row] = tot > 0.f ? m + __logf(tot) : -INFINITY;
    }
    sync();  // s_part may be reused by the next unit
}

template <int D, int NT, bool NAMED_BAR>
__device__ __forceinline__ void merge_unit(const MergeUnit mu, int G, const float* __restrict__ part_o,
                                           const float* __restrict__ part_lse, __nv_bfloat16* __restrict__ out,
                                           float* __restrict__ lse, float (*s_part)[6], int tid) {
    auto sync = [] {
        if constexpr (NAMED_BAR) named_bar_sync(1, NT);
        else __syncthreads();
    };
    const int rows = mu.g < 0 ? G : 1;
    const int n_elem = rows * (D / 4);  // float4 elements of the unit's output rows (<= 256)
    const size_t row0 = static_cast<size_t>(mu.seq) * G + (mu.g < 0 ? 0 : mu.g);  // (r*H + h)*G + g = r*Hq + h*G + g
    const int n = mu.n;
    if (n == 0) {
        if (tid < n_elem) reinterpret_cast<uint2*>(out + row0 * D)[tid] = make_uint2(0u, 0u);
        if (tid < rows) lse[row0 + tid] = -INFINITY;
        return;
    }
    const int PG = NT / n_elem;  // part groups
    const int e4 = tid % n_elem, grp = tid / n_elem;
    const int gl = e4 / (D / 4), c4 = e4 % (D / 4);  // row inside the unit, float4 column
    const int g = mu.g < 0 ? gl : mu.g;
    float m = -INFINITY, tot = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    if (grp < PG) {
        const float* pl = part_lse + static_cast<size_t>(mu.p0) * G + g;  // [part][g]
        const float* po = part_o + (static_cast<size_t>(mu.p0) * G + g) * D + c4 * 4;
        const size_t stride = static_cast<size_t>(G) * D;
        for (int i = grp; i < n; i += 8 * PG) {
            float4 v[8];
            float w[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int ii = i + u * PG;
                const int ic = ii < n ? ii : i;
                v[u] = __ldcg(reinterpret_cast<const float4*>(po + ic * stride));
                w[u] = ii < n ? __ldcg(pl + ic * G) : -INFINITY;
            }
            float m_new = m;
#pragma unroll
            for (int u = 0; u < 8; ++u) m_new = fmaxf(m_new, w[u]);
            const float resc = m_new == -INFINITY ? 1.f : __expf(m - m_new);  // m = -inf on the first batch -> 0
            tot *= resc, a0 *= resc, a1 *= resc, a2 *= resc, a3 *= resc;
            m = m_new;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float e = m == -INFINITY ? 0.f : __expf(w[u] - m);  // -inf -> 0; all parts empty so far -> 0
                tot += e, a0 += e * v[u].x, a1 += e * v[u].y, a2 += e * v[u].z, a3 += e * v[u].w;
            }
        }
        float* sp = s_part[tid];
        sp[0] = m, sp[1] = tot, sp[2] = a0, sp[3] = a1, sp[4] = a2, sp[5] = a3;
    }
    sync();
    if (grp == 0) {
        float M = m;
        for (int k = 1; k < PG; ++k) M = fmaxf(M, s_part[k * n_elem + e4][0]);
        float sc = M == -INFINITY ? 0.f : __expf(m - M);
        tot *= sc, a0 *= sc, a1 *= sc, a2 *= sc, a3 *= sc;
        for (int k = 1; k < PG; ++k) {
            const float* sp = s_part[k * n_elem + e4];
            sc = M == -INFINITY ? 0.f : __expf(sp[0] - M);  // a group without parts has m = -inf -> 0
            tot += sc * sp[1], a0 += sc * sp[2], a1 += sc * sp[3], a2 += sc * sp[4], a3 += sc * sp[5];
        }
        const float inv = tot > 0.f ? 1.f / tot : 0.f;
        const __nv_bfloat162 lo = __floats2bfloat162_rn(a0 * inv, a1 * inv), hi = __floats2bfloat162_rn(a2 * inv, a3 * inv);
        reinterpret_cast<uint2*>(out + (row0 + gl) * D)[c4] =
            make_uint2(*reinterpret_cast<const uint32_t*>(&lo), *reinterpret_cast<const uint32_t*>(&hi));
        if (c4 == 0) lse[row0 + gl] = tot > 0.f ? M + __logf(tot) : -INFINITY;
    }
    sync();  // s_part may be reused by the next unit
}

// A small record (at most kMergeBigParts parts) merged by G * D/4 threads, one float4 element each, every
// part visited in order: no shared memory, no barrier, so the sub-groups of a CTA merge different
// records at the same time.
template <int D>
__device__ __forceinline__ void merge_small(const int4 rec, int G, const float* __restrict__ part_o,
                                            const float* __restrict__ part_lse, __nv_bfloat16* __restrict__ out,
                                            float* __restrict__ lse, int e4) {
    constexpr int kB = kMergeBatch;  // loads in flight per thread
    const int n = rec.z, g = e4 / (D / 4), c4 = e4 % (D / 4);
    const size_t row = static_cast<size_t>(rec.x) * G + g;
    if (n == 0) {
        reinterpret_cast<uint2*>(out + row * D)[c4] = make_uint2(0u, 0u);
        if (c4 == 0) lse[row] = -INFINITY;
        return;
    }
    const float* pl = part_lse + static_cast<size_t>(rec.y) * G + g;
    const float* po = part_o + (static_cast<size_t>(rec.y) * G + g) * D + c4 * 4;
    const size_t stride = static_cast<size_t>(G) * D;
    float m = -INFINITY, tot = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    for (int i = 0; i < n; i += kB) {
        float4 v[kB];
        float w[kB];
#pragma unroll
        for (int u = 0; u < kB; ++u) {
            const int ic = i + u < n ? i + u : i;
            v[u] = __ldcg(reinterpret_cast<const float4*>(po + ic * stride));
            w[u] = i + u < n ? __ldcg(pl + ic * G) : -INFINITY;
        }
        float m_new = m;
#pragma unroll
        for (int u = 0; u < kB; ++u) m_new = fmaxf(m_new, w[u]);
        const float resc = m_new == -INFINITY ? 1.f : __expf(m - m_new);
        tot *= resc, a0 *= resc, a1 *= resc, a2 *= resc, a3 *= resc;
        m = m_new;
#pragma unroll
        for (int u = 0; u < kB; ++u) {
            const float e = m == -INFINITY ? 0.f : __expf(w[u] - m);  // parts of an open-ended plan may be empty
            tot += e, a0 += e * v[u].x, a1 += e * v[u].y, a2 += e * v[u].z, a3 += e * v[u].w;
        }
    }
    const float inv = tot > 0.f ? 1.f / tot : 0.f;
    const __nv_bfloat162 lo = __floats2bfloat162_rn(a0 * inv, a1 * inv), hi = __floats2bfloat162_rn(a2 * inv, a3 * inv);
    reinterpret_cast<uint2*>(out + row * D)[c4] =
        make_uint2(*reinterpret_cast<const uint32_t*>(&lo), *reinterpret_cast<const uint32_t*>(&hi));
    if (c4 == 0) lse[row] = tot > 0.f ? m + __logf(tot) : -INFINITY;
}

// Stand-alone merge kernel (tangram_merge_partials, and the fallback of tangram_decode_attention when
// the grid cannot be launched cooperatively): one CTA per unit.
template <int D>
__global__ void __launch_bounds__(kMergeThreads)
tangram_merge_kernel(const int32_t* __restrict__ merge_recs, int n_small, const float* __restrict__ part_o,
                     const float* __restrict__ part_lse, __nv_bfloat16* __restrict__ out,
                     float* __restrict__ lse, int G, int S) {
    __shared__ float s_part[kMergeThreads][6];
    const MergeUnit mu = unit_of(merge_recs, n_small, blockIdx.x, G, S, D / 4);
    // everything above reads plan data only; the partials / outputs need the decode grid to be done
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (mu.g < 0) merge_unit<D, kMergeThreads, false>(mu, G, part_o, part_lse, out, lse, s_part, threadIdx.x);
    else merge_big_unit<D, kMergeThreads, false>(mu, G, part_o, part_lse, out, lse, s_part, threadIdx.x);
}

// ------------------------------------------------------------------ NEXT-4: block-table growth on the device
// The lengths of one decode step and the Vectorized Block Table update by ONE thread block of
// NT threads (a power of two): thread i owns rows i, i + NT, ...  A row that needs a page and has a free slot takes
// free_pages[cursor + (number of such rows before it)] -- a block-wide exclusive scan keeps the oracle's row order.
template <int NT, bool NAMED_BAR>
__device__ __forceinline__ void block_sync() {
    if constexpr (NAMED_BAR) named_bar_sync(1, NT);
    else __syncthreads();
}

// kv_len[seq] += 1 for every sequence whose appended row was stored (its row holds a page for token n and the plan
// has an item covering it); the others are counted as dropped.
template <int NT, bool NAMED_BAR>
__device__ __forceinline__ void step_lengths(const GrowParams& g, int tid) {
    for (int seq = tid; seq < g.R * g.H; seq += NT) {
        const int n = g.kv_len[seq];
        if (n < g.seq_cap[seq] && n < g.plan_cover[seq]) g.kv_len[seq] = n + 1;
        else if (g.overflow) atomicAdd(g.overflow, 1);
    }
    block_sync<NT, NAMED_BAR>();
}

template <int NT, bool NAMED_BAR>
__device__ __forceinline__ void extend_rows(const GrowParams& g, int page_tokens, int tid, int* s_scan /* >= 33 ints */) {
    const int lane = tid & 31, wid = tid >> 5;
    const int cursor0 = g.grow_state[0];
    int granted = 0;  // pages asked for by the rows of earlier chunks (same value in every thread)
    for (int row0 = 0; row0 < g.n_rows; row0 += NT) {
        const int row = row0 + tid;
        bool want = false, can = false;
        int have = 0, lo = 0, r = 0, c = 0;
        if (row < g.n_rows) {
            r = row / g.C, c = row % g.C;
            int longest = 0;
            for (int k = 0; k < g.Hp; ++k) longest = max(longest, g.kv_len[r * g.H + g.perm[c * g.Hp + k]]);
            have = g.row_pages[row], lo = g.row_ptr[row];
            want = longest >= have * page_tokens;
            can = want && have < g.row_ptr[row + 1] - lo;
        }
        // block-wide exclusive scan of `can`
        const unsigned bal = __ballot_sync(0xffffffffu, can);
        if (lane == 0) s_scan[wid] = __popc(bal);
        block_sync<NT, NAMED_BAR>();
        if (wid == 0) {
            const int v = lane < NT / 32 ? s_scan[lane] : 0;
            int inc = v;
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            s_scan[lane] = inc - v;                      // exclusive prefix of the warp totals
            if (lane == 31) s_scan[32] = inc;            // chunk total
        }
        block_sync<NT, NAMED_BAR>();
        const int idx = cursor0 + granted + s_scan[wid] + __popc(bal & ((1u << lane) - 1u));
        const int total = s_scan[32];
        // a free-list entry that is not a page of the pool is never written into the tables (the appends store through
        // the tables without a hardware bound, unlike the TMA reads): the row is starved instead
        const int new_page = can && idx < g.n_free ? g.free_pages[idx] : -1;
        const bool ok = new_page >= 0 && new_page < g.n_pool_pages;
        if (ok) {
            g.tbl_pages[lo + have] = new_page;
            g.row_pages[row] = have + 1;
            for (int k = 0; k < g.Hp; ++k) g.seq_cap[r * g.H + g.perm[c * g.Hp + k]] = (have + 1) * page_tokens;
        }
        if (want && !ok) atomicAdd(g.grow_state + 1, 1);
        granted += total;
        block_sync<NT, NAMED_BAR>();                     // s_scan is reused by the next chunk
    }
    if (tid == 0) g.grow_state[0] = min(cursor0 + granted, max(cursor0, g.n_free));
}

// Stand-alone: tangram_extend_tables_device (do_lengths = 0) and the follow-up of tangram_decode_step when the
// decode grid cannot run its tail phase (do_lengths = 1).
__global__ void __launch_bounds__(1024) tangram_grow_kernel(const GrowParams g, int page_tokens, int do_lengths) {
    __shared__ int s_scan[33];
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (do_lengths) step_lengths<1024, false>(g, threadIdx.x);
    if (g.free_pages) extend_rows<1024, false>(g, page_tokens, threadIdx.x, s_scan);
}

// ------------------------------------------------------------------ a4: split-KV decode kernel
template <int D, bool TIMED, int NH, int PAGE>
__global__ void __launch_bounds__(Smem<D, PAGE>::kThreads, 1)
tangram_decode_kernel(const __grid_constant__ CUtensorMap kv_map, const DecodeParams p) {
    using L = Smem<D, PAGE>;
    constexpr int kPage = PAGE;
    constexpr int kNW = L::kNW;
    constexpr int kTile = L::kTile, kHalf = L::kHalf, kRowF = L::kRowF;
    extern __shared__ uint8_t smem_raw[];
    // 128-byte-swizzled TMA tiles need a 1024-byte aligned base
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));

    const int NS = p.n_stages, NQ = p.n_qslots, G = p.G;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t tiles = smem_u32(smem);
    uint8_t* q_ring = smem + L::off_q(NS);
    uint8_t* desc_ring = smem + L::off_desc(NS, G, NQ);
    float* scratch_o = reinterpret_cast<float*>(smem + L::off_scratch(NS, G, NQ));
    float* scratch_ml = reinterpret_cast<float*>(smem + L::off_ml(NS, G, NQ));
    const uint32_t bars = smem_u32(smem + L::off_bar(NS, G, NQ));
    const int q_slot_bytes = L::q_slot(G);
    auto full_bar = [&](int w, int s) { return bars + (w * kMaxStages + s) * 8; };
    auto empty_bar = [&](int w, int s) { return bars + (kNW * kMaxStages + w * kMaxStages + s) * 8; };
    auto qfull_bar = [&](int s) { return bars + (2 * kNW * kMaxStages + s) * 8; };
    auto qempty_bar = [&](int s) { return bars + (2 * kNW * kMaxStages + kMaxQSlots + s) * 8; };

    if (TIMED && threadIdx.x == 0) {
        p.worker_ns[4 * blockIdx.x] = globaltimer();
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        p.worker_ns[4 * blockIdx.x + 2] = smid;  // kept by tangram_decode_partials; the in-grid merge overwrites it
    }
    // The CTA's own list head (plan data) is on its way while the barriers are set up: the first TMA of the CTA
    // is then one memory round trip behind the start of the CTA, not two.
    int head_word = 0;
    if (warp == kNW) {
        head_word = __ldg(reinterpret_cast<const int*>(p.list_heads) + static_cast<size_t>(blockIdx.x) * 32 + lane);
        if (lane == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(&kv_map) : "memory");
    }
    if (threadIdx.x == 0) {
        for (int w = 0; w < kNW; ++w)
            for (int s = 0; s < NS; ++s) {
                mbar_init(full_bar(w, s), 1);
                mbar_init(empty_bar(w, s), 1);
            }
        for (int s = 0; s < NQ; ++s) {
            mbar_init(qfull_bar(s), 1);
            mbar_init(qempty_bar(s), kNW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kNW) {
        // ============================== producer warp ==============================
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
        uint32_t stage = 0, phase = 0;  // lane w < 8 tracks consumer warp w's ring
        // Work lists: list blockIdx.x is this CTA's own; with a dynamic tail (n_lists > gridDim.x) further
        // lists are claimed from a global counter.  The claim is issued as late as possible -- when the
        // producer starts the LAST item of the current list -- so that a CTA never sits on a list another
        // CTA could already run; its latency is covered by that item's TMA issue, and the consumers still
        // hold a full ring (192 KB) of tiles while the next list's range and first item are fetched.
        const bool dynamic = p.n_lists > static_cast<int>(gridDim.x);
        auto claim = [&]() {
            int v = 0;
            if (lane == 0) v = atomicAdd(p.sched, 1) + static_cast<int>(gridDim.x);
            return v;
        };
        // Open-ended plan: an item ends where its sequence ends NOW.  In a fused decode step (k_new given) the
        // sequence gains one token in this launch if its row holds a page for it; the item that covers that
        // token index is the sequence's TAIL item, and the CTA that runs it stores the new K / V row first.
        auto open_end = [&](DeviceItem& it, bool& tail) {
            tail = false;
            if (!p.kv_len) return;
            const int sq = it.req * p.H + it.kv_head;
            int n = __ldcg(p.kv_len + sq);
            if (p.k_new) {
                const bool room = n < __ldcg(p.seq_cap + sq);
                tail = room && it.tok_begin <= n && n < it.tok_end;
                n += room ? 1 : 0;
            }
            it.tok_end = min(it.tok_end, n);
        };
        // One 128-byte list head (a single coalesced load, lane L reads word L) carries the list's item
        // range, its first item and that item's first 16 page ids, so the first TMA of a list is two
        // dependent memory round trips away from the claim instead of four.
        int64_t cb, ce;
        DeviceItem next;
        bool next_tail = false;
        int head_pid_lo = 0, head_pid_hi = 0;  // page ids of tiles (lane - rot) mod NW and that + NW of the list's first item
        auto take_head = [&](int w) {
            cb = __shfl_sync(0xffffffffu, w, 0);
            ce = cb + __shfl_sync(0xffffffffu, w, 1);
            next.req = __shfl_sync(0xffffffffu, w, 4), next.kv_head = __shfl_sync(0xffffffffu, w, 5);
            next.tbl_row = __shfl_sync(0xffffffffu, w, 6), next.slot = __shfl_sync(0xffffffffu, w, 7);
            next.tok_begin = __shfl_sync(0xffffffffu, w, 8), next.tok_end = __shfl_sync(0xffffffffu, w, 9);
            next.part_slot = __shfl_sync(0xffffffffu, w, 10), next.n_parts = __shfl_sync(0xffffffffu, w, 11);
            if (ce > cb) open_end(next, next_tail);
            const int i0 = (lane - (next.part_slot & (kNW - 1))) & (kNW - 1);
            head_pid_lo = __shfl_sync(0xffffffffu, w, 12 + i0);
            head_pid_hi = __shfl_sync(0xffffffffu, w, 12 + kNW + i0);
        };
        // Page ids: through the read-only (non-coherent) path only in launches that cannot write the tables; a fused
        // decode step grows them in its tail phase (extend_rows), so there they are read from L2.
        const bool tables_grow = p.k_new != nullptr;
        auto load_pid = [&](const int32_t* a) { return tables_grow ? __ldcg(a) : __ldg(a); };
        auto load_head = [&](int list) {
            take_head(__ldg(reinterpret_cast<const int*>(p.list_heads) + static_cast<size_t>(list) * 32 + lane));
        };
        take_head(head_word);
        // Programmatic dependent launch (tangram_decode_step with TANGRAM_STEP_OVERLAP): everything up to here read
        // plan data, lengths and tables, which the predecessor on the stream does not write.  The producer may
        // also fill its (empty) tile rings with the first item's KV tiles -- the cache is not the predecessor's
        // either -- and only then waits for the predecessor, before the first q / k_new / v_new access.
        bool pdl_wait = p.pdl != 0;
        int prefilled = 0;              // tiles of the first item already issued per lane (0 .. NS)
        int pre_pid = 0;                // page id of the lane's next tile after the prefill
        if (pdl_wait) {
            if (ce > cb && !next_tail && lane < kNW) {
                const int n_tiles = max(0, next.tok_end - next.tok_begin + kPage - 1) / kPage;
                const int32_t* ids = p.tbl_pages + next.tbl_row + next.tok_begin / kPage;
                int i = (lane - (next.part_slot & (kNW - 1))) & (kNW - 1);
                int pid = head_pid_lo;
                if (i < n_tiles && pid < 0) pid = load_pid(ids + i);
                while (i < n_tiles && prefilled < NS) {
                    const int i_next = i + kNW;
                    int pid_next = i_next < 2 * kNW ? head_pid_hi : 0;
                    if (i_next < n_tiles && (i_next >= 2 * kNW || pid_next < 0)) pid_next = load_pid(ids + i_next);
                    mbar_arrive_expect_tx(full_bar(lane, stage), kTile);
                    tma_load_tile(tiles + (lane * NS + stage) * kTile, &kv_map, full_bar(lane, stage),
                                  (pid * p.Hp + next.slot) * (2 * kPage), policy);
                    if (++stage == static_cast<uint32_t>(NS)) stage = 0, phase ^= 1;
                    i = i_next, pid = pid_next, ++prefilled;
                }
                pre_pid = pid;
            }
            __syncwarp();
            asm volatile("griddepcontrol.wait;" ::: "memory");
        }
        // The next launch on the stream may be scheduled -- unless this grid waits inside (in-grid merge) and is NOT
        // gang-scheduled: CTAs of a dependent grid that became resident early would sit on SMs (waiting for this grid
        // to complete) that CTAs of this grid still need, and the waits in the tail phase would never end.
        if (p.early_trigger) asm volatile("griddepcontrol.launch_dependents;");
        const int q_epoch = p.q_host ? __ldcg(p.sched + 4) + 1 : 0;
        int seq = 0;  // running item number = position in the item / query ring
        for (;;) {
            int fut = 0;
            if (dynamic && cb == ce) fut = claim();
            for (int64_t it = cb; it < ce; ++it, ++seq) {
                const DeviceItem item = next;
                const bool tail = next_tail;
                const bool head_item = it == cb;
                if (it + 1 < ce) {
                    next = p.items[it + 1];
                    open_end(next, next_tail);
                }
                const bool claim_here = dynamic && it + 1 == ce;  // last item of the list: claim the next list
                const int qs = seq % NQ;
                const uint32_t qpar = (seq / NQ) & 1;
                if (tail) {
                    // fused KV append: token index tok_end - 1 is the new one.  16-byte chunks of the K row then
                    // the V row; the proxy fence orders these generic-proxy stores before the TMA (async proxy)
                    // reads of the same page issued below by this warp.
                    const int n = item.tok_end - 1;
                    const int page = __ldcg(p.tbl_pages + item.tbl_row + n / kPage);
                    const size_t row_k = ((static_cast<size_t>(page) * p.Hp + item.slot) * 2) * kPage + n % kPage;
                    const size_t sq = static_cast<size_t>(item.req) * p.H + item.kv_head;
                    constexpr int chunks = D / 8;
                    // (a page id outside the pool -- tables synced from a host that was given a wrong free list --
                    // is never stored through; the TMA reads of such a page are clamped by the tensor map)
                    for (int c = lane; c < 2 * chunks && static_cast<unsigned>(page) < static_cast<unsigned>(p.n_pool_pages); c += 32) {
                        const bool is_v = c >= chunks;
                        const int cc = is_v ? c - chunks : c;
                        const uint4 val = __ldcg((is_v ? p.v_new : p.k_new) + sq * chunks + cc);
                        p.pool_w[(row_k + (is_v ? kPage : 0)) * chunks + cc] = val;
                    }
                    asm volatile("fence.proxy.async;" ::: "memory");
                    __syncwarp();
                }
                if (lane == 0) {
                    mbar_wait(qempty_bar(qs), qpar ^ 1);
                    *reinterpret_cast<DeviceItem*>(desc_ring + qs * 32) = item;
                    if (p.q_host) {  // the item's query block is staged by some CTA's consumer warps: wait for its flag
                        const int32_t* flag = p.q_flags + item.req * p.H + item.kv_head;
                        int seen;
                        TANGRAM_SPIN_INIT;
                        do {
                            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(flag) : "memory");
                            TANGRAM_SPIN_POLL(TANGRAM_WAIT_Q_FLAG, item.req * p.H + item.kv_head);
                        } while (seen != q_epoch);
                        asm volatile("fence.proxy.async;" ::: "memory");  // generic-proxy stores -> bulk (async proxy) read
                    }
                    const uint32_t qbytes = static_cast<uint32_t>(G * D * 2);
                    mbar_arrive_expect_tx(qfull_bar(qs), qbytes);
                    bulk_load(smem_u32(q_ring + qs * q_slot_bytes),
                              p.q + (static_cast<size_t>(item.req) * p.Hq + static_cast<size_t>(item.kv_head) * G) * D,
                              qbytes, qfull_bar(qs));
                }
                const int n_tiles = max(0, item.tok_end - item.tok_begin + kPage - 1) / kPage;
                const int rot = item.part_slot & (kNW - 1);  // which warp gets the item's first tile
                if (lane < kNW) {
                    const int32_t* ids = p.tbl_pages + item.tbl_row + item.tok_begin / kPage;
                    int i = (lane - rot) & (kNW - 1);
                    int pid;
                    if (prefilled) {  // (first item of a PDL launch: its first tiles are already in flight)
                        i += prefilled * kNW, pid = pre_pid, prefilled = 0;
                    } else {
                        pid = head_item ? head_pid_lo : 0;
                        // a list head caches the page ids its first item had at upload time; a slot that got its
                        // page later (table growth) is read from the table
                        if (i < n_tiles && (!head_item || pid < 0)) pid = load_pid(ids + i);
                    }
                    // lane 0 issues the claim kClaimTiles tiles before the end of the item's TMA issue: late
                    // enough that the CTA does not hoard a list, early enough to cover the claim -> list
                    // head -> first TMA chain (~3 us) with tiles that are still being issued
                    bool to_claim = claim_here && lane == 0;
                    while (i < n_tiles) {
                        if (to_claim && i + kClaimTiles >= n_tiles) {
                            fut = atomicAdd(p.sched, 1) + static_cast<int>(gridDim.x);
                            to_claim = false;
                        }
                        const int i_next = i + kNW;
                        int pid_next = head_item && i_next < 2 * kNW ? head_pid_hi : 0;
                        if (i_next < n_tiles && (!head_item || i_next >= 2 * kNW || pid_next < 0)) pid_next = load_pid(ids + i_next);
                        mbar_wait(empty_bar(lane, stage), phase ^ 1);
                        mbar_arrive_expect_tx(full_bar(lane, stage), kTile);
                        tma_load_tile(tiles + (lane * NS + stage) * kTile, &kv_map, full_bar(lane, stage),
                                      (pid * p.Hp + item.slot) * (2 * kPage), policy);
                        if (++stage == static_cast<uint32_t>(NS)) stage = 0, phase ^= 1;
                        i = i_next, pid = pid_next;
                    }
                    if (to_claim) fut = atomicAdd(p.sched, 1) + static_cast<int>(gridDim.x);
                }
                prefilled = 0;
                __syncwarp();
            }
            if (!dynamic) break;
            const int nxt = __shfl_sync(0xffffffffu, fut, 0);
            if (nxt >= p.n_lists) break;
            load_head(nxt);
        }
        if (lane == 0) {
            // end-of-work sentinel for the consumers
            const int qs = seq % NQ;
            mbar_wait(qempty_bar(qs), ((seq / NQ) & 1) ^ 1);
            DeviceItem stop{};
            stop.n_parts = -1;
            *reinterpret_cast<DeviceItem*>(desc_ring + qs * 32) = stop;
            mbar_arrive(qfull_bar(qs));
            if (dynamic) {
                // the last CTA to finish re-arms the counters for the next launch on this plan
                if (atomicAdd(p.sched + 1, 1) == static_cast<int>(gridDim.x) - 1) p.sched[0] = 0, p.sched[1] = 0;
            }
        }
        return;
    }

    // ================================ consumer warps ================================
    if (p.q_host) {
        // Queries in pinned host memory: this CTA's share of the R*H query blocks (G x d bf16 each) crosses the bus
        // once, now, while the producer already streams KV tiles; sched[4] counts the launches on this plan.
        const int epoch = __ldcg(p.sched + 4) + 1;
        const int n_blocks = p.R * p.H, v16 = G * D / 8;  // 16-byte words per block
        auto stage = [&](int blk) {
            const uint4* src = p.q_host + static_cast<size_t>(blk) * v16;
            uint4* dst = reinterpret_cast<uint4*>(const_cast<__nv_bfloat16*>(p.q)) + static_cast<size_t>(blk) * v16;
            for (int i = lane; i < v16; i += 32) dst[i] = src[i];
            __threadfence();
            __syncwarp();
            if (lane == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p.q_flags + blk), "r"(epoch) : "memory");
        };
        if (warp == kNW - 1) {
            // the block this CTA's own first item needs goes first (several CTAs may fetch the same block: harmless),
            // so that no CTA's start waits behind the whole batch on the bus
            const int* hd = reinterpret_cast<const int*>(p.list_heads) + static_cast<size_t>(blockIdx.x) * 32;
            if (__ldg(hd + 1) > 0) stage(__ldg(hd + 4) * p.H + __ldg(hd + 5));
        }
        for (int blk = static_cast<int>(blockIdx.x) + warp * static_cast<int>(gridDim.x); blk < n_blocks;
             blk += kNW * static_cast<int>(gridDim.x))
            stage(blk);
    }
    // Query head `row + 8 hf` of the GQA group is held by this quad in half hf of the 16-row A operand: NH = 1 uses
    // rows 0..7 only (G <= 8: the upper rows are fed zeros and their accumulators dropped), NH = 2 all sixteen.
    const int row = lane >> 2;
    const int qd = lane & 3;
    bool row_ok[NH];
#pragma unroll
    for (int hf = 0; hf < NH; ++hf) row_ok[hf] = row + 8 * hf < G;
    uint32_t stage = 0, phase = 0;
    constexpr float kNegInf = -INFINITY;

    for (int it = 0;; ++it) {
        const int qs = it % NQ;
        mbar_wait(qfull_bar(qs), (it / NQ) & 1);
        const DeviceItem item = *reinterpret_cast<const DeviceItem*>(desc_ring + qs * 32);
        if (item.n_parts < 0) break;  // producer's end-of-work sentinel
        uint32_t qa[NH][D / 16][2];
#pragma unroll
        for (int hf = 0; hf < NH; ++hf) {
            const uint8_t* qrow = q_ring + qs * q_slot_bytes + (row + 8 * hf) * D * 2;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                qa[hf][ks][0] = row_ok[hf] ? *reinterpret_cast<const uint32_t*>(qrow + (ks * 16 + qd * 2) * 2) : 0u;
                qa[hf][ks][1] = row_ok[hf] ? *reinterpret_cast<const uint32_t*>(qrow + (ks * 16 + 8 + qd * 2) * 2) : 0u;
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(qempty_bar(qs));

        const int n_tok = max(0, item.tok_end - item.tok_begin);  // 0: an open-ended item beyond the current length
        const int n_tiles = (n_tok + kPage - 1) / kPage;
        const int rot = item.part_slot & (kNW - 1);  // a function of the item only: results do not depend on which CTA runs it
        float m[NH], l[NH];
        float o[NH][D / 8][2];
#pragma unroll
        for (int hf = 0; hf < NH; ++hf) {
            m[hf] = kNegInf, l[hf] = 0.f;
#pragma unroll
            for (int nt = 0; nt < D / 8; ++nt) o[hf][nt][0] = o[hf][nt][1] = 0.f;
        }

        for (int i = (warp - rot) & (kNW - 1); i < n_tiles; i += kNW) {
            mbar_wait(full_bar(warp, stage), phase);
            const uint32_t tb = tiles + (warp * NS + stage) * kTile;
            const int tile_valid = min(kPage, n_tok - i * kPage);  // retained tokens in this (page, head) tile
            if (tile_valid < kPage) {
                // ragged tail: V rows of tokens that are not retained may hold anything (NaN
                // included) and 0 * NaN would poison the PV product -- zero them.
                if (lane < 8 * (D / 64))
                    for (int rr = kPage + tile_valid; rr < 2 * kPage; ++rr)
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(tb + (lane >> 3) * kHalf + rr * 128 +
                                                                                   (lane & 7) * 16),
                                     "r"(0u)
                                     : "memory");
                __syncwarp();
            }
            // a tile is processed 16 tokens at a time (one pass at P = 16, two at P = 32)
#pragma unroll 1
            for (int sb = 0; sb < kPage / 16; ++sb) {
            const int valid = min(16, tile_valid - sb * 16);
            if (valid <= 0) break;
            // ---- S = Q K^T : 16 query rows (8 or 16 used) x 16 tokens
            float s[NH][2][2];
#pragma unroll
            for (int hf = 0; hf < NH; ++hf) s[hf][0][0] = s[hf][0][1] = s[hf][1][0] = s[hf][1][1] = 0.f;
            {
                const int tok = sb * 16 + ((lane >> 4) << 3) + (lane & 7);
                const uint32_t rbase = tb + tok * 128;
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const int ck = ((ks & 3) << 1) + ((lane >> 3) & 1);
                    uint32_t b0, b1, b2, b3;
                    ldsm_x4(rbase + (ks >> 2) * kHalf + ((ck ^ (tok & 7)) << 4), b0, b1, b2, b3);
                    if constexpr (NH == 1) {
                        mma_rows07(s[0][0][0], s[0][0][1], qa[0][ks][0], qa[0][ks][1], b0, b1);
                        mma_rows07(s[0][1][0], s[0][1][1], qa[0][ks][0], qa[0][ks][1], b2, b3);
                    } else {
                        mma_rows16(s[0][0][0], s[0][0][1], s[NH - 1][0][0], s[NH - 1][0][1], qa[0][ks][0], qa[NH - 1][ks][0],
                                   qa[0][ks][1], qa[NH - 1][ks][1], b0, b1);
                        mma_rows16(s[0][1][0], s[0][1][1], s[NH - 1][1][0], s[NH - 1][1][1], qa[0][ks][0], qa[NH - 1][ks][0],
                                   qa[0][ks][1], qa[NH - 1][ks][1], b2, b3);
                    }
                }
            }
            // ---- online softmax (exp2 domain)
            float m_new[NH];
            bool grew = false;
#pragma unroll
            for (int hf = 0; hf < NH; ++hf) {
                float tmax = kNegInf;
#pragma unroll
                for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const float x = s[hf][nt][e] * p.scale_log2;
                        s[hf][nt][e] = (nt * 8 + qd * 2 + e < valid) ? x : kNegInf;
                        tmax = fmaxf(tmax, s[hf][nt][e]);
                    }
                tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
                tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
                m_new[hf] = fmaxf(m[hf], tmax);
                grew = grew || m_new[hf] > m[hf];
            }
            if (__any_sync(0xffffffffu, grew)) {
#pragma unroll
                for (int hf = 0; hf < NH; ++hf) {
                    const float corr = exp2f(m[hf] - m_new[hf]);  // m = -inf on the first tile -> 0
                    l[hf] *= corr;
#pragma unroll
                    for (int nt = 0; nt < D / 8; ++nt) o[hf][nt][0] *= corr, o[hf][nt][1] *= corr;
                    m[hf] = m_new[hf];
                }
            }
            uint32_t pa[NH][2];
#pragma unroll
            for (int hf = 0; hf < NH; ++hf) {
                const float p00 = exp2f(s[hf][0][0] - m[hf]), p01 = exp2f(s[hf][0][1] - m[hf]);
                const float p10 = exp2f(s[hf][1][0] - m[hf]), p11 = exp2f(s[hf][1][1] - m[hf]);
                l[hf] += (p00 + p01) + (p10 + p11);
                pa[hf][0] = pack_bf16(p00, p01), pa[hf][1] = pack_bf16(p10, p11);
            }
            // ---- O += P V
            {
                const int vrow = kPage + sb * 16 + (((lane >> 3) & 1) << 3) + (lane & 7);
                const uint32_t rbase = tb + vrow * 128;
#pragma unroll
                for (int cg = 0; cg < D / 8; cg += 2) {
                    const int ck = (cg & 7) + (lane >> 4);
                    uint32_t v0, v1, v2, v3;
                    ldsm_x4_t(rbase + (cg >> 3) * kHalf + ((ck ^ (vrow & 7)) << 4), v0, v1, v2, v3);
                    if constexpr (NH == 1) {
                        mma_rows07(o[0][cg][0], o[0][cg][1], pa[0][0], pa[0][1], v0, v1);
                        mma_rows07(o[0][cg + 1][0], o[0][cg + 1][1], pa[0][0], pa[0][1], v2, v3);
                    } else {
                        mma_rows16(o[0][cg][0], o[0][cg][1], o[NH - 1][cg][0], o[NH - 1][cg][1], pa[0][0], pa[NH - 1][0], pa[0][1],
                                   pa[NH - 1][1], v0, v1);
                        mma_rows16(o[0][cg + 1][0], o[0][cg + 1][1], o[NH - 1][cg + 1][0], o[NH - 1][cg + 1][1], pa[0][0],
                                   pa[NH - 1][0], pa[0][1], pa[NH - 1][1], v2, v3);
                    }
                }
            }
            }  // 16-token passes
            if (tile_valid < kPage) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(warp, stage));
            if (++stage == static_cast<uint32_t>(NS)) stage = 0, phase ^= 1;
        }

        // ---- combine the eight warp states of this item
#pragma unroll
        for (int hf = 0; hf < NH; ++hf) {
            l[hf] += __shfl_xor_sync(0xffffffffu, l[hf], 1);
            l[hf] += __shfl_xor_sync(0xffffffffu, l[hf], 2);
            if (row_ok[hf]) {
                float* so = scratch_o + (warp * G + row + 8 * hf) * kRowF + qd * 2;
#pragma unroll
                for (int nt = 0; nt < D / 8; ++nt)
                    *reinterpret_cast<float2*>(so + nt * 8) = make_float2(o[hf][nt][0], o[hf][nt][1]);
                if (qd == 0) *reinterpret_cast<float2*>(scratch_ml + (warp * G + row + 8 * hf) * 2) = make_float2(m[hf], l[hf]);
            }
        }
        named_bar_sync(1, kNW * 32);
        for (int idx = threadIdx.x; idx < G * (D / 2); idx += kNW * 32) {
            const int g = idx / (D / 2), c2 = idx % (D / 2);
            float mw[kNW], M = kNegInf;
#pragma unroll
            for (int w = 0; w < kNW; ++w) {
                mw[w] = scratch_ml[(w * G + g) * 2];
                M = fmaxf(M, mw[w]);
            }
            const bool none = M == kNegInf;  // no tile at all (empty open-ended item): o = 0, lse = -inf
            float Lsum = 0.f, ax = 0.f, ay = 0.f;
#pragma unroll
            for (int w = 0; w < kNW; ++w) {
                const float e = none ? 0.f : exp2f(mw[w] - M);  // warps without a tile have m = -inf -> weight 0
                Lsum += e * scratch_ml[(w * G + g) * 2 + 1];
                const float2 v = *reinterpret_cast<const float2*>(scratch_o + (w * G + g) * kRowF + c2 * 2);
                ax += e * v.x, ay += e * v.y;
            }
            const float inv = none ? 0.f : 1.f / Lsum;
            const float lse_nat = none ? kNegInf : (M + log2f(Lsum)) * 0.6931471805599453f;
            if (item.n_parts == 1) {
                const size_t hq = static_cast<size_t>(item.req) * p.Hq + static_cast<size_t>(item.kv_head) * G + g;
                *reinterpret_cast<__nv_bfloat162*>(p.out + hq * D + c2 * 2) = __floats2bfloat162_rn(ax * inv, ay * inv);
                if (c2 == 0) p.lse[hq] = lse_nat;
            } else {
                const size_t ps = static_cast<size_t>(item.part_slot) * G + g;
                *reinterpret_cast<float2*>(p.part_o + ps * D + c2 * 2) = make_float2(ax * inv, ay * inv);
                if (c2 == 0) p.part_lse[ps] = lse_nat;
            }
        }
        named_bar_sync(1, kNW * 32);  // scratch may be overwritten by the next item
        // In-grid merge: the part is published with one fire-and-forget release (every thread's stores precede the
        // barrier above, the release is cumulative) -- nobody waits for it here.
        if (p.tail_merge && item.n_parts != 1 && threadIdx.x == 0)
            asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p.seq_done + item.req * p.H + item.kv_head), "r"(1u)
                         : "memory");
    }
    if (TIMED && threadIdx.x == 0) p.worker_ns[4 * blockIdx.x + 1] = globaltimer();

    if (p.tail_merge) {
        // a5 inside the persistent grid, without a grid barrier.  Every multi-part item was published by a release
        // add on its sequence's counter (above); a CTA that is out of work lists merges its share of the records,
        // waiting record by record until the counter shows all the parts of THIS launch: (launches so far + 1) x parts
        // (the counters are never reset; unsigned wrap-around is harmless because a counter is only compared for
        // equality with a target it cannot overshoot).  Records are visited in sequence order -- the order in which
        // the work lists complete them -- so a CTA that runs out of work early merges what is already complete while
        // the others still stream, and after the last part of the launch is written only the records that contain
        // parts of the last lists remain.
        // Who may wait: a waiting CTA waits for parts that another CTA of the grid writes, so every CTA of the grid
        // must be resident: the launcher enables this phase only for a grid that fits on the device and launches it
        // cooperatively -- gang scheduling also keeps the CTAs of other grids, a programmatically dependent successor
        // in particular, off the SMs this grid still needs.  Every CTA takes a ticket when its
        // lists are done (merge_ctas = the grid; the ticket decides who does the step's bookkeeping below).
        // Small records: sub-group `sub` of G*D/4 threads takes records (first + j*M)*K + sub, every thread polls
        // and merges on its own, no barrier inside.  Big records (more than kMergeBigParts parts: the sequences the
        // last rounds of the dynamic tail dice finely) come after the small ones, one (query head, column block)
        // per unit.
        // In a fused decode step the very last arrival does not merge: all CTAs are out of work then, every append
        // has happened, and it updates the lengths and grows the block tables for the next step.
        const bool fused = p.k_new != nullptr;
        const int grid_all = static_cast<int>(gridDim.x);
        const int n_late = min(grid_all, p.merge_ctas);  // CTAs that stay for the tail phase
        int* s_ticket = reinterpret_cast<int*>(smem + L::off_flag(NS, G, NQ));
        __threadfence();
        named_bar_sync(1, kNW * 32);
        if (threadIdx.x == 0) *s_ticket = atomicAdd(p.sched + 2, 1);
        named_bar_sync(1, kNW * 32);
        const int rank = *s_ticket - (grid_all - n_late);  // < 0: an early arrival
        if (rank >= 0) {
            const int grid = fused && n_late > 1 ? n_late - 1 : n_late;  // the CTAs that merge
            const bool merger = rank < grid;
            const int n_elem = G * (D / 4), K = (kNW * 32) / n_elem, sub = threadIdx.x / n_elem;
            const int n_big_units = p.n_merge_units - p.n_merge_small;
            // the previous launch on this plan is complete (the producer waited for it before the first item)
            const unsigned epoch1 = static_cast<unsigned>(__ldcg(p.sched + 5)) + 1u;
            auto wait_parts = [&](int seq, int n) {  // every thread for itself: acquire, then its own loads
                const unsigned want = epoch1 * static_cast<unsigned>(n);
                unsigned seen;
                TANGRAM_SPIN_INIT;
                for (;;) {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(p.seq_done + seq) : "memory");
                    if (seen == want) break;
                    TANGRAM_SPIN_POLL(TANGRAM_WAIT_SEQ_PARTS, seq);
                    if (TANGRAM_BARRIER_NANOSLEEP > 0) __nanosleep(TANGRAM_BARRIER_NANOSLEEP);
                }
                if (TIMED && threadIdx.x == 0) p.worker_ns[4 * blockIdx.x + 2] = globaltimer();  // the CTA's last wait passed
            };
            float(*s_part)[6] = reinterpret_cast<float(*)[6]>(scratch_o);
            if (merger) {
                // ... the small records start at the CTA after the last one holding a big unit
                const int first = (rank - n_big_units % grid + grid) % grid;
                if (sub < K) {
                    int sidx = first * K + sub;
                    int4 rec = make_int4(0, 0, 0, 0);
                    if (sidx < p.n_merge_small) rec = __ldg(reinterpret_cast<const int4*>(p.merge_recs) + sidx);
                    for (; sidx < p.n_merge_small; sidx += grid * K) {
                        int4 nxt = make_int4(0, 0, 0, 0);
                        if (sidx + grid * K < p.n_merge_small)
                            nxt = __ldg(reinterpret_cast<const int4*>(p.merge_recs) + sidx + grid * K);
                        if (rec.z > 0) wait_parts(rec.x, rec.z);
                        merge_small<D>(rec, G, p.part_o, p.part_lse, p.out, p.lse, threadIdx.x - sub * n_elem);
                        rec = nxt;
                    }
                }
                if (n_big_units > 0) named_bar_sync(1, kNW * 32);  // the merge scratch is shared by the whole CTA
                for (int u = rank; u < n_big_units; u += grid) {
                    const MergeUnit mu = unit_of(p.merge_recs, p.n_merge_small, p.n_merge_small + u, G, p.merge_split, D / 4);
                    wait_parts(mu.seq, mu.n);
                    merge_big_unit<D, kNW * 32, true>(mu, G, p.part_o, p.part_lse, p.out, p.lse, s_part, threadIdx.x);
                }
            }
            if (fused && (!merger || n_late == 1)) {
                // the last ticket: every CTA is out of work, every append of this step has happened
                named_bar_sync(1, kNW * 32);
                step_lengths<kNW * 32, true>(p.grow, threadIdx.x);
                if (p.grow.free_pages) extend_rows<kNW * 32, true>(p.grow, kPage, threadIdx.x, reinterpret_cast<int*>(scratch_o));
            }
            // every merge thread of the CTA is done before "merges done" is stamped and the exit counter moves (the
            // last CTA out re-arms the tickets and closes the epoch)
            named_bar_sync(1, kNW * 32);
            if (TIMED && threadIdx.x == 0) p.worker_ns[4 * blockIdx.x + 3] = globaltimer();
        }
        if (threadIdx.x == 0 && atomicAdd(p.sched + 3, 1) == grid_all - 1) {
            p.sched[2] = 0, p.sched[3] = 0;  // last CTA out re-arms the tickets for the next launch
            p.sched[5] += 1;                 // ... closes this launch's merge epoch
            if (p.q_host) p.sched[4] += 1;   // ... and its query-staging epoch
        }
    }
}

// ------------------------------------------------------------------ NEXT-1: KV append
// One warp per (request, KV head): the new K row and V row (d bf16 each) go to token index
// n = kv_len[r][h] of the head's ragged pages; kv_len becomes n + 1.  A head whose row holds no page for
// token n (seq_cap = row_pages x P tokens are full) keeps its length and the row is counted in *overflow.
__global__ void __launch_bounds__(128)
tangram_append_kernel(const int4* __restrict__ seq_info, const int32_t* __restrict__ seq_cap,
                      const int32_t* __restrict__ tbl_pages,
                      const uint4* __restrict__ k_new, const uint4* __restrict__ v_new, uint4* __restrict__ pool,
                      int32_t* __restrict__ kv_len, int32_t* __restrict__ overflow, int n_seq, int Hp, int d, int kPage,
                      int n_pool_pages) {
    const int seq = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (seq >= n_seq) return;
    const int4 si = seq_info[seq];  // {first slot of the row, slot capacity in tokens, slot, row}
    const int n = kv_len[seq];
    if (n >= seq_cap[seq]) {
        if (lane == 0 && overflow) atomicAdd(overflow, 1);
        return;
    }
    const int chunks = d / 8;  // 16-byte chunks per row
    const int page = tbl_pages[si.x + n / kPage];
    if (static_cast<unsigned>(page) >= static_cast<unsigned>(n_pool_pages)) {  // not a page of this pool: never stored to
        if (lane == 0 && overflow) atomicAdd(overflow, 1);
        return;
    }
    // pool[page][slot][kv][token][d]
    const size_t row_k = ((static_cast<size_t>(page) * Hp + si.z) * 2 + 0) * kPage + n % kPage;
    const size_t row_v = ((static_cast<size_t>(page) * Hp + si.z) * 2 + 1) * kPage + n % kPage;
    for (int c = lane; c < 2 * chunks; c += 32) {
        const bool is_v = c >= chunks;
        const int cc = is_v ? c - chunks : c;
        const uint4 val = (is_v ? v_new : k_new)[static_cast<size_t>(seq) * chunks + cc];
        pool[(is_v ? row_v : row_k) * chunks + cc] = val;
    }
    __syncwarp();
    if (lane == 0) kv_len[seq] = n + 1;
}

// ------------------------------------------------------------------ staging small host buffers
// dst (device) <- src (pinned, device-mapped host memory), 16 bytes per thread and step.  For the few hundred KB of
// a decode step's queries a kernel that pulls the bytes over the bus is ready ~10 us sooner than a copy-engine
// transfer and its stream hand-off to the next kernel.
__global__ void __launch_bounds__(256)
tangram_stage_kernel(uint4* __restrict__ dst, const uint4* __restrict__ src, size_t n16) {
    asm volatile("griddepcontrol.launch_dependents;");  // a dependent decode kernel may start its prologue now
    for (size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n16;
         i += static_cast<size_t>(gridDim.x) * blockDim.x)
        dst[i] = src[i];
}

// ------------------------------------------------------------------ measurement aid: a read-only HBM stream
// 16-byte streaming loads, four in flight per thread, grid-stride; the xor keeps the loads alive.  This is the
// ceiling a read-only kernel such as a4 can be held against (MEASURED_PEAKS.json's copy is a read+write stream).
__global__ void __launch_bounds__(512)
tangram_read_stream_kernel(const uint4* __restrict__ src, size_t n16, uint32_t* __restrict__ sink) {
    uint32_t acc = 0;
    size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const size_t stride = static_cast<size_t>(gridDim.x) * blockDim.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const uint4 a = __ldcs(src + i), b = __ldcs(src + i + stride), c = __ldcs(src + i + 2 * stride),
                    d = __ldcs(src + i + 3 * stride);
        acc ^= a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
    }
    for (; i < n16; i += stride) {
        const uint4 a = __ldcs(src + i);
        acc ^= a.x ^ a.y ^ a.z ^ a.w;
    }
    if (acc == 0x9e3779b9u) atomicAdd(sink, 1u);  // practically never; only keeps `acc` observable
}

// ------------------------------------------------------------------ host-side launch helpers
static int cuda_fail(cudaError_t e, const char* what) {
    return fail(TANGRAM_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            sym = nullptr;
        return reinterpret_cast<EncodeTiledFn>(sym);
    }();
    return fn;
}

// The pool [n_pages][Hp][2][P][d] bf16 seen as rows of d elements: dim0 = 64 elements (128 B, the
// swizzle span), dim1 = row, dim2 = which 64-element half of the row.  One box = the 2P rows (K then
// V) of one (page, slot).
static int make_kv_map(CUtensorMap* map, const void* pool, int64_t n_pool_pages, int Hp, int d, int kPage) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return fail(TANGRAM_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const cuuint64_t rows = static_cast<cuuint64_t>(n_pool_pages) * Hp * 2 * kPage;
    const cuuint64_t gdim[3] = {64, rows, static_cast<cuuint64_t>(d / 64)};
    const cuuint64_t gstride[2] = {static_cast<cuuint64_t>(d) * 2, 128};
    const cuuint32_t box[3] = {64, static_cast<cuuint32_t>(2 * kPage), static_cast<cuuint32_t>(d / 64)};
    const cuuint32_t estride[3] = {1, 1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(pool), gdim, gstride, box,
                           estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(TANGRAM_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return TANGRAM_OK;
}

// -1: TANGRAM_STEP_OVERLAP not tried yet; 1: the driver took the programmatic stream serialization attribute;
// 0: it refused (the flag is then ignored)
static int g_overlap_state = -1;

// CTAs of the decode kernel that can be co-resident on the current device (SMs x occupancy).
template <int D, bool TIMED, int NH, int PAGE>
static int max_coresident(int dev, int smem) {
    int sms = 0, per_sm = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tangram_decode_kernel<D, TIMED, NH, PAGE>, Smem<D, PAGE>::kThreads, smem) !=
        cudaSuccess)
        return 0;
    return sms * per_sm;
}

template <int D, bool TIMED, int NH, int PAGE>
static int launch_split(const tangram_device_plan* dp, DecodeParams prm, const CUtensorMap& map, cudaStream_t stream,
                        bool want_tail_merge, bool* merged) {
    using L = Smem<D, PAGE>;
    const int smem = L::total(prm.n_stages, prm.G, prm.n_qslots);
    cudaError_t e = cudaFuncSetAttribute(tangram_decode_kernel<D, TIMED, NH, PAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute");
    // The tail merge needs a grid barrier, i.e. a cooperative launch with every CTA resident.  The answer is
    // cached per (device, shared-memory size).
    static thread_local int cached_dev = -1, cached_smem = -1, cached_max = 0;
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    // the in-grid merge gives every thread one float4 of a record: it needs G * d/4 <= consumer threads (d = 256,
    // or d = 128 with G > 8, use the stand-alone merge kernel)
    const bool fits = D <= 128 && prm.G * (D / 4) <= L::kNW * 32;
    if (want_tail_merge && fits && (cached_smem != smem || cached_dev != dev))
        cached_max = max_coresident<D, TIMED, NH, PAGE>(dev, smem), cached_smem = smem, cached_dev = dev;
    // The CTAs of the tail phase wait for parts that other CTAs write, so the whole grid must be resident at once:
    // the in-grid merge is used only in a grid that fits on the device and is therefore launched cooperatively
    // (gang-scheduled).  A larger grid runs as a plain launch with no wait inside and is followed by the stand-alone
    // merge kernel (and, for a fused step, the length / table-growth kernel): the occupancy figure assumes a free
    // device, and with another plan's grid, any long kernel, MPS or an SM-limited context next to it the waiters of a
    // plain launch could hold every slot the not-yet-scheduled CTAs need.
    const bool coresident = cached_max > 0 && dp->n_static <= cached_max;
    prm.tail_merge = want_tail_merge && fits && coresident;
    prm.merge_ctas = dp->n_static;
    *merged = prm.tail_merge;
    if (prm.q_host && !prm.tail_merge) {
        // no co-resident grid, no in-kernel staging: the staging kernel runs first and the decode kernel is
        // launched behind it with programmatic stream serialization (it waits before its first query load)
        const int rc = tangram_stage_from_host(const_cast<__nv_bfloat16*>(prm.q), prm.q_host, (size_t)prm.R * prm.Hq * D * 2, stream);
        if (rc != TANGRAM_OK) return rc;
        prm.q_host = nullptr, prm.pdl = 1;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)dp->n_static), cfg.blockDim = dim3(L::kThreads), cfg.dynamicSmemBytes = smem, cfg.stream = stream;
    // Programmatic dependent launch: if the driver refuses the attribute once, it is not asked again (a failing
    // launch inside a stream capture would invalidate the capture).
    if (g_overlap_state == 0) prm.pdl = 0;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeCooperative;
    // A grid whose CTAs wait for one another (in-grid merge) is launched cooperatively whenever it fits on the device:
    // gang scheduling is what makes the waits safe next to OTHER grids -- in particular next to a programmatically
    // dependent successor, whose CTAs become resident while this grid still runs.  (A plain launch behind a
    // programmatic dependency was 1.8 us per layer-step faster in the graph loop and deadlocked about once in three
    // runs of the 200-step graph test: dependent CTAs took SMs that CTAs of this grid had not reached yet.)  A grid
    // larger than the device cannot be gang-scheduled: it runs as a plain launch without the tail phase (above).
    attr[0].val.cooperative = prm.tail_merge ? 1 : 0;
    prm.early_trigger = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr, cfg.numAttrs = prm.pdl ? 2 : 1;
    e = cudaLaunchKernelEx(&cfg, tangram_decode_kernel<D, TIMED, NH, PAGE>, map, prm);
    if (prm.pdl) {
        if (e == cudaSuccess) g_overlap_state = 1;
        else {
            (void)cudaGetLastError();
            g_overlap_state = 0, prm.pdl = 0, cfg.numAttrs = 1;  // the kernel then must not wait for a predecessor
            attr[0].val.cooperative = prm.tail_merge ? 1 : 0;
            e = cudaLaunchKernelEx(&cfg, tangram_decode_kernel<D, TIMED, NH, PAGE>, map, prm);
        }
    }
    if (e != cudaSuccess) return cuda_fail(e, "decode kernel launch");
    return TANGRAM_OK;
}

template <int D, int PAGE>
static int launch_decode(const tangram_device_plan* dp, DecodeParams prm, const CUtensorMap& map,
                         cudaStream_t stream, int which) {
    const int n_small = (int)(dp->n_merge_seqs - dp->n_big_merge_seqs);
    // Column blocks per row of a big record (a power of two <= D/4): more blocks = more part groups per record
    // (fewer dependent round trips: a CTA of 256 threads covers 8 * 256 * S / (D/4) parts of one block per round)
    // but also more units, i.e. more waves over the grid.  Cost model in units of one L2 round trip, measured on
    // B200: a unit costs ~2.5 (record, reduction tree, store) + its rounds.
    int S = 1;
    {
        const int64_t n_big = dp->n_big_merge_seqs, grid = std::max(1, dp->n_static);
        double best = 1e30;
        for (int cand = 1; cand <= D / 4 && n_big > 0; cand *= 2) {
            const int64_t waves = (n_big * prm.G * cand + grid - 1) / grid;
            const int64_t per_round = (int64_t)8 * 256 * cand / (D / 4);
            const int64_t rounds = (dp->max_merge_parts + per_round - 1) / per_round;
            const double cost = (double)waves * (2.5 + (double)rounds);
            if (cost < best) best = cost, S = cand;
        }
    }
    const int n_units = n_small + (int)dp->n_big_merge_seqs * prm.G * S;
    prm.merge_recs = dp->merge_seqs, prm.n_merge_small = n_small, prm.n_merge_units = n_units, prm.merge_split = S;
    const bool fused = prm.k_new != nullptr;
    bool merged = false;
    if (which & kRunSplit) {
        // a fused step always wants the tail phase (lengths + table growth), even with nothing to merge
        const bool want = (which & kRunMerge) && (n_units > 0 || fused || prm.q_host);
        int rc;
        if constexpr (D <= 128) {
            if (prm.G > 8)
                rc = prm.worker_ns ? launch_split<D, true, 2, PAGE>(dp, prm, map, stream, want, &merged)
                                   : launch_split<D, false, 2, PAGE>(dp, prm, map, stream, want, &merged);
            else
                rc = prm.worker_ns ? launch_split<D, true, 1, PAGE>(dp, prm, map, stream, want, &merged)
                                   : launch_split<D, false, 1, PAGE>(dp, prm, map, stream, want, &merged);
        } else {
            rc = prm.worker_ns ? launch_split<D, true, 1, PAGE>(dp, prm, map, stream, want, &merged)
                               : launch_split<D, false, 1, PAGE>(dp, prm, map, stream, want, &merged);
        }
        if (rc != TANGRAM_OK) return rc;
    }
    if (!(which & kRunMerge) || merged) return TANGRAM_OK;
    if (n_units > 0) {
        // Stand-alone merge kernel by programmatic dependent launch: its grid is scheduled while the decode
        // grid drains and blocks in griddepcontrol.wait until that grid has completed and flushed its writes.
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)n_units), cfg.blockDim = dim3(kMergeThreads), cfg.dynamicSmemBytes = 0, cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr, cfg.numAttrs = 1;
        const float* po = prm.part_o;
        const float* pl = prm.part_lse;
        cudaError_t e = cudaLaunchKernelEx(&cfg, tangram_merge_kernel<D>, dp->merge_seqs, n_small, po, pl, prm.out, prm.lse,
                                           (int)prm.G, S);
        if (e != cudaSuccess) return cuda_fail(e, "merge kernel launch");
    }
    if (fused) {  // lengths + table growth of a fused step whose grid could not run its tail phase
        tangram_grow_kernel<<<1, 1024, 0, stream>>>(prm.grow, PAGE, 1);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "grow kernel launch");
    }
    return TANGRAM_OK;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Largest GQA group: 16 query heads per KV head (both halves of the mma A operand) at d <= 128; at d = 256 the
// accumulators of 16 rows do not fit the register file, so 8.
static int max_gqa(int head_dim) { return head_dim == 256 ? 8 : kMaxG; }

template <int D, int PAGE>
static cudaError_t occupancy_of(int gqa, int* per_sm) {
    using L = Smem<D, PAGE>;
    const int ns = L::max_stages(gqa);
    const int smem = L::total(ns, gqa, L::max_qslots(ns, gqa));
    if (D <= 128 && gqa > 8) {
        if constexpr (D <= 128) {
            cudaError_t e = cudaFuncSetAttribute(tangram_decode_kernel<D, false, 2, PAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
            return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, tangram_decode_kernel<D, false, 2, PAGE>, L::kThreads, smem);
        }
    }
    cudaError_t e = cudaFuncSetAttribute(tangram_decode_kernel<D, false, 1, PAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, tangram_decode_kernel<D, false, 1, PAGE>, L::kThreads, smem);
}

}  // namespace tangram

using namespace tangram;

extern "C" int tangram_query_max_ctas(int device, int32_t head_dim, int32_t gqa, int32_t* n_cta_out) {
    if (!n_cta_out || (head_dim != 64 && head_dim != 128 && head_dim != 256) || gqa < 1 || gqa > max_gqa(head_dim))
        return fail(TANGRAM_ERR_INVALID_ARG, "query_max_ctas: head_dim=%d gqa=%d (GQA groups up to %d at this head_dim)",
                    head_dim, gqa, max_gqa(head_dim));
    int sms = 0, per_sm = 0;
    cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
    if (head_dim == 256) e = occupancy_of<256, 16>(gqa, &per_sm);
    else if (head_dim == 128) e = occupancy_of<128, 16>(gqa, &per_sm);
    else e = occupancy_of<64, 16>(gqa, &per_sm);
    if (e != cudaSuccess) return cuda_fail(e, "occupancy query");
    *n_cta_out = sms * per_sm;
    return TANGRAM_OK;
}

// Blob layout (all sections 256-byte aligned), shared by tangram_blob_bytes and tangram_upload.
namespace {
struct BlobLayout {
    size_t items, windptr, pindptr, pages, mseq, heads, seqinfo, row_ptr, row_pages, perm, seq_cap, cover, q_flags, seq_done, grow, sched, total;
};
int64_t table_slots(const tangram_tables* t) {
    return t->tbl_indptr ? t->tbl_indptr[(int64_t)t->R * t->C] : t->n_pages_used;
}
BlobLayout blob_layout(const tangram_tables* t, const tangram_plan* p) {
    BlobLayout b{};
    const size_t n_seq = (size_t)t->R * t->H, n_rows = (size_t)t->R * t->C;
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t at = off;
        off += align_up(bytes, 256);
        return at;
    };
    b.items = take(sizeof(DeviceItem) * (size_t)p->n_items);
    b.windptr = take(sizeof(int64_t) * ((size_t)p->W + 1));
    b.pindptr = take(sizeof(int64_t) * (n_seq + 1));
    b.pages = take(sizeof(int32_t) * (size_t)table_slots(t));
    b.mseq = take(4 * sizeof(int32_t) * n_seq);  // merge records (upper bound)
    b.heads = take(128 * (size_t)p->W);          // list heads
    b.seqinfo = take(16 * n_seq);                // per-sequence table info (KV append, compaction)
    b.row_ptr = take(sizeof(int32_t) * (n_rows + 1));
    b.row_pages = take(sizeof(int32_t) * n_rows);
    b.perm = take(sizeof(int32_t) * (size_t)t->H);
    b.seq_cap = take(sizeof(int32_t) * n_seq);
    b.cover = take(sizeof(int32_t) * n_seq);
    b.q_flags = take(sizeof(int32_t) * n_seq);
    b.seq_done = take(sizeof(uint32_t) * n_seq);
    b.grow = take(16);
    b.sched = take(32);
    b.total = off + 256;
    return b;
}
}  // namespace

extern "C" size_t tangram_blob_bytes(const tangram_tables* t, const tangram_plan* p) {
    if (!t || !p) return 0;
    return blob_layout(t, p).total;
}

extern "C" int tangram_upload(const tangram_tables* t, const tangram_plan* p, void* dev_blob, size_t bytes,
                              void* stream, tangram_device_plan* dp) {
    if (!t || !p || !dev_blob || !dp || !p->items || !p->worker_indptr || !p->part_indptr || !t->tbl_pages ||
        !t->tbl_indptr || !t->cluster_of || !t->slot_of || !t->perm)
        return fail(TANGRAM_ERR_INVALID_ARG, "upload: NULL argument");
    if (p->n_items > INT32_MAX) return fail(TANGRAM_ERR_INVALID_ARG, "upload: more than 2^31 items");
    if (t->P != 16 && t->P != 32) return fail(TANGRAM_ERR_INVALID_ARG, "upload: page size %d (kernels need 16 or 32)", t->P);
    const int kPage = t->P;
    const BlobLayout lay = blob_layout(t, p);
    const size_t need = lay.total;
    if (bytes < need) return fail(TANGRAM_ERR_BUFFER_TOO_SMALL, "upload: blob %zu < %zu bytes", bytes, need);
    if (reinterpret_cast<uintptr_t>(dev_blob) % 256 != 0)
        return fail(TANGRAM_ERR_INVALID_ARG, "upload: dev_blob must be 256-byte aligned");
    const int64_t n_seq = (int64_t)t->R * t->H, n_rows = (int64_t)t->R * t->C, n_slots = table_slots(t);
    if (n_slots > INT32_MAX) return fail(TANGRAM_ERR_INVALID_ARG, "upload: page table larger than 2^31 entries");
    std::vector<uint8_t> host(need, 0);
    DeviceItem* di = reinterpret_cast<DeviceItem*>(host.data() + lay.items);
    int32_t* cover = reinterpret_cast<int32_t*>(host.data() + lay.cover);
    for (int64_t i = 0; i < p->n_items; ++i) {
        const tangram_item& s = p->items[i];
        const int64_t row_off = t->tbl_indptr[(int64_t)s.req * t->C + s.cluster];
        di[i] = DeviceItem{s.req, s.kv_head, (int32_t)row_off, s.slot, s.tok_begin, s.tok_end, s.part_slot, s.n_parts};
        int32_t& cv = cover[(int64_t)s.req * t->H + s.kv_head];
        cv = std::max(cv, s.tok_end);
    }
    std::memcpy(host.data() + lay.windptr, p->worker_indptr, sizeof(int64_t) * ((size_t)p->W + 1));
    std::memcpy(host.data() + lay.pindptr, p->part_indptr, sizeof(int64_t) * ((size_t)n_seq + 1));
    std::memcpy(host.data() + lay.pages, t->tbl_pages, sizeof(int32_t) * (size_t)n_slots);
    int64_t max_page = -1;
    for (int64_t row = 0; row < n_rows; ++row) {
        const int64_t lo = t->tbl_indptr[row], hi = t->tbl_indptr[row + 1];
        const int64_t have = t->row_pages ? t->row_pages[row] : hi - lo;
        if (have < 0 || have > hi - lo) return fail(TANGRAM_ERR_INVALID_ARG, "upload: row_pages[%lld] out of range", (long long)row);
        for (int64_t i = lo; i < lo + have; ++i) {
            if (t->tbl_pages[i] < 0) return fail(TANGRAM_ERR_INVALID_ARG, "upload: negative page id in the tables");
            max_page = std::max<int64_t>(max_page, t->tbl_pages[i]);
        }
    }
    int32_t* mseq = reinterpret_cast<int32_t*>(host.data() + lay.mseq);
    int64_t n_mseq = 0;
    int64_t n_empty = 0;
    auto push = [&](int64_t sq) {  // record = {sequence, first part slot, parts, 0}
        int32_t* rec = mseq + 4 * n_mseq++;
        rec[0] = (int32_t)sq, rec[1] = (int32_t)p->part_indptr[sq];
        rec[2] = (int32_t)(p->part_indptr[sq + 1] - p->part_indptr[sq]), rec[3] = 0;
    };
    for (int64_t sq = 0; sq < n_seq; ++sq)  // empty sequences first ...
        if (p->part_indptr[sq + 1] - p->part_indptr[sq] == 0) push(sq);
    n_empty = n_mseq;
    for (int64_t sq = 0; sq < n_seq; ++sq) {  // ... then the small multi-part ones
        const int64_t np = p->part_indptr[sq + 1] - p->part_indptr[sq];
        if (np > 1 && np <= kMergeBigParts) push(sq);
    }
    const int64_t n_not_big = n_mseq;
    for (int64_t sq = 0; sq < n_seq; ++sq)  // ... then the big ones (one merge unit per query head)
        if (p->part_indptr[sq + 1] - p->part_indptr[sq] > kMergeBigParts) push(sq);
    int32_t n_dev_lists = 0;
    {   // list head = {item_begin, n_items, 0, 0, first item (8 words), its first 16 page ids, 0 x 4}.
        // The first n_static lists belong to the CTAs and are kept as they are; of the dynamic-tail lists only
        // the non-empty ones are uploaded (in plan order): claiming an empty list costs a CTA an atomic and a
        // dependent load for nothing, which is most of the tail on a small batch.  A slot without a page yet
        // (-1, growth headroom) stays -1 here and is read from the table at run time.
        int32_t* heads = reinterpret_cast<int32_t*>(host.data() + lay.heads);
        for (int32_t k = 0; k < p->W; ++k) {
            const int64_t ib = p->worker_indptr[k], ie = p->worker_indptr[k + 1];
            if (k >= p->n_static && ie == ib) continue;
            int32_t* hd = heads + 32 * n_dev_lists++;
            hd[0] = (int32_t)ib, hd[1] = (int32_t)(ie - ib);
            if (ie > ib) {
                std::memcpy(hd + 4, &di[ib], sizeof(DeviceItem));
                const DeviceItem& f = di[ib];
                const int64_t first_pg = (int64_t)f.tbl_row + f.tok_begin / kPage;
                const int64_t n_tiles = (f.tok_end - f.tok_begin + kPage - 1) / kPage;
                for (int64_t i = 0; i < 16 && i < n_tiles; ++i) hd[12 + i] = t->tbl_pages[first_pg + i];
            }
        }
    }
    {   // {first slot of the row, slot capacity in tokens, slot, row} and the tokens the row's pages hold
        int32_t* si = reinterpret_cast<int32_t*>(host.data() + lay.seqinfo);
        int32_t* cap = reinterpret_cast<int32_t*>(host.data() + lay.seq_cap);
        for (int32_t r = 0; r < t->R; ++r)
            for (int32_t h = 0; h < t->H; ++h, si += 4) {
                const int64_t row = (int64_t)r * t->C + t->cluster_of[h];
                const int64_t slots = t->tbl_indptr[row + 1] - t->tbl_indptr[row];
                si[0] = (int32_t)t->tbl_indptr[row];
                si[1] = (int32_t)(slots * t->P);
                si[2] = t->slot_of[h], si[3] = (int32_t)row;
                cap[(int64_t)r * t->H + h] = (int32_t)((t->row_pages ? t->row_pages[row] : slots) * t->P);
            }
    }
    {
        int32_t* rp = reinterpret_cast<int32_t*>(host.data() + lay.row_ptr);
        int32_t* rg = reinterpret_cast<int32_t*>(host.data() + lay.row_pages);
        for (int64_t row = 0; row <= n_rows; ++row) rp[row] = (int32_t)t->tbl_indptr[row];
        for (int64_t row = 0; row < n_rows; ++row)
            rg[row] = t->row_pages ? t->row_pages[row] : (int32_t)(t->tbl_indptr[row + 1] - t->tbl_indptr[row]);
        std::memcpy(host.data() + lay.perm, t->perm, sizeof(int32_t) * (size_t)t->H);
        int32_t* gs = reinterpret_cast<int32_t*>(host.data() + lay.grow);
        gs[0] = (int32_t)t->n_pages_used;  // the free list's cursor
    }
    // pageable source: the runtime stages it before returning, so `host` may die at scope exit
    cudaError_t e = cudaMemcpyAsync(dev_blob, host.data(), need, cudaMemcpyHostToDevice, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e, "upload: cudaMemcpyAsync");
    e = cudaStreamSynchronize(static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e, "upload: cudaStreamSynchronize");
    uint8_t* base = static_cast<uint8_t*>(dev_blob);
    dp->R = t->R, dp->H = t->H, dp->C = t->C, dp->Hp = t->Hp, dp->P = t->P, dp->W = n_dev_lists, dp->mode = p->mode;
    dp->n_static = p->n_static;
    dp->min_pool_pages = max_page + 1;
    dp->sched = reinterpret_cast<int32_t*>(base + lay.sched);
    dp->merge_seqs = reinterpret_cast<const int32_t*>(base + lay.mseq);
    dp->n_merge_seqs = n_mseq;
    dp->n_empty_seqs = n_empty;
    dp->list_heads = base + lay.heads;
    dp->seq_info = reinterpret_cast<const int32_t*>(base + lay.seqinfo);
    dp->n_big_merge_seqs = n_mseq - n_not_big;
    dp->max_merge_parts = 0;
    for (int64_t sq = 0; sq < n_seq; ++sq)
        dp->max_merge_parts = std::max<int64_t>(dp->max_merge_parts, p->part_indptr[sq + 1] - p->part_indptr[sq]);
    dp->n_items = p->n_items, dp->n_part_slots = p->n_part_slots;
    dp->items = base + lay.items;
    dp->worker_indptr = reinterpret_cast<const int64_t*>(base + lay.windptr);
    dp->part_indptr = reinterpret_cast<const int64_t*>(base + lay.pindptr);
    dp->tbl_pages = reinterpret_cast<const int32_t*>(base + lay.pages);
    dp->n_slots = n_slots;
    dp->row_ptr = reinterpret_cast<const int32_t*>(base + lay.row_ptr);
    dp->row_pages = reinterpret_cast<int32_t*>(base + lay.row_pages);
    dp->perm = reinterpret_cast<const int32_t*>(base + lay.perm);
    dp->seq_cap = reinterpret_cast<int32_t*>(base + lay.seq_cap);
    dp->plan_cover = reinterpret_cast<const int32_t*>(base + lay.cover);
    dp->grow_state = reinterpret_cast<int32_t*>(base + lay.grow);
    dp->q_flags = reinterpret_cast<int32_t*>(base + lay.q_flags);
    dp->seq_done = reinterpret_cast<uint32_t*>(base + lay.seq_done);
    return TANGRAM_OK;
}

extern "C" int tangram_overlap_state(void) { return g_overlap_state; }

extern "C" int tangram_reset_plan(const tangram_device_plan* dp, void* stream) {
    if (!dp || !dp->sched) return fail(TANGRAM_ERR_INVALID_ARG, "reset_plan: NULL argument");
    cudaError_t e = cudaMemsetAsync(dp->sched, 0, 32, static_cast<cudaStream_t>(stream));
    if (e == cudaSuccess && dp->q_flags)
        e = cudaMemsetAsync(dp->q_flags, 0, sizeof(int32_t) * (size_t)dp->R * dp->H, static_cast<cudaStream_t>(stream));
    if (e == cudaSuccess && dp->seq_done)
        e = cudaMemsetAsync(dp->seq_done, 0, sizeof(uint32_t) * (size_t)dp->R * dp->H, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e, "reset_plan: cudaMemsetAsync");
    return TANGRAM_OK;
}

extern "C" size_t tangram_workspace_bytes(int64_t n_part_slots, int32_t gqa, int32_t head_dim) {
    if (n_part_slots < 0 || gqa < 1 || head_dim < 1) return 0;
    return align_up((size_t)n_part_slots * gqa * head_dim * 4, 256) + align_up((size_t)n_part_slots * gqa * 4, 256) + 256;
}

static GrowParams grow_params(const tangram_device_plan* dp, int32_t* kv_len_dev, const int32_t* free_pages_dev,
                              int64_t n_free, int32_t* overflow_dev) {
    GrowParams g{};
    g.row_ptr = dp->row_ptr, g.row_pages = dp->row_pages, g.perm = dp->perm;
    g.tbl_pages = const_cast<int32_t*>(dp->tbl_pages), g.seq_cap = dp->seq_cap, g.plan_cover = dp->plan_cover;
    g.kv_len = kv_len_dev, g.grow_state = dp->grow_state, g.free_pages = free_pages_dev, g.overflow = overflow_dev;
    g.n_free = (int32_t)std::min<int64_t>(n_free, INT32_MAX), g.n_rows = dp->R * dp->C;
    g.R = dp->R, g.H = dp->H, g.C = dp->C, g.Hp = dp->Hp;
    g.n_pool_pages = INT32_MAX;  // the pool's size is not known here; tangram_decode_step fills it in
    return g;
}

// Arguments of a fused decode step beyond those of plain attention (all null / 0 for tangram_decode_attention).
struct StepArgs {
    const void* k_new = nullptr;
    const void* v_new = nullptr;
    int32_t* kv_len_w = nullptr;
    const int32_t* free_pages = nullptr;
    int64_t n_free = 0;
    int32_t* overflow = nullptr;
    uint32_t flags = 0;
    const void* q_host = nullptr;  // queries in pinned host memory, staged into q (device) by the kernel itself
};

static int run_attention(const tangram_device_plan* dp, const void* q, const void* kv_pool, int64_t n_pool_pages,
                         const int32_t* kv_len_dev, int32_t Hq, int32_t d, float sm_scale, void* out, float* lse, void* workspace,
                         size_t workspace_bytes, uint64_t* worker_ns, void* stream, int which, const StepArgs& step = StepArgs()) {
    const bool split = (which & kRunSplit) != 0;
    if (!dp || !out || !lse || (split && (!q || !kv_pool))) return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: NULL argument");
    if (d != 64 && d != 128 && d != 256)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: head_dim %d not in {64, 128, 256}", d);
    if (!page_supported(dp->P, d))
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: page size %d at head_dim %d (kernels need 16, or 32 at head_dim <= 128)",
                    dp->P, d);
    if (dp->H < 1 || Hq < 1 || Hq % dp->H != 0 || Hq / dp->H > max_gqa(d))
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: Hq=%d H=%d (need Hq %% H == 0 and Hq/H <= %d at head_dim %d)", Hq,
                    dp->H, max_gqa(d), d);
    if (dp->W < 1 || dp->n_static < 1 || dp->n_static > dp->W) return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: empty plan");
    if (split && n_pool_pages < 1) return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: empty pool");
    if (split && n_pool_pages < dp->min_pool_pages)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: kv_pool has %lld pages, the tables use page id %lld",
                    (long long)n_pool_pages, (long long)dp->min_pool_pages - 1);
    // q and kv_pool are read by the split kernel only: the merge-only entry point checks out / workspace alone
    if ((split && (reinterpret_cast<uintptr_t>(q) % 16 || reinterpret_cast<uintptr_t>(kv_pool) % 128)) ||
        reinterpret_cast<uintptr_t>(out) % 16 || reinterpret_cast<uintptr_t>(workspace) % 16)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: misaligned pointer");
    if (split) {
        // q is read with bulk asynchronous copies (cp.async.bulk), which must not be pointed at host memory: from
        // page-locked, device-mapped memory they complete most of the time and now and then never (measured on B200:
        // the launch hangs once in a few hundred to a few thousand calls).  Host-resident queries go through
        // tangram_decode_attention_host, which stages them with ordinary loads.
        cudaPointerAttributes at;
        const cudaError_t pe = cudaPointerGetAttributes(&at, q);
        if (pe != cudaSuccess) (void)cudaGetLastError();
        else if (at.type == cudaMemoryTypeHost)
            return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention: q is host memory (use tangram_decode_attention_host)");
    }
    const int G = Hq / dp->H;
    const size_t need = tangram_workspace_bytes(dp->n_part_slots, G, d);
    if (dp->n_part_slots > 0 && (!workspace || workspace_bytes < need))
        return fail(TANGRAM_ERR_BUFFER_TOO_SMALL, "decode_attention: workspace %zu < %zu bytes", workspace_bytes, need);

    CUtensorMap map;
    std::memset(&map, 0, sizeof map);
    if (split) {
        const int rc = make_kv_map(&map, kv_pool, n_pool_pages, dp->Hp, d, dp->P);
        if (rc != TANGRAM_OK) return rc;
    }

    DecodeParams prm{};
    prm.items = static_cast<const DeviceItem*>(dp->items);
    prm.worker_indptr = dp->worker_indptr;
    prm.tbl_pages = dp->tbl_pages;
    prm.q = static_cast<const __nv_bfloat16*>(q);
    prm.out = static_cast<__nv_bfloat16*>(out);
    prm.lse = lse;
    prm.part_o = static_cast<float*>(workspace);
    prm.part_lse = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) +
                                            align_up((size_t)dp->n_part_slots * G * d * 4, 256));
    prm.worker_ns = reinterpret_cast<unsigned long long*>(worker_ns);
    prm.tail_merge = 0, prm.merge_recs = nullptr, prm.n_merge_units = 0, prm.n_merge_small = 0, prm.merge_split = 1;
    prm.Hq = Hq, prm.G = G, prm.Hp = dp->Hp;
    prm.n_lists = dp->W;
    prm.list_heads = dp->list_heads;
    prm.sched = dp->sched;
    prm.seq_done = dp->seq_done;
    prm.kv_len = kv_len_dev, prm.H = dp->H, prm.R = dp->R;
    prm.q_host = static_cast<const uint4*>(step.q_host), prm.q_flags = dp->q_flags;
    if (step.k_new) {
        prm.k_new = static_cast<const uint4*>(step.k_new), prm.v_new = static_cast<const uint4*>(step.v_new);
        prm.pool_w = static_cast<uint4*>(const_cast<void*>(kv_pool));
        prm.n_pool_pages = (int32_t)std::min<int64_t>(n_pool_pages, INT32_MAX);
        prm.seq_cap = dp->seq_cap, prm.kv_len_w = step.kv_len_w;
        prm.grow = grow_params(dp, step.kv_len_w, step.free_pages, step.n_free, step.overflow);
        prm.grow.n_pool_pages = prm.n_pool_pages;
    }
    prm.pdl = (step.flags & TANGRAM_STEP_OVERLAP) ? 1 : 0;

    const float scale = sm_scale != 0.f ? sm_scale : 1.f / std::sqrt(static_cast<float>(d));
    prm.scale_log2 = scale * 1.4426950408889634f;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    auto go = [&](auto tag) {
        using L = decltype(tag);
        prm.n_stages = L::max_stages(G), prm.n_qslots = L::max_qslots(prm.n_stages, G);
        return 0;
    };
    if (dp->P == 32) {
        if (d == 128) return go(Smem<128, 32>()), launch_decode<128, 32>(dp, prm, map, st, which);
        return go(Smem<64, 32>()), launch_decode<64, 32>(dp, prm, map, st, which);
    }
    if (d == 256) return go(Smem<256, 16>()), launch_decode<256, 16>(dp, prm, map, st, which);
    if (d == 128) return go(Smem<128, 16>()), launch_decode<128, 16>(dp, prm, map, st, which);
    return go(Smem<64, 16>()), launch_decode<64, 16>(dp, prm, map, st, which);
}

extern "C" int tangram_decode_attention(const tangram_device_plan* dp, const void* q, const void* kv_pool,
                                        int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq, int32_t d, float sm_scale, void* out,
                                        float* lse, void* workspace, size_t workspace_bytes, uint64_t* worker_ns,
                                        void* stream) {
    return run_attention(dp, q, kv_pool, n_pool_pages, kv_len_dev, Hq, d, sm_scale, out, lse, workspace,
                         workspace_bytes, worker_ns, stream, kRunSplit | kRunMerge);
}

// ------------------------------------------------------------------ the call that allocates nothing
// Split-KV workspace for callers that cannot allocate one (include/tangram.h, tangram_decode_attention_static): a
// serving engine in its decode loop has given all free HBM to its page pool and must not call cudaMalloc there.
// The array is part of the module image: each GPU that loads the library holds these bytes until the process ends.
// It is shared by every call on the device and is never cleared (nothing in it needs to start at zero: a merge reads
// only partials that the same call wrote).
static __device__ __align__(256) unsigned char g_static_workspace[TANGRAM_STATIC_WORKSPACE_BYTES];

// Device address of g_static_workspace on the CURRENT device.  In host code the name `g_static_workspace` is only
// the host-side handle of the symbol, not an address a kernel may be given: the real address differs per device and
// comes from cudaGetSymbolAddress, asked once per device with that device current and then kept.
static int static_workspace_on_current_device(void** ptr_out) {
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static void* ptr_of[kMaxDevices] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "decode_attention_static: cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention_static: device ordinal %d (at most %d devices)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_workspace);
        if (e != cudaSuccess) return cuda_fail(e, "decode_attention_static: cudaGetSymbolAddress");
        if (!p || reinterpret_cast<uintptr_t>(p) % 256)
            return fail(TANGRAM_ERR_CUDA, "decode_attention_static: static workspace at %p on device %d", p, dev);
        ptr_of[dev] = p;
    }
    *ptr_out = ptr_of[dev];
    return TANGRAM_OK;
}

extern "C" int tangram_decode_attention_static(const tangram_device_plan* dp, const void* q, const void* kv_pool,
                                               int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq, int32_t d,
                                               float sm_scale, void* out, float* lse, uint64_t* worker_ns, void* stream) {
    if (!dp) return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention_static: NULL plan");
    if (dp->H < 1 || Hq < 1 || Hq % dp->H != 0 || d < 1)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention_static: Hq=%d H=%d d=%d", Hq, dp->H, d);
    // the limit first: a plan with more parts than the fixed array holds is refused before anything is launched
    const size_t need = tangram_workspace_bytes(dp->n_part_slots, Hq / dp->H, d);
    if (need > (size_t)TANGRAM_STATIC_WORKSPACE_BYTES)
        return fail(TANGRAM_ERR_BUFFER_TOO_SMALL,
                    "decode_attention_static: the plan's %lld part slots need %zu bytes, the static workspace holds %zu "
                    "(use tangram_decode_attention with a workspace of your own)",
                    (long long)dp->n_part_slots, need, (size_t)TANGRAM_STATIC_WORKSPACE_BYTES);
    void* ws = nullptr;
    const int rc = static_workspace_on_current_device(&ws);
    if (rc != TANGRAM_OK) return rc;
    return run_attention(dp, q, kv_pool, n_pool_pages, kv_len_dev, Hq, d, sm_scale, out, lse, ws,
                         (size_t)TANGRAM_STATIC_WORKSPACE_BYTES, worker_ns, stream, kRunSplit | kRunMerge);
}

extern "C" int tangram_decode_partials(const tangram_device_plan* dp, const void* q, const void* kv_pool,
                                       int64_t n_pool_pages, const int32_t* kv_len_dev, int32_t Hq, int32_t d, float sm_scale, void* out,
                                       float* lse, void* workspace, size_t workspace_bytes, uint64_t* worker_ns,
                                       void* stream) {
    return run_attention(dp, q, kv_pool, n_pool_pages, kv_len_dev, Hq, d, sm_scale, out, lse, workspace,
                         workspace_bytes, worker_ns, stream, kRunSplit);
}

extern "C" int tangram_merge_partials(const tangram_device_plan* dp, int32_t Hq, int32_t d, void* out, float* lse,
                                      void* workspace, size_t workspace_bytes, void* stream) {
    return run_attention(dp, nullptr, nullptr, 0, nullptr, Hq, d, 0.f, out, lse, workspace, workspace_bytes, nullptr, stream,
                         kRunMerge);
}

extern "C" int tangram_decode_step(const tangram_device_plan* dp, const void* q, const void* k_new, const void* v_new,
                                   void* kv_pool, int64_t n_pool_pages, int32_t* kv_len_dev, const int32_t* free_pages_dev,
                                   int64_t n_free, int32_t Hq, int32_t d, float sm_scale, void* out, float* lse,
                                   void* workspace, size_t workspace_bytes, int32_t* overflow_dev, uint32_t flags,
                                   uint64_t* worker_ns, void* stream) {
    if (!k_new || !v_new || !kv_len_dev) return fail(TANGRAM_ERR_INVALID_ARG, "decode_step: NULL argument");
    if (reinterpret_cast<uintptr_t>(k_new) % 16 || reinterpret_cast<uintptr_t>(v_new) % 16)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_step: misaligned pointer");
    if (n_free < 0 || (flags & ~TANGRAM_STEP_OVERLAP)) return fail(TANGRAM_ERR_INVALID_ARG, "decode_step: bad n_free / flags");
    StepArgs step;
    step.k_new = k_new, step.v_new = v_new, step.kv_len_w = kv_len_dev, step.free_pages = free_pages_dev;
    step.n_free = n_free, step.overflow = overflow_dev, step.flags = flags;
    return run_attention(dp, q, kv_pool, n_pool_pages, kv_len_dev, Hq, d, sm_scale, out, lse, workspace, workspace_bytes,
                         worker_ns, stream, kRunSplit | kRunMerge, step);
}

extern "C" int tangram_extend_tables_device(const tangram_device_plan* dp, const int32_t* kv_len_dev,
                                            const int32_t* free_pages_dev, int64_t n_free, void* stream) {
    if (!dp || !kv_len_dev || !free_pages_dev || n_free < 0)
        return fail(TANGRAM_ERR_INVALID_ARG, "extend_tables_device: NULL argument");
    const GrowParams g = grow_params(dp, const_cast<int32_t*>(kv_len_dev), free_pages_dev, n_free, nullptr);
    tangram_grow_kernel<<<1, 1024, 0, static_cast<cudaStream_t>(stream)>>>(g, dp->P, 0);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "grow kernel launch");
    return TANGRAM_OK;
}

extern "C" int tangram_sync_tables(const tangram_tables* t, const tangram_device_plan* dp, void* stream) {
    if (!t || !dp || !t->tbl_pages || !t->tbl_indptr || !t->cluster_of)
        return fail(TANGRAM_ERR_INVALID_ARG, "sync_tables: NULL argument");
    const int64_t n_rows = (int64_t)t->R * t->C, n_seq = (int64_t)t->R * t->H;
    if (t->R != dp->R || t->H != dp->H || t->C != dp->C || t->P != dp->P || table_slots(t) != dp->n_slots)
        return fail(TANGRAM_ERR_INVALID_ARG, "sync_tables: the tables do not have the shape of the uploaded ones");
    std::vector<int32_t> rows((size_t)n_rows), cap((size_t)n_seq);
    for (int64_t row = 0; row < n_rows; ++row) {
        rows[(size_t)row] = t->row_pages ? t->row_pages[row] : (int32_t)(t->tbl_indptr[row + 1] - t->tbl_indptr[row]);
    }
    for (int32_t r = 0; r < t->R; ++r)
        for (int32_t h = 0; h < t->H; ++h)
            cap[(size_t)r * t->H + h] = rows[(size_t)r * t->C + t->cluster_of[h]] * t->P;
    const int32_t gs[4] = {(int32_t)t->n_pages_used, 0, 0, 0};
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaMemcpyAsync(const_cast<int32_t*>(dp->tbl_pages), t->tbl_pages, sizeof(int32_t) * (size_t)dp->n_slots,
                                    cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dp->row_pages, rows.data(), sizeof(int32_t) * rows.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dp->seq_cap, cap.data(), sizeof(int32_t) * cap.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dp->grow_state, gs, 4, cudaMemcpyHostToDevice, st);  // cursor only
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);  // the sources are host temporaries
    if (e != cudaSuccess) return cuda_fail(e, "sync_tables");
    return TANGRAM_OK;
}

extern "C" int tangram_download_tables(const tangram_device_plan* dp, tangram_tables* t, int64_t* n_starved_out, void* stream) {
    if (!t || !dp || !t->tbl_pages || !t->row_pages)
        return fail(TANGRAM_ERR_INVALID_ARG, "download_tables: NULL argument (row_pages is required)");
    if (t->R != dp->R || t->C != dp->C || t->tbl_pages_cap < dp->n_slots)
        return fail(TANGRAM_ERR_INVALID_ARG, "download_tables: the host tables are smaller than the uploaded ones");
    int32_t gs[4] = {0, 0, 0, 0};
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaMemcpyAsync(t->tbl_pages, dp->tbl_pages, sizeof(int32_t) * (size_t)dp->n_slots, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(t->row_pages, dp->row_pages, sizeof(int32_t) * (size_t)dp->R * dp->C, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(gs, dp->grow_state, sizeof gs, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "download_tables");
    t->n_pages_used = gs[0];
    if (n_starved_out) *n_starved_out = gs[1];
    return TANGRAM_OK;
}

extern "C" int tangram_append_kv(const tangram_device_plan* dp, const void* k_new, const void* v_new, void* kv_pool,
                                 int64_t n_pool_pages, int32_t d, int32_t* kv_len_dev, int32_t* overflow_dev,
                                 void* stream) {
    if (!dp || !k_new || !v_new || !kv_pool || !kv_len_dev)
        return fail(TANGRAM_ERR_INVALID_ARG, "append_kv: NULL argument");
    if (d != 64 && d != 128 && d != 256)
        return fail(TANGRAM_ERR_INVALID_ARG, "append_kv: head_dim %d not in {64, 128, 256}", d);
    if (!page_supported(dp->P, d))
        return fail(TANGRAM_ERR_INVALID_ARG, "append_kv: page size %d at head_dim %d (kernels need 16, or 32 at head_dim <= 128)", dp->P, d);
    if (n_pool_pages < 1 || n_pool_pages < dp->min_pool_pages)
        return fail(TANGRAM_ERR_INVALID_ARG, "append_kv: kv_pool has %lld pages, the tables need %lld", (long long)n_pool_pages,
                    (long long)dp->min_pool_pages);
    if (reinterpret_cast<uintptr_t>(k_new) % 16 || reinterpret_cast<uintptr_t>(v_new) % 16 ||
        reinterpret_cast<uintptr_t>(kv_pool) % 16)
        return fail(TANGRAM_ERR_INVALID_ARG, "append_kv: misaligned pointer");
    const int n_seq = dp->R * dp->H;
    tangram_append_kernel<<<(n_seq + 3) / 4, 128, 0, static_cast<cudaStream_t>(stream)>>>(
        reinterpret_cast<const int4*>(dp->seq_info), dp->seq_cap, dp->tbl_pages, static_cast<const uint4*>(k_new),
        static_cast<const uint4*>(v_new), static_cast<uint4*>(kv_pool), kv_len_dev, overflow_dev, n_seq, dp->Hp, d, dp->P,
        (int)std::min<int64_t>(n_pool_pages, INT32_MAX));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "append kernel launch");
    return TANGRAM_OK;
}

extern "C" int tangram_read_stream(const void* src_dev, size_t bytes, uint32_t* sink_dev, void* stream) {
    if (!src_dev || !sink_dev || bytes % 16 || reinterpret_cast<uintptr_t>(src_dev) % 16)
        return fail(TANGRAM_ERR_INVALID_ARG, "read_stream: NULL / misaligned argument");
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e, "read_stream: device query");
    tangram_read_stream_kernel<<<sms * 16, 512, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<const uint4*>(src_dev),
                                                                                        bytes / 16, sink_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "read_stream launch");
    return TANGRAM_OK;
}

extern "C" int tangram_decode_attention_host(const tangram_device_plan* dp, const void* q_host, void* q_stage_dev,
                                             const void* kv_pool, int64_t n_pool_pages, const int32_t* kv_len_dev,
                                             int32_t Hq, int32_t d, float sm_scale, void* out, float* lse, void* workspace,
                                             size_t workspace_bytes, uint64_t* worker_ns, void* stream) {
    if (!dp || !q_host || !q_stage_dev || Hq < 1 || d < 1)
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention_host: NULL argument");
    if (reinterpret_cast<uintptr_t>(q_host) % 16) return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention_host: misaligned q_host");
    cudaPointerAttributes at;
    const cudaError_t e = cudaPointerGetAttributes(&at, q_host);
    if (e != cudaSuccess || (at.type != cudaMemoryTypeHost && at.type != cudaMemoryTypeManaged && at.type != cudaMemoryTypeDevice)) {
        (void)cudaGetLastError();
        return fail(TANGRAM_ERR_INVALID_ARG, "decode_attention_host: q_host is not page-locked (device-mapped) memory");
    }
    StepArgs step;
    step.q_host = q_host;
    return run_attention(dp, q_stage_dev, kv_pool, n_pool_pages, kv_len_dev, Hq, d, sm_scale, out, lse, workspace,
                         workspace_bytes, worker_ns, stream, kRunSplit | kRunMerge, step);
}

extern "C" int tangram_stage_from_host(void* dst_dev, const void* src_host, size_t bytes, void* stream) {
    if (!dst_dev || !src_host) return fail(TANGRAM_ERR_INVALID_ARG, "stage_from_host: NULL argument");
    if (bytes % 16 || reinterpret_cast<uintptr_t>(dst_dev) % 16 || reinterpret_cast<uintptr_t>(src_host) % 16)
        return fail(TANGRAM_ERR_INVALID_ARG, "stage_from_host: pointers and size must be multiples of 16 bytes");
    if (bytes == 0) return TANGRAM_OK;
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, src_host);
    if (e != cudaSuccess || (at.type != cudaMemoryTypeHost && at.type != cudaMemoryTypeManaged && at.type != cudaMemoryTypeDevice)) {
        (void)cudaGetLastError();
        return fail(TANGRAM_ERR_INVALID_ARG, "stage_from_host: the source is not page-locked (device-mapped) memory");
    }
    const size_t n16 = bytes / 16;
    const unsigned grid = static_cast<unsigned>(std::min<size_t>((n16 + 255) / 256, 592));
    tangram_stage_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<uint4*>(dst_dev),
                                                                            static_cast<const uint4*>(src_host), n16);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "stage kernel launch");
    return TANGRAM_OK;
}
