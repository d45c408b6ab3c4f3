// NEXT-2 of SURVEY.md §8(f): per-head Top-k selection (Eq. 4: I = Top(ceil(B N), s)) and
// compaction K~ = K[I,:], V~ = V[I,:] (Eq. 1) into the ragged pages (:190).  Contract:
// include/tangram.h (tangram_compact_topk).  Three launches on the caller's stream; the third is launched behind
// the second by programmatic dependent launch and the two OVERLAP: a row's gather starts when that row's select is
// done (per-row ready flags), so the issue-bound select hides behind the HBM-bound gather:
//
//   1. compact_prepare_kernel   one CTA: clamps keep[r][h] to [0, min(N_r, table capacity)] (the reserved
//      budget is a hard capacity bound, :176), counts the clamped heads, and scans ceil(keep / P) into a
//      tile index (tile = the P token slots of one (page, head)) in QUEUE order -- the order in which the select
//      kernel takes the rows and the gather kernel moves them; zeroes the counters and the rows' ready flags, and
//      decides from the batch whether the call is gather-heavy (select and gather then share every SM).
//   2. topk_select_kernel       one CTA (512 or 1024 threads, by row length) per (request, KV head): radix select
//      (digits of 11, 11 and 10 bits, shared-memory atomic histograms, 16-byte loads) over a monotone integer image
//      of the fp32 score finds the threshold key T and how many of the entries equal to T are kept (the lowest
//      token indices first, reading A30).  After the first digit the entries that share the threshold's digit are
//      usually few (<= 4096): one more pass over the row buffers them in shared memory, where the other two digits
//      are resolved; otherwise the kernel falls back to whole-row passes.  An ordered pass then writes the retained
//      token indices in ascending order: the entry at token i goes to position (#greater before i) +
//      min(#equal before i, need); every warp owns a contiguous segment, so that pass needs one block barrier in
//      total.  Integer work on fp32 bit patterns: the result is the unique Top-k under the tie rule, bit-exact
//      against the sort-based oracle.  A finished row is published with a release store to its ready flag.
//   3. compact_gather_kernel    persistent grid, warps claim chunks of tiles from a global counter (the same
//      run-time balancing as the decode kernel's dynamic tail: per-SM bandwidth differs on B200).  A warp
//      moves one tile: up to P K rows and P V rows of d bf16 each, gathered with 16-byte loads (16 in
//      flight per lane) and stored as two contiguous runs of the page.  HBM-bound: 4*d bytes read +
//      4*d bytes written per retained token-head.  Before the first tile of a row the warp waits for the row's
//      ready flag (acquire); the kernel's CTAs become resident as soon as every select CTA has started.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdlib>

#include "tangram.h"
#include "tangram_internal.h"

namespace tangram {

constexpr int kCPage = 16;           // rows of a gather tile (= one page at P = 16, half a page at P = 32)
constexpr int kSelBins = 2048;        // 11-bit digits
constexpr int kSelCand = 4096;        // candidates (entries in the first digit's bin) the select kernel buffers
constexpr int kSelLongRow = 49152;    // rows longer than this get 1024-thread CTAs, shorter ones 512 (two per SM)
constexpr int kGatherThreads = 256;
constexpr int kGatherChunk = 8;      // tiles claimed at once

constexpr int kMaxSms = 256;          // per-SM slots of the workspace (B200: 148 SMs)
// Cost model behind the gather-heavy decision (measured on B200, 8b shapes): the select kernel alone handles
// ~150 scores per ns on the whole device, the gather moves ~6400 bytes per ns.
constexpr long long kSelScoresPerNs = 150, kGatherBytesPerNs = 6400;

// Workspace (int32 words): [0] chunk counter of the gather, [1] total tiles, [2] row counter of the select,
// [3] 1 = gather-heavy call (one select CTA per SM stays, the others leave their registers to the gather), [4..7] pad;
// then keep_eff[n_seq], base[n_seq] (tokens every head held before the call), tile_indptr[n_seq + 1] (first tile of
// every QUEUE POSITION), order[n_seq] (the row at every queue position), ready[n_seq] (1 = the row's indices are
// written) and sm_first[kMaxSms] (select CTAs that arrived on every SM).
struct CompactWs {
    int32_t* counter;
    int32_t* keep_eff;
    int32_t* base;
    int32_t* tile_indptr;
    int32_t* order;
    int32_t* ready;
    int32_t* sm_first;
};
static __host__ __device__ inline size_t compact_ws_words(int64_t n_seq) { return 8 + 5 * (size_t)n_seq + 1 + kMaxSms; }

// fp32 score -> uint32 key with the same order (larger score = larger key); -0.0 and +0.0 compare equal
// as they do as fp32 values.
__device__ __forceinline__ uint32_t score_key(float x) {
    const uint32_t u = __float_as_uint(x + 0.0f);  // -0 + 0 = +0 (round to nearest); every other value is unchanged
    return u ^ (static_cast<uint32_t>(static_cast<int32_t>(u) >> 31) | 0x80000000u);
}

// overlap: 0 = never share the SMs (the select keeps all its CTAs), 1 = always, 2 = decide from the batch
__global__ void __launch_bounds__(1024)
compact_prepare_kernel(const int32_t* __restrict__ seq_cap, const int32_t* __restrict__ ctx_len,
                       const int32_t* __restrict__ keep, int32_t* __restrict__ kv_len, int n_seq, int H,
                       int32_t* __restrict__ counter, int32_t* __restrict__ keep_eff, int32_t* __restrict__ base,
                       int32_t* __restrict__ tile_indptr, int32_t* __restrict__ order, int32_t* __restrict__ ready,
                       int32_t* __restrict__ sm_first, int32_t* __restrict__ clamped, int row_bytes, int overlap) {
    __shared__ int s_warp[32];
    __shared__ int s_run, s_bad, s_heavy;
    asm volatile("griddepcontrol.launch_dependents;");  // the select grid may be set up while this CTA works
    __shared__ unsigned long long s_kept, s_scored;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_run = 0, s_bad = 0, s_kept = 0ull, s_scored = 0ull;
    for (int i = tid; i < kMaxSms; i += blockDim.x) sm_first[i] = 0;
    __syncthreads();
    // ---- per row: the clamped keep, where its rows go, the new length; batch totals for the cost model
    unsigned long long kept = 0ull, scored = 0ull;
    int bad = 0;
    for (int seq = tid; seq < n_seq; seq += blockDim.x) {
        const int want = keep[seq];
        const int have = kv_len ? kv_len[seq] : 0;  // chunked prefill: the rows go behind what the head holds
        const int N = ctx_len[seq / H];
        const int cap = min(N, seq_cap[seq] - have);  // seq_cap: tokens the pages of the head's row hold
        const int k = max(0, min(want, cap));
        bad += k != want;
        keep_eff[seq] = k;
        base[seq] = have;
        ready[seq] = 0;
        if (kv_len) kv_len[seq] = have + k;
        kept += static_cast<unsigned long long>(k);
        if (k > 0 && k < N) scored += static_cast<unsigned long long>(N);  // rows that need a selection
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        kept += __shfl_xor_sync(0xffffffffu, kept, o), scored += __shfl_xor_sync(0xffffffffu, scored, o);
        bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if (lane == 0) {
        if (kept) atomicAdd(&s_kept, kept);
        if (scored) atomicAdd(&s_scored, scored);
        if (bad) atomicAdd(&s_bad, bad);
    }
    __syncthreads();
    if (tid == 0) {
        // gather-heavy: the gather's estimated time is at least three times the select's.  Then one select CTA per SM
        // is enough (at half the threads and next to a gather CTA it takes ~2.2 x as long: 8b 37 -> 77 us, and still
        // ends long before the gather) and the gather gets the other half of the SM's registers from the start.
        const unsigned long long gather_ns = s_kept * static_cast<unsigned long long>(row_bytes) / kGatherBytesPerNs;
        const unsigned long long select_ns = s_scored / kSelScoresPerNs;
        s_heavy = overlap == 1 || (overlap == 2 && gather_ns >= 3 * select_ns);
    }
    __syncthreads();
    const bool heavy = s_heavy != 0;
    // ---- the queue: requests by context length, all H rows of a request together (ties: lower request first).
    // Gather-heavy: SHORTEST first, so that the first rows are ready after a few microseconds and the select's own
    // tail (the long rows) hides behind the gather.  Otherwise longest first: longest-processing-time-first over the
    // persistent select CTAs.
    const int R = n_seq / H;
    for (int r = tid; r < R; r += blockDim.x) {
        const int n = ctx_len[r];
        int rank = 0;
        for (int o = 0; o < R; ++o) {
            const int m = ctx_len[o];
            rank += (heavy ? m < n : m > n) || (m == n && o < r);
        }
        for (int h = 0; h < H; ++h) order[rank * H + h] = r * H + h;
    }
    __syncthreads();
    // ---- exclusive scan of the tiles over the queue positions
    for (int first = 0; first < n_seq; first += blockDim.x) {
        const int pos = first + tid;
        const int tiles = pos < n_seq ? (keep_eff[order[pos]] + kCPage - 1) / kCPage : 0;
        int incl = tiles;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        int before = s_run;
        for (int w = 0; w < warp; ++w) before += s_warp[w];
        if (pos < n_seq) tile_indptr[pos] = before + incl - tiles;
        __syncthreads();
        if (tid == blockDim.x - 1) s_run = before + incl;
        __syncthreads();
    }
    if (tid == 0) {
        tile_indptr[n_seq] = s_run;
        counter[0] = 0, counter[1] = s_run, counter[2] = 0, counter[3] = heavy ? 1 : 0;
        if (clamped && s_bad) atomicAdd(clamped, s_bad);
    }
}

// Calls fn(key) for the aligned 16-byte groups [v0, v1) of a score row, in no particular order, U loads in
// flight per thread.
template <int NT, int U, typename F>
__device__ __forceinline__ void for_each_key(const float4* __restrict__ sv, int v0, int v1, int tid, F&& fn) {
    int i = v0 + tid;
    for (; i + (U - 1) * NT < v1; i += U * NT) {
        float4 x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = __ldg(sv + i + u * NT);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            fn(score_key(x[u].x)), fn(score_key(x[u].y)), fn(score_key(x[u].z)), fn(score_key(x[u].w));
        }
    }
    for (; i < v1; i += NT) {
        const float4 x = __ldg(sv + i);
        fn(score_key(x.x)), fn(score_key(x.y)), fn(score_key(x.z)), fn(score_key(x.w));
    }
}

// The same for a whole score row s[0..N): <= 3 entries before the first 16-byte boundary, the aligned groups,
// <= 3 entries after the last one.
template <int NT, int U, typename F>
__device__ __forceinline__ void for_each_key_row(const float* __restrict__ s, int N, int tid, F&& fn) {
    const int head = min(N, static_cast<int>((4u - (static_cast<uint32_t>(reinterpret_cast<uintptr_t>(s)) >> 2)) & 3u));
    const int nvec = (N - head) >> 2;
    const int tail0 = head + 4 * nvec;
    if (tid < head) fn(score_key(__ldg(s + tid)));
    if (tid < N - tail0) fn(score_key(__ldg(s + tail0 + tid)));
    for_each_key<NT, U>(reinterpret_cast<const float4*>(s + head), 0, nvec, tid, fn);
}

// Block-wide radix select of the k-th largest key (1 <= k <= number of entries): digits of 11, 11 and 10 bits
// from the top, one shared-memory atomic histogram per digit.  radix_passes runs digits [pass_begin, pass_end):
// each_key(add) must call add(key) once for every entry (split among the NT threads in any way; entries whose
// higher digits do not match the prefix found so far are ignored).  State, the same in every thread: `prefix` /
// `mask` = the digits fixed so far, `krem` = rank still to be found among the entries that match them, `cand` =
// how many entries match.  After the last digit prefix is the threshold key T and krem = how many of the entries
// equal to T belong to the k largest.
struct RadixState {
    uint32_t prefix, mask, krem, cand;
};
template <int NT, typename EachKey>
__device__ __forceinline__ void radix_passes(EachKey&& each_key, int pass_begin, int pass_end, RadixState& st,
                                             uint32_t* s_hist, uint32_t* s_wsum, uint32_t* s_pick) {
    constexpr int kWarps = NT / 32;
    constexpr int kBpt = kSelBins / NT;  // adjacent bins a thread owns in the scan
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll 1
    for (int pass = pass_begin; pass < pass_end; ++pass) {
        const int shift = pass == 0 ? 21 : (pass == 1 ? 10 : 0);
        const uint32_t dmask = pass == 2 ? 1023u : 2047u;
        const uint32_t prefix = st.prefix, mask = st.mask, krem = st.krem;
        for (int b = tid; b < kSelBins; b += NT) s_hist[b] = 0u;
        __syncthreads();
        each_key([&](uint32_t key) {
            if ((key & mask) == prefix) atomicAdd(&s_hist[(key >> shift) & dmask], 1u);
        });
        __syncthreads();
        {   // thread owns bins kBpt tid ..; `gt` = entries in higher bins (block-wide suffix sum)
            uint32_t c[kBpt], mine = 0;
#pragma unroll
            for (int j = 0; j < kBpt; ++j) c[j] = s_hist[kBpt * tid + j], mine += c[j];
            uint32_t incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t v = __shfl_down_sync(0xffffffffu, incl, o);
                if (lane + o < 32) incl += v;
            }
            if (lane == 0) s_wsum[warp] = incl;
            __syncthreads();
            // entries in the warps after this one: a warp-wide suffix sum over the (<= 32) warp totals
            uint32_t after = lane < kWarps ? s_wsum[lane] : 0u;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t v = __shfl_down_sync(0xffffffffu, after, o);
                if (lane + o < 32) after += v;
            }
            const uint32_t warp_incl = __shfl_sync(0xffffffffu, after, warp);  // totals of warps warp .. kWarps-1
            uint32_t gt = incl - mine + (warp_incl - s_wsum[warp]);
#pragma unroll
            for (int j = kBpt - 1; j >= 0; --j) {
                if (gt < krem && krem <= gt + c[j]) {  // exactly one bin satisfies this
                    s_pick[0] = prefix | (static_cast<uint32_t>(kBpt * tid + j) << shift);
                    s_pick[1] = krem - gt;
                    s_pick[2] = c[j];
                }
                gt += c[j];
            }
        }
        __syncthreads();
        st.prefix = s_pick[0], st.krem = s_pick[1], st.cand = s_pick[2];
        st.mask = mask | (dmask << shift);
    }
}

// One (request, KV head) row by one CTA of NT threads.  (A thread-block cluster per row with the histograms
// exchanged through distributed shared memory was measured too: the remote loads and cluster barriers cost
// more than the extra SMs bring -- 8b 40 -> 46 us with 2 CTAs per row, 220 us with 8.)
template <int NT>
struct SelectSmem {
    uint32_t hist[kSelBins];
    uint32_t wsum[NT / 32];
    uint32_t pick[3];
    uint32_t cnt[2][NT / 32];                   // (greater, equal) counts of the warps' segments
    uint32_t ckey[kSelCand], cidx[kSelCand];    // candidates: entries in the first digit's bin
    uint32_t ncand;
    int row;                                    // the row the CTA claimed
};

template <int NT>
__device__ __forceinline__ void select_row(SelectSmem<NT>& sm, const int seq, const float* __restrict__ scores,
                                           int64_t n_max, const int32_t* __restrict__ ctx_len,
                                           const int32_t* __restrict__ keep_eff, int H, int32_t* __restrict__ idx_out) {
    constexpr int kSelWarps = NT / 32;
    constexpr int kU = NT == 1024 ? 4 : 8;  // 16-byte loads in flight per thread (register budget: 64 / 32)
    uint32_t* s_hist = sm.hist;
    uint32_t* s_wsum = sm.wsum;
    uint32_t* s_pick = sm.pick;
    uint32_t(*s_cnt)[kSelWarps] = sm.cnt;
    uint32_t* s_ckey = sm.ckey;
    uint32_t* s_cidx = sm.cidx;
    uint32_t& s_ncand = sm.ncand;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = ctx_len[seq / H];
    const int k = keep_eff[seq];
    if (k <= 0) return;
    const float* s = scores + static_cast<size_t>(seq) * n_max;
    int32_t* idx = idx_out + static_cast<size_t>(seq) * n_max;
    if (k >= N) {  // everything is retained
        for (int i = tid; i < N; i += NT) idx[i] = i;
        return;
    }
    // The row is <= 3 head entries, nvec aligned float4 groups, <= 3 tail entries.  Warp w owns the contiguous
    // groups [v0, v1) in the ordered parts below.
    const int head = min(N, static_cast<int>((4u - (static_cast<uint32_t>(reinterpret_cast<uintptr_t>(s)) >> 2)) & 3u));
    const int nvec = (N - head) >> 2;
    const int tail0 = head + 4 * nvec;
    const float4* sv = reinterpret_cast<const float4*>(s + head);
    const int wseg = ((nvec + kSelWarps - 1) / kSelWarps + 31) & ~31;
    const int v0 = min(nvec, warp * wseg), v1 = min(nvec, v0 + wseg);

    // ---- threshold: keep every key > T and the first `need` entries with key == T
    auto whole_row = [&](auto&& add) { for_each_key_row<NT, kU>(s, N, tid, add); };
    RadixState st{0u, 0u, static_cast<uint32_t>(k), static_cast<uint32_t>(N)};
    radix_passes<NT>(whole_row, 0, 1, st, s_hist, s_wsum, s_pick);  // first digit: one pass over the row (from HBM)
    const bool buffered = st.cand <= static_cast<uint32_t>(kSelCand);
    if (buffered) {
        // Usual case: few entries share the threshold's first digit.  ONE more pass over the row collects them
        // in shared memory and counts, per warp segment, the entries above that digit (certainly retained); the
        // remaining two digits and the (greater, equal) split of the candidates are then found in shared memory.
        // Three passes over the row in total (this one, the first digit, the placement) instead of five.
        if (tid == 0) s_ncand = 0u;
        __syncthreads();
        const uint32_t top = st.prefix >> 21;
        auto collect = [&](uint32_t key, int token) {
            if ((key >> 21) == top) {
                const uint32_t slot = atomicAdd(&s_ncand, 1u);
                s_ckey[slot] = key, s_cidx[slot] = static_cast<uint32_t>(token);
            }
        };
        if (tid < head) collect(score_key(__ldg(s + tid)), tid);
        if (tid < N - tail0) collect(score_key(__ldg(s + tail0 + tid)), tail0 + tid);
        uint32_t cg_ = 0;
        auto scan4 = [&](const float4 x, int v) {
            const uint32_t key[4] = {score_key(x.x), score_key(x.y), score_key(x.z), score_key(x.w)};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                cg_ += (key[j] >> 21) > top;
                collect(key[j], head + 4 * v + j);
            }
        };
        int v = v0 + lane;
        for (; v + 7 * 32 < v1; v += 8 * 32) {
            float4 x[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) x[u] = __ldg(sv + v + u * 32);
#pragma unroll
            for (int u = 0; u < 8; ++u) scan4(x[u], v + u * 32);
        }
        for (; v < v1; v += 32) scan4(__ldg(sv + v), v);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cg_ += __shfl_xor_sync(0xffffffffu, cg_, o);
        if (lane == 0) s_cnt[0][warp] = cg_, s_cnt[1][warp] = 0u;
        __syncthreads();
        const int n_cand = static_cast<int>(s_ncand);  // == st.cand
        radix_passes<NT>([&](auto&& add) { for (int i = tid; i < n_cand; i += NT) add(s_ckey[i]); }, 1, 3, st, s_hist,
                         s_wsum, s_pick);
        // candidates above / at the threshold, added to their warp segment's counts (head and tail entries are
        // placed separately below)
        for (int i = tid; i < n_cand; i += NT) {
            const int token = static_cast<int>(s_cidx[i]);
            if (token < head || token >= tail0) continue;
            const int w = ((token - head) >> 2) / wseg;
            if (s_ckey[i] > st.prefix) atomicAdd(&s_cnt[0][w], 1u);
            else if (s_ckey[i] == st.prefix) atomicAdd(&s_cnt[1][w], 1u);
        }
    } else {
        radix_passes<NT>(whole_row, 1, 3, st, s_hist, s_wsum, s_pick);
    }
    const uint32_t T = st.prefix, need = st.krem;

    // ---- ordered pass: position of token i = #greater before i + min(#equal before i, need).
    // Every warp needs the (greater, equal) counts of the segments before its own: from the buffered path above, or
    // by counting its groups (16-byte loads, 8 in flight); after the only block barrier of this part it walks its
    // groups 32 at a time: a lane holds four consecutive tokens and a packed (greater, equal) warp scan gives their
    // positions.
    auto cnt4 = [&](const float4 x, uint32_t& g, uint32_t& e) {
        const uint32_t a = score_key(x.x), b = score_key(x.y), c = score_key(x.z), d = score_key(x.w);
        g += (a > T) + (b > T) + (c > T) + (d > T);
        e += (a == T) + (b == T) + (c == T) + (d == T);
    };
    if (!buffered) {
        uint32_t cg_ = 0, ce_ = 0;
        int v = v0 + lane;
        for (; v + 7 * 32 < v1; v += 8 * 32) {
            float4 x[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) x[u] = __ldg(sv + v + u * 32);
#pragma unroll
            for (int u = 0; u < 8; ++u) cnt4(x[u], cg_, ce_);
        }
        for (; v < v1; v += 32) cnt4(__ldg(sv + v), cg_, ce_);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cg_ += __shfl_xor_sync(0xffffffffu, cg_, o), ce_ += __shfl_xor_sync(0xffffffffu, ce_, o);
        if (lane == 0) s_cnt[0][warp] = cg_, s_cnt[1][warp] = ce_;
    }
    __syncthreads();
    const uint32_t lt = (1u << lane) - 1u;
    // the head entries come first, the tail entries last; both are placed by warp 0 (lane j holds entry j)
    uint32_t run_gt = 0, run_eq = 0;
    {
        const bool in_head = lane < head;
        const uint32_t key = in_head ? score_key(__ldg(s + lane)) : 0u;
        const bool gt = in_head && key > T, eq = in_head && key == T;
        const unsigned bg = __ballot_sync(0xffffffffu, gt), be = __ballot_sync(0xffffffffu, eq);
        const uint32_t eq_before = __popc(be & lt);
        if (warp == 0 && (gt || (eq && eq_before < need))) idx[__popc(bg & lt) + min(eq_before, need)] = lane;
        run_gt = __popc(bg), run_eq = __popc(be);
    }
    uint32_t all_gt = run_gt, all_eq = run_eq;
    {   // lane w reads warp w's counts
        uint32_t ag_ = lane < kSelWarps ? s_cnt[0][lane] : 0u, ae_ = lane < kSelWarps ? s_cnt[1][lane] : 0u;
        uint32_t bg_ = lane < warp ? ag_ : 0u, be_ = lane < warp ? ae_ : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            bg_ += __shfl_xor_sync(0xffffffffu, bg_, o), be_ += __shfl_xor_sync(0xffffffffu, be_, o);
            ag_ += __shfl_xor_sync(0xffffffffu, ag_, o), ae_ += __shfl_xor_sync(0xffffffffu, ae_, o);
        }
        run_gt += bg_, run_eq += be_, all_gt += ag_, all_eq += ae_;
    }
    if (warp == 0) {
        const bool in_tail = lane < N - tail0;
        const uint32_t key = in_tail ? score_key(__ldg(s + tail0 + lane)) : 0u;
        const bool gt = in_tail && key > T, eq = in_tail && key == T;
        const unsigned bg = __ballot_sync(0xffffffffu, gt), be = __ballot_sync(0xffffffffu, eq);
        const uint32_t eq_before = all_eq + __popc(be & lt);
        if (gt || (eq && eq_before < need)) idx[all_gt + __popc(bg & lt) + min(eq_before, need)] = tail0 + lane;
    }
    auto place4 = [&](const float4 x, int v) {  // group v of the row: tokens head + 4 v .. + 3, lane-major order
        const uint32_t key[4] = {score_key(x.x), score_key(x.y), score_key(x.z), score_key(x.w)};
        uint32_t p = 0;
        if (v < v1) {
#pragma unroll
            for (int j = 0; j < 4; ++j) p += (key[j] > T) + ((key[j] == T) << 16);
        }
        if (!__any_sync(0xffffffffu, p != 0u)) return;  // nothing retained in these 128 tokens
        uint32_t incl = p;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const uint32_t tot = __shfl_sync(0xffffffffu, incl, 31);
        if (p) {
            // the lane's retained tokens take consecutive positions from (#greater before) + min(#equal before, need)
            uint32_t e = run_eq + ((incl - p) >> 16);
            uint32_t pos = run_gt + ((incl - p) & 0xffffu) + min(e, need);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const bool eq = key[j] == T;
                const bool keep = key[j] > T || (eq && e < need);
                if (keep) idx[pos] = head + 4 * v + j;
                pos += keep, e += eq;
            }
        }
        run_gt += tot & 0xffffu, run_eq += tot >> 16;
    };
    int v = v0;  // warp-uniform: rows of 32 groups
    for (; v + 3 * 32 < v1; v += 4 * 32) {
        float4 x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) x[u] = v + u * 32 + lane < v1 ? __ldg(sv + v + u * 32 + lane) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int u = 0; u < 4; ++u) place4(x[u], v + u * 32 + lane);
    }
    for (; v < v1; v += 32) place4(v + lane < v1 ? __ldg(sv + v + lane) : make_float4(0.f, 0.f, 0.f, 0.f), v + lane);
}

// Persistent grid: every CTA claims rows from the queue `order` until it is empty.  The select is bound by
// instruction issue and latency per row, not by bandwidth, so what matters is that no SM ends up with two long rows
// while another holds two short ones (round 1: one CTA per row in launch order, SM busy cycles min / avg / max =
// 5.7 K / 45 K / 63 K on 8b).  The gather kernel is launched behind this one programmatically: its CTAs may become
// resident once every CTA here has started, and they wait row by row for `ready`.  On a gather-heavy call
// (counter[3], two 512-thread CTAs per SM launched) only the first CTA to arrive on an SM stays: the other leaves
// its half of the register file to a gather CTA.
template <int NT>
__global__ void __launch_bounds__(NT, 1024 / NT)
topk_select_kernel(const float* __restrict__ scores, int64_t n_max, const int32_t* __restrict__ ctx_len,
                   const int32_t* __restrict__ keep_eff, int H, int n_seq, const int32_t* __restrict__ order,
                   int32_t* __restrict__ counter, int32_t* __restrict__ ready, int32_t* __restrict__ sm_first,
                   int32_t* __restrict__ idx_out) {
    __shared__ SelectSmem<NT> sm;
    // launched behind the prepare kernel programmatically: wait for its results, then let the gather in
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");
    if (NT < 1024 && __ldcg(counter + 3)) {
        if (threadIdx.x == 0) {
            unsigned smid;
            asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            sm.row = atomicAdd(sm_first + (smid % kMaxSms), 1);
        }
        __syncthreads();
        if (sm.row > 0) return;
    }
    int done = -1;  // the row whose indices this CTA wrote last
    for (;;) {
        __syncthreads();  // the previous row is done with the shared state, and all its indices are written
        if (threadIdx.x == 0) {
            if (done >= 0) {
                __threadfence();
                asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(ready + done), "r"(1) : "memory");
            }
            sm.row = atomicAdd(counter + 2, 1);
        }
        __syncthreads();
        const int slot = sm.row;
        if (slot >= n_seq) return;
        done = order[slot];
        select_row<NT>(sm, done, scores, n_max, ctx_len, keep_eff, H, idx_out);
    }
}

// NEXT-4: implicit per-head retention ratios of the global flat Top-k (Eq. 3; what Budget
// Calibration records on every sample, :156).  One CTA per request: radix select over the flattened scores of
// all H heads (head-major; ties to the lower flat index), then per-head counts of the entries above the
// threshold; the entries equal to it are granted in head order until `need` of them are taken.
template <int NT>
__global__ void __launch_bounds__(NT, 1024 / NT)
implicit_ratio_kernel(const float* __restrict__ scores, int64_t n_max, const int32_t* __restrict__ ctx_len, int H,
                      double rho, int32_t* __restrict__ counts_out, double* __restrict__ ratios_out) {
    constexpr int kU = NT == 1024 ? 4 : 8;
    extern __shared__ uint32_t s_ge[];  // [2][H]: entries greater than / equal to the threshold, per head
    __shared__ uint32_t s_hist[kSelBins];
    __shared__ uint32_t s_wsum[NT / 32];
    __shared__ uint32_t s_pick[3];
    const int r = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const int N = ctx_len[r];
    const float* s = scores + static_cast<size_t>(r) * H * n_max;
    const double total_f = static_cast<double>(static_cast<int64_t>(H) * N);
    const double want = ceil(rho * total_f);  // Eq. 3: ceil(rho H N)
    const uint32_t total = static_cast<uint32_t>(H) * static_cast<uint32_t>(N);
    const uint32_t k = want <= 0.0 ? 0u : (want >= total_f ? total : static_cast<uint32_t>(want));
    if (k == 0u || k == total) {
        for (int h = tid; h < H; h += NT) {
            counts_out[r * H + h] = k ? N : 0;
            ratios_out[r * H + h] = k ? 1.0 : 0.0;
        }
        return;
    }
    RadixState st{0u, 0u, k, total};
    radix_passes<NT>(
        [&](auto&& add) {
            for (int h = 0; h < H; ++h) for_each_key_row<NT, kU>(s + static_cast<size_t>(h) * n_max, N, tid, add);
        },
        0, 3, st, s_hist, s_wsum, s_pick);
    const uint32_t T = st.prefix, need = st.krem;
    for (int h = tid; h < 2 * H; h += NT) s_ge[h] = 0u;
    __syncthreads();
    for (int h = 0; h < H; ++h) {
        uint32_t g = 0, e = 0;
        for_each_key_row<NT, kU>(s + static_cast<size_t>(h) * n_max, N, tid, [&](uint32_t key) { g += key > T, e += key == T; });
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) g += __shfl_xor_sync(0xffffffffu, g, o), e += __shfl_xor_sync(0xffffffffu, e, o);
        if (lane == 0) {
            if (g) atomicAdd(&s_ge[h], g);
            if (e) atomicAdd(&s_ge[H + h], e);
        }
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t left = need;
        for (int h = 0; h < H; ++h) {
            const uint32_t take = min(s_ge[H + h], left);
            left -= take;
            const uint32_t c = s_ge[h] + take;
            counts_out[r * H + h] = static_cast<int32_t>(c);
            ratios_out[r * H + h] = static_cast<double>(c) / static_cast<double>(N);
        }
    }
}

template <int D>
__global__ void __launch_bounds__(kGatherThreads, 2)
compact_gather_kernel(const int4* __restrict__ seq_info, const int32_t* __restrict__ tbl_pages,
                      const int32_t* __restrict__ idx, int64_t n_max, const uint4* __restrict__ k_dense,
                      const uint4* __restrict__ v_dense, uint4* __restrict__ pool, int Hp, int n_seq,
                      int32_t* __restrict__ counter, const int32_t* __restrict__ keep_eff,
                      const int32_t* __restrict__ base, const int32_t* __restrict__ tile_indptr,
                      const int32_t* __restrict__ order, const int32_t* __restrict__ ready, int P) {
    constexpr int kChunks = D / 8;           // 16-byte chunks per row
    constexpr int kRowsPerLd = 32 / kChunks;  // rows one warp-wide load covers
    constexpr int kLds = kCPage / kRowsPerLd; // loads per lane for the K rows of a tile (same for V)
    constexpr int kPasses = D == 256 ? 2 : 1;
    constexpr int kLdsP = kLds / kPasses;
    const int lane = threadIdx.x & 31;
    const int sub = lane / kChunks, ch = lane % kChunks;
    const int total = __ldg(counter + 1);
    // The select kernel may still be running: a row's indices are read only after its ready flag (acquire by lane 0,
    // then a warp barrier) and through L2 (ld.cg), never through the non-coherent path.
    auto wait_row = [&](int seq) {
        if (lane == 0) {
            int seen;
            TANGRAM_SPIN_INIT;
            do {
                asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(ready + seq) : "memory");
                TANGRAM_SPIN_POLL(TANGRAM_WAIT_ROW_READY, seq);
            } while (seen == 0);
        }
        __syncwarp();
    };
    for (;;) {
        int first = 0;
        if (lane == 0) first = atomicAdd(counter, kGatherChunk);
        first = __shfl_sync(0xffffffffu, first, 0);
        if (first >= total) break;
        const int last = min(first + kGatherChunk, total);
        // queue position of the chunk's first tile: largest pos with tile_indptr[pos] <= first
        int lo = 0, hi = n_seq;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(tile_indptr + mid) <= first) lo = mid;
            else hi = mid;
        }
        int pos = lo;
        int pos_end = __ldg(tile_indptr + pos + 1);
        int seq = -1;
        for (int tile = first; tile < last; ++tile) {
            while (tile >= pos_end) ++pos, pos_end = __ldg(tile_indptr + pos + 1), seq = -1;  // skips heads that keep nothing
            if (seq < 0) seq = __ldg(order + pos), wait_row(seq);
            const int tl = tile - __ldg(tile_indptr + pos);  // tile inside the sequence: its retained rows 16 tl ..
            const int4 si = __ldg(seq_info + seq);           // {table row offset, capacity tokens, slot, -}
            const int n_rows = min(kCPage, __ldg(keep_eff + seq) - tl * kCPage);
            // lane j < n_rows: source token of the tile's row j and where it goes -- token slot base + 16 tl + j
            // of the head (with base = 0 the tile is exactly one page; behind an earlier chunk it straddles two)
            int my_tok = 0;
            uint32_t my_dst = 0;  // row index in the pool (rows of d elements): < 2^32 for pools up to 550 GB
            if (lane < n_rows) {
                my_tok = __ldcg(idx + static_cast<size_t>(seq) * n_max + tl * kCPage + lane);
                const int slot = __ldg(base + seq) + tl * kCPage + lane;
                const int page = __ldg(tbl_pages + si.x + slot / P);
                // pool[page][slot][kv][token][d]: row index of the K row; the V row is P rows further
                my_dst = ((static_cast<uint32_t>(page) * Hp + si.z) * 2) * P + slot % P;
            }
            // (at d = 256 a tile goes in two halves of eight rows: 16 + 16 loads would not fit the register budget)
#pragma unroll
            for (int half = 0; half < kPasses; ++half) {
                uint4 kreg[kLdsP], vreg[kLdsP];
#pragma unroll
                for (int j = 0; j < kLdsP; ++j) {
                    const int row = (half * kLdsP + j) * kRowsPerLd + sub;
                    const int tok = __shfl_sync(0xffffffffu, my_tok, row);
                    if (row < n_rows) {
                        const size_t src = (static_cast<size_t>(seq) * n_max + tok) * kChunks + ch;
                        kreg[j] = __ldcs(k_dense + src);
                        vreg[j] = __ldcs(v_dense + src);
                    }
                }
#pragma unroll
                for (int j = 0; j < kLdsP; ++j) {
                    const int row = (half * kLdsP + j) * kRowsPerLd + sub;
                    const uint32_t dst = __shfl_sync(0xffffffffu, my_dst, row);
                    if (row < n_rows) {
                        pool[static_cast<size_t>(dst) * kChunks + ch] = kreg[j];
                        pool[static_cast<size_t>(dst + P) * kChunks + ch] = vreg[j];
                    }
                }
            }
        }
    }
    // the grid ends after the select grid: whatever follows on the stream sees both complete
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

static int cuda_fail2(cudaError_t e, const char* what) {
    return fail(TANGRAM_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

}  // namespace tangram

using namespace tangram;

extern "C" size_t tangram_compact_workspace_bytes(int32_t R, int32_t H) {
    if (R < 1 || H < 1) return 0;
    return (compact_ws_words((int64_t)R * H) * 4 + 255) / 256 * 256;
}

static int compact_impl(const tangram_device_plan* dp, const float* scores, const void* k_dense, const void* v_dense,
                        int64_t n_max, const int32_t* ctx_len_dev, const int32_t* keep_dev, int32_t* kv_len_dev,
                        void* kv_pool, int64_t n_pool_pages, int32_t d, int32_t* idx_out, int32_t* clamped_dev,
                        void* workspace, size_t workspace_bytes, void* stream) {
    if (!dp || !scores || !k_dense || !v_dense || !ctx_len_dev || !keep_dev || !kv_pool || !idx_out || !workspace)
        return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk: NULL argument");
    if (d != 64 && d != 128 && d != 256)
        return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk: head_dim %d not in {64, 128, 256}", d);
    if (dp->P != 16 && !(dp->P == 32 && d <= 128))
        return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk: page size %d at head_dim %d (kernels need 16, or 32 at head_dim <= 128)", dp->P, d);
    if (n_max < 1 || n_max > (1 << 30) || n_pool_pages < 1 || n_pool_pages < dp->min_pool_pages)
        return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk: n_max=%lld n_pool_pages=%lld", (long long)n_max,
                    (long long)n_pool_pages);
    if (reinterpret_cast<uintptr_t>(k_dense) % 16 || reinterpret_cast<uintptr_t>(v_dense) % 16 ||
        reinterpret_cast<uintptr_t>(kv_pool) % 16 || reinterpret_cast<uintptr_t>(workspace) % 16)
        return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk: misaligned pointer");
    const int64_t n_seq64 = (int64_t)dp->R * dp->H;
    if (n_seq64 < 1 || n_seq64 > (1 << 24)) return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk: R*H=%lld", (long long)n_seq64);
    const int n_seq = (int)n_seq64;
    const size_t need = tangram_compact_workspace_bytes(dp->R, dp->H);
    if (workspace_bytes < need)
        return fail(TANGRAM_ERR_BUFFER_TOO_SMALL, "compact_topk: workspace %zu < %zu bytes", workspace_bytes, need);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int32_t* ws = static_cast<int32_t*>(workspace);
    CompactWs w{ws, ws + 8, ws + 8 + n_seq, ws + 8 + 2 * n_seq, ws + 8 + 3 * n_seq + 1, ws + 8 + 4 * n_seq + 1,
                ws + 8 + 5 * n_seq + 1};
    const int4* seq_info = reinterpret_cast<const int4*>(dp->seq_info);
    static thread_local int sms_dev = -1, sms = 0;
    int dev = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return cuda_fail2(e, "cudaGetDevice");
    if (dev != sms_dev) {
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
            return cuda_fail2(e, "cudaDeviceGetAttribute");
        sms_dev = dev;
    }
    // Select grid: rows of ordinary length get two 512-thread CTAs per SM (and, on a gather-heavy call, give one of
    // them up to the gather: the decision is the prepare kernel's, from the batch).  Very long rows get one
    // 1024-thread CTA per SM: a row then has a whole SM, and the gather follows as the select CTAs leave.
    // TANGRAM_COMPACT_OVERLAP = 0 / 1 forces the decision (measurement aid); default: decide from the batch.
    const bool wide = n_max > kSelLongRow;
    const char* ov = getenv("TANGRAM_COMPACT_OVERLAP");
    const int overlap_env = ov && (ov[0] == '0' || ov[0] == '1') && !ov[1] ? ov[0] - '0' : 2;
    compact_prepare_kernel<<<1, 1024, 0, st>>>(dp->seq_cap, ctx_len_dev, keep_dev, kv_len_dev, n_seq, dp->H, w.counter,
                                               w.keep_eff, w.base, w.tile_indptr, w.order, w.ready, w.sm_first, clamped_dev,
                                               8 * d, wide ? 0 : overlap_env);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail2(e, "compact prepare launch");
    static int pdl_state = -1;  // programmatic stream serialization: -1 not tried, 1 accepted, 0 refused
    {
        cudaLaunchConfig_t cfg{};
        cfg.blockDim = dim3(wide ? 1024 : 512), cfg.gridDim = dim3((unsigned)(wide ? std::min(n_seq, sms) : std::min(n_seq, 2 * sms)));
        cfg.dynamicSmemBytes = 0, cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        const int64_t n_max_ = n_max;
        const int H_ = dp->H;
        const int32_t* keep_c = w.keep_eff;
        const int32_t* order_c = w.order;
        auto go = [&]() {
            return wide ? cudaLaunchKernelEx(&cfg, topk_select_kernel<1024>, scores, n_max_, ctx_len_dev, keep_c, H_, n_seq, order_c,
                                             w.counter, w.ready, w.sm_first, idx_out)
                        : cudaLaunchKernelEx(&cfg, topk_select_kernel<512>, scores, n_max_, ctx_len_dev, keep_c, H_, n_seq, order_c,
                                             w.counter, w.ready, w.sm_first, idx_out);
        };
        cfg.numAttrs = pdl_state != 0 ? 1 : 0;
        e = go();
        if (cfg.numAttrs == 1) {
            if (e == cudaSuccess) pdl_state = 1;
            else {
                (void)cudaGetLastError();
                pdl_state = 0, cfg.numAttrs = 0;
                e = go();
            }
        }
    }
    if (e != cudaSuccess) return cuda_fail2(e, "top-k select launch");
    const uint4* kd = static_cast<const uint4*>(k_dense);
    const uint4* vd = static_cast<const uint4*>(v_dense);
    uint4* pool = static_cast<uint4*>(kv_pool);
    // The gather is launched behind the select with programmatic stream serialization and never waits for the whole
    // select grid, only for the rows it is about to move.  If the driver refuses the attribute once it is not asked
    // again (a failing launch inside a stream capture would invalidate the capture); a plain launch is correct too.
    auto gather = [&](auto kernel, int& grid) -> cudaError_t {
        if (grid == 0) {  // persistent grid: SMs x resident CTAs
            int per_sm = 0;
            const cudaError_t e2 = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kGatherThreads, 0);
            if (e2 != cudaSuccess) return e2;
            grid = sms * (per_sm > 0 ? per_sm : 1);
        }
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)grid), cfg.blockDim = dim3(kGatherThreads), cfg.dynamicSmemBytes = 0, cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr, cfg.numAttrs = pdl_state != 0 ? 1 : 0;
        const int64_t n_max_ = n_max;
        const int Hp = dp->Hp, P = dp->P;
        const int32_t* tbl = dp->tbl_pages;
        const int32_t* idx_c = idx_out;
        cudaError_t e2 = cudaLaunchKernelEx(&cfg, kernel, seq_info, tbl, idx_c, n_max_, kd, vd, pool, Hp, n_seq, w.counter,
                                            (const int32_t*)w.keep_eff, (const int32_t*)w.base, (const int32_t*)w.tile_indptr,
                                            (const int32_t*)w.order, (const int32_t*)w.ready, P);
        if (cfg.numAttrs == 1) {
            if (e2 == cudaSuccess) pdl_state = 1;
            else {
                (void)cudaGetLastError();
                pdl_state = 0, cfg.numAttrs = 0;
                e2 = cudaLaunchKernelEx(&cfg, kernel, seq_info, tbl, idx_c, n_max_, kd, vd, pool, Hp, n_seq, w.counter,
                                        (const int32_t*)w.keep_eff, (const int32_t*)w.base, (const int32_t*)w.tile_indptr,
                                        (const int32_t*)w.order, (const int32_t*)w.ready, P);
            }
        }
        return e2;
    };
    static thread_local int grid_dev = -1, grid256 = 0, grid128 = 0, grid64 = 0;  // cached per (thread, device)
    if (grid_dev != dev) grid_dev = dev, grid256 = grid128 = grid64 = 0;
    if (d == 256) e = gather(compact_gather_kernel<256>, grid256);
    else if (d == 128) e = gather(compact_gather_kernel<128>, grid128);
    else e = gather(compact_gather_kernel<64>, grid64);
    if (e != cudaSuccess) return cuda_fail2(e, "compact gather launch");
    return TANGRAM_OK;
}

extern "C" int tangram_implicit_ratios(const float* scores, int32_t R, int32_t H, int64_t n_max,
                                       const int32_t* ctx_len_dev, double rho, int32_t* counts_out,
                                       double* ratios_out, void* stream) {
    if (!scores || !ctx_len_dev || !counts_out || !ratios_out)
        return fail(TANGRAM_ERR_INVALID_ARG, "implicit_ratios: NULL argument");
    if (R < 1 || H < 1 || H > 4096 || n_max < 1 || (int64_t)H * n_max > INT32_MAX)
        return fail(TANGRAM_ERR_INVALID_ARG, "implicit_ratios: R=%d H=%d n_max=%lld (H * n_max must fit 31 bits)", R, H,
                    (long long)n_max);
    if (!(rho >= 0.0 && rho <= 1.0)) return fail(TANGRAM_ERR_INVALID_ARG, "implicit_ratios: rho=%g not in [0, 1]", rho);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t smem = 2 * sizeof(uint32_t) * (size_t)H;
    if ((int64_t)H * n_max > kSelLongRow)
        implicit_ratio_kernel<1024><<<R, 1024, smem, st>>>(scores, n_max, ctx_len_dev, H, rho, counts_out, ratios_out);
    else
        implicit_ratio_kernel<512><<<R, 512, smem, st>>>(scores, n_max, ctx_len_dev, H, rho, counts_out, ratios_out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail2(e, "implicit ratio launch");
    return TANGRAM_OK;
}

extern "C" int tangram_compact_topk(const tangram_device_plan* dp, const float* scores, const void* k_dense,
                                    const void* v_dense, int64_t n_max, const int32_t* ctx_len_dev,
                                    const int32_t* keep_dev, void* kv_pool, int64_t n_pool_pages, int32_t d,
                                    int32_t* idx_out, int32_t* clamped_dev, void* workspace, size_t workspace_bytes,
                                    void* stream) {
    return compact_impl(dp, scores, k_dense, v_dense, n_max, ctx_len_dev, keep_dev, nullptr, kv_pool, n_pool_pages, d,
                        idx_out, clamped_dev, workspace, workspace_bytes, stream);
}

extern "C" int tangram_compact_topk_chunk(const tangram_device_plan* dp, const float* scores, const void* k_dense,
                                          const void* v_dense, int64_t n_max, const int32_t* chunk_len_dev,
                                          const int32_t* keep_dev, int32_t* kv_len_dev, void* kv_pool,
                                          int64_t n_pool_pages, int32_t d, int32_t* idx_out, int32_t* clamped_dev,
                                          void* workspace, size_t workspace_bytes, void* stream) {
    if (!kv_len_dev) return fail(TANGRAM_ERR_INVALID_ARG, "compact_topk_chunk: NULL kv_len_dev");
    return compact_impl(dp, scores, k_dense, v_dense, n_max, chunk_len_dev, keep_dev, kv_len_dev, kv_pool, n_pool_pages,
                        d, idx_out, clamped_dev, workspace, workspace_bytes, stream);
}
