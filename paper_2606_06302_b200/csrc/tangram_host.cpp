// Host side of the Tangram hot path: Budget Reservation (a1), Ragged Paging tables (a2) and the
// Ahead-of-Time partition planner (a3).  Pure integer / fp64 code, no CUDA.  See include/tangram.h
// for the contract of every entry point and the PAPER.md passages they implement.
// Compiled with -ffp-contract=off: fp64 expressions are evaluated exactly as written.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <numeric>
#include <vector>
#if defined(__x86_64__) && defined(__GNUC__)
#include <immintrin.h>
#endif
#ifdef _OPENMP
#include <omp.h>
#endif

#include "tangram.h"
#include "tangram_internal.h"

namespace tangram {

static thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

// Algorithm 1 for one layer.  round() is half-up.
static void algorithm1(const double* B, const int32_t* perm, int32_t H, int32_t Hp, int32_t n_cta,
                       int32_t* S) {
    const int32_t C = H / Hp;
    std::fill(S, S + C, 1);
    double omega = 0.0;
    for (int32_t h = 0; h < H; ++h) omega += B[h];
    if (omega == 0.0) return;
    const double tau = omega / static_cast<double>(n_cta);
    for (int32_t i = 0; i < C; ++i) {
        double phi = 0.0;
        for (int32_t k = 0; k < Hp; ++k) phi += B[perm[i * Hp + k]];
        const double s = std::floor(phi / tau + 0.5);
        S[i] = s < 1.0 ? 1 : static_cast<int32_t>(s);
    }
}

struct RawItem {
    int32_t worker, r, h, tb, te;
};

}  // namespace tangram

using namespace tangram;

extern "C" const char* tangram_last_error(void) { return g_err; }

extern "C" int tangram_reserve_budgets(const double* mu, const double* sigma, double alpha, int32_t H,
                                       const int32_t* ctx_len, int32_t R, const int32_t* demand,
                                       double* B_out, int32_t* reserved_out, int32_t* kv_len_out) {
    if (!mu || !sigma || !ctx_len || !B_out || !reserved_out || !kv_len_out)
        return fail(TANGRAM_ERR_INVALID_ARG, "reserve_budgets: NULL argument");
    if (H < 1 || R < 1) return fail(TANGRAM_ERR_INVALID_ARG, "reserve_budgets: H=%d R=%d", H, R);
    std::vector<double> B(H);
    for (int32_t h = 0; h < H; ++h) {
        const double margin = alpha * sigma[h];
        const double b = std::min(1.0, mu[h] + margin);  // Eq. 5
        if (!(b > 0.0))
            return fail(TANGRAM_ERR_INVALID_ARG, "reserve_budgets: head %d has B=%g, not in (0,1]", h, b);
        B[h] = b;
    }
    for (int32_t r = 0; r < R; ++r) {
        if (ctx_len[r] < 1)
            return fail(TANGRAM_ERR_INVALID_ARG, "reserve_budgets: ctx_len[%d]=%d < 1", r, ctx_len[r]);
        if (demand)
            for (int32_t h = 0; h < H; ++h)
                if (demand[(size_t)r * H + h] < 0)
                    return fail(TANGRAM_ERR_INVALID_ARG, "reserve_budgets: demand[%d][%d] < 0", r, h);
    }
    std::copy(B.begin(), B.end(), B_out);
    for (int32_t r = 0; r < R; ++r) {
        const double N = static_cast<double>(ctx_len[r]);
        for (int32_t h = 0; h < H; ++h) {
            const double want = std::ceil(B[h] * N);  // Eq. 4: ceil(B N)
            int32_t n = want > N ? ctx_len[r] : static_cast<int32_t>(want);
            n = std::max(1, std::min(ctx_len[r], n));
            const size_t i = (size_t)r * H + h;
            reserved_out[i] = n;
            kv_len_out[i] = demand ? std::min(demand[i], n) : n;  // overflow truncation, :176
        }
    }
    return TANGRAM_OK;
}

extern "C" int tangram_build_ragged_tables(const double* B, const int32_t* reserved, int32_t R,
                                           int32_t H, int32_t n_clusters, int32_t page_size,
                                           const int32_t* free_pages, int64_t n_free, uint32_t flags,
                                           int32_t* kv_len_inout, tangram_tables* out) {
    if (!B || !reserved || !out) return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: NULL argument");
    if (R < 1 || H < 1 || n_clusters < 1 || H % n_clusters != 0)
        return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: H=%d not a multiple of n_clusters=%d (R=%d)", H,
                    n_clusters, R);
    if (page_size <= 0) return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: page_size=%d", page_size);
    if (n_free < 0 || (n_free > 0 && !free_pages))
        return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: bad free list");
    const int32_t C = n_clusters, Hp = H / C;
    const int32_t headroom = out->headroom_pages;
    if (headroom < 0 || headroom > (1 << 20))
        return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: headroom_pages=%d", headroom);

    // Budget-Aware Clustering (:227-233): stable ascending sort on B only.
    std::vector<int32_t> order(H);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return B[a] < B[b]; });

    // capacity of every (request, cluster) row: the cluster's largest reservation (:190)
    std::vector<int32_t> cap((size_t)R * C);
    int64_t need = 0;
    for (int32_t r = 0; r < R; ++r)
        for (int32_t c = 0; c < C; ++c) {
            int32_t mx = 0;
            for (int32_t k = 0; k < Hp; ++k) {
                const int32_t v = reserved[(size_t)r * H + order[c * Hp + k]];
                if (v < 0) return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: reserved < 0");
                mx = std::max(mx, v);
            }
            cap[(size_t)r * C + c] = mx;
            need += (mx + page_size - 1) / page_size;
        }
    out->R = R, out->H = H, out->C = C, out->Hp = Hp, out->P = page_size;
    out->n_pages_used = need;
    const int64_t n_slots = need + (int64_t)R * C * headroom;
    out->n_slots = n_slots;
    if (need > n_free)
        return fail(TANGRAM_ERR_OUT_OF_PAGES, "build_ragged_tables: need %lld pages, free list has %lld",
                    (long long)need, (long long)n_free);
    if (!out->tbl_pages) return TANGRAM_OK;  // query
    if (!out->perm || !out->cluster_of || !out->slot_of || !out->tbl_indptr)
        return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: NULL output array");
    if (headroom > 0 && !out->row_pages)
        return fail(TANGRAM_ERR_INVALID_ARG, "build_ragged_tables: headroom_pages > 0 needs the row_pages array");
    if (out->tbl_pages_cap < n_slots)
        return fail(TANGRAM_ERR_BUFFER_TOO_SMALL, "build_ragged_tables: tbl_pages_cap %lld < %lld",
                    (long long)out->tbl_pages_cap, (long long)n_slots);
    for (int32_t j = 0; j < H; ++j) {
        out->perm[j] = order[j];
        out->cluster_of[order[j]] = j / Hp;
        out->slot_of[order[j]] = j % Hp;
    }
    int64_t cur = 0, slot = 0;  // next free-list entry, next table slot
    out->tbl_indptr[0] = 0;
    for (int64_t row = 0; row < (int64_t)R * C; ++row) {
        const int64_t n = (cap[row] + page_size - 1) / page_size;
        std::memcpy(out->tbl_pages + slot, free_pages + cur, sizeof(int32_t) * (size_t)n);
        std::fill(out->tbl_pages + slot + n, out->tbl_pages + slot + n + headroom, -1);  // growth slots: no page yet
        cur += n, slot += n + headroom;
        out->tbl_indptr[row + 1] = slot;
        if (out->row_pages) out->row_pages[row] = (int32_t)n;
    }
    if ((flags & TANGRAM_FILL_GROUP) && kv_len_inout)
        for (int32_t r = 0; r < R; ++r)
            for (int32_t h = 0; h < H; ++h)
                kv_len_inout[(size_t)r * H + h] = cap[(size_t)r * C + out->cluster_of[h]];
    return TANGRAM_OK;
}

// ---- NEXT-4: Vectorized Block Table update (:244): every (request, cluster) row whose longest head has filled
// the row's pages takes the next free page.  Pass 1 finds those rows for all groups at once -- OpenMP across
// (cluster, block of 16 requests), AVX-512 inside a block: one gather of the H_p member lengths per lane, a
// vector max, a compare against pages x P -- and leaves one mask bit per row; pass 2 hands out the pages in row
// order (the free list is consumed in (request, cluster) order, so it is a sequential walk over the set bits).
namespace tangram {

static void rows_needing_a_page_scalar(const tangram_tables* t, const int32_t* kv_len, int32_t c, int32_t r0,
                                       int32_t r1, uint8_t* need) {
    const int32_t H = t->H, C = t->C, Hp = t->Hp, P = t->P;
    for (int32_t r = r0; r < r1; ++r) {
        int32_t longest = 0;
        for (int32_t k = 0; k < Hp; ++k) longest = std::max(longest, kv_len[(size_t)r * H + t->perm[c * Hp + k]]);
        const int64_t row = (int64_t)r * C + c;
        need[row] = (int64_t)longest >= (int64_t)t->row_pages[row] * P;
    }
}

#if defined(__x86_64__) && defined(__GNUC__)
__attribute__((target("avx512f"))) static void rows_needing_a_page_avx512(const tangram_tables* t, const int32_t* kv_len,
                                                                         int32_t c, int32_t r0, int32_t r1, uint8_t* need) {
    const int32_t H = t->H, C = t->C, Hp = t->Hp, P = t->P;
    const __m512i lane = _mm512_setr_epi32(0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 15);
    int32_t r = r0;
    // 16 requests per step; the 32-bit gather indices must not overflow
    if ((int64_t)t->R * H < INT32_MAX && (int64_t)t->R * C < INT32_MAX)
        for (; r + 16 <= r1; r += 16) {
            const __m512i rr = _mm512_add_epi32(_mm512_set1_epi32(r), lane);
            const __m512i seq0 = _mm512_mullo_epi32(rr, _mm512_set1_epi32(H));
            __m512i longest = _mm512_setzero_si512();
            for (int32_t k = 0; k < Hp; ++k) {
                const __m512i idx = _mm512_add_epi32(seq0, _mm512_set1_epi32(t->perm[c * Hp + k]));
                longest = _mm512_max_epi32(longest, _mm512_i32gather_epi32(idx, kv_len, 4));
            }
            const __m512i row = _mm512_add_epi32(_mm512_mullo_epi32(rr, _mm512_set1_epi32(C)), _mm512_set1_epi32(c));
            const __m512i have = _mm512_i32gather_epi32(row, t->row_pages, 4);
            // longest >= have * P  (lengths and capacities are far below 2^31)
            const __mmask16 m = _mm512_cmpge_epi32_mask(longest, _mm512_mullo_epi32(have, _mm512_set1_epi32(P)));
            for (int32_t i = 0; i < 16; ++i) need[((int64_t)r + i) * C + c] = (m >> i) & 1;
        }
    rows_needing_a_page_scalar(t, kv_len, c, r, r1, need);
}
static bool have_avx512() { return __builtin_cpu_supports("avx512f"); }
#else
static bool have_avx512() { return false; }
#endif

}  // namespace tangram

extern "C" int tangram_extend_tables(tangram_tables* t, const int32_t* kv_len, const int32_t* free_pages, int64_t n_free,
                                     int32_t n_threads, int64_t* n_extended_out, int64_t* n_starved_out) {
    if (!t || !kv_len || (n_free > 0 && !free_pages) || n_free < 0)
        return fail(TANGRAM_ERR_INVALID_ARG, "extend_tables: NULL argument");
    if (!t->row_pages || !t->tbl_indptr || !t->tbl_pages || !t->perm)
        return fail(TANGRAM_ERR_INVALID_ARG, "extend_tables: the tables were built without row_pages (growth headroom)");
    const int32_t R = t->R, C = t->C;
    const int64_t n_rows = (int64_t)R * C;
    std::vector<uint8_t> need((size_t)n_rows, 0);
    const bool simd = have_avx512();
    const int32_t blocks = (R + 255) / 256;  // 256 requests = 16 vector steps per task
    const int64_t n_tasks = (int64_t)C * blocks;
#ifdef _OPENMP
    const int nt = n_threads > 0 ? n_threads : std::min<int64_t>(omp_get_max_threads(), std::max<int64_t>(1, n_rows / 2048));
#pragma omp parallel for schedule(static) num_threads(nt) if (nt > 1)
#endif
    for (int64_t task = 0; task < n_tasks; ++task) {
        const int32_t c = (int32_t)(task / blocks), r0 = (int32_t)(task % blocks) * 256, r1 = std::min(R, r0 + 256);
#if defined(__x86_64__) && defined(__GNUC__)
        if (simd) rows_needing_a_page_avx512(t, kv_len, c, r0, r1, need.data());
        else
#endif
            rows_needing_a_page_scalar(t, kv_len, c, r0, r1, need.data());
    }
    (void)simd, (void)n_threads;
    int64_t cursor = t->n_pages_used, extended = 0, starved = 0;
    for (int64_t row = 0; row < n_rows; ++row) {
        if (!need[(size_t)row]) continue;
        const int64_t lo = t->tbl_indptr[row], slots = t->tbl_indptr[row + 1] - lo;
        const int32_t have = t->row_pages[row];
        if (have >= slots || cursor >= n_free) {
            ++starved;
            continue;
        }
        t->tbl_pages[lo + have] = free_pages[cursor++];
        t->row_pages[row] = have + 1;
        ++extended;
    }
    t->n_pages_used = cursor;
    if (n_extended_out) *n_extended_out = extended;
    if (n_starved_out) *n_starved_out = starved;
    return TANGRAM_OK;
}

extern "C" int tangram_plan_partitions(const tangram_tables* t, const double* B, const int32_t* kv_len,
                                       int32_t n_workers, int32_t granule_tokens,
                                       int32_t overhead_granules, int32_t mode, int32_t static_splits,
                                       int32_t dyn_permille, int32_t dyn_rounds, tangram_plan* out) {
    if (!t || !B || !kv_len || !out) return fail(TANGRAM_ERR_INVALID_ARG, "plan_partitions: NULL argument");
    if (!t->perm || !t->cluster_of || !t->slot_of || !t->tbl_indptr)
        return fail(TANGRAM_ERR_INVALID_ARG, "plan_partitions: tables not filled");
    const int32_t R = t->R, H = t->H, C = t->C, Hp = t->Hp, P = t->P;
    const int32_t NW = n_workers, g = granule_tokens, c0 = overhead_granules;
    if (NW < 1 || g < 1 || P < 1 || g % P != 0 || c0 < 0)
        return fail(TANGRAM_ERR_INVALID_ARG,
                    "plan_partitions: W=%d granule=%d (must be a positive multiple of P=%d) overhead=%d", NW, g, P, c0);
    if (dyn_permille < 0 || dyn_permille >= 1000 || dyn_rounds < 0 || dyn_rounds > 16 ||
        (dyn_permille > 0) != (dyn_rounds > 0))
        return fail(TANGRAM_ERR_INVALID_ARG, "plan_partitions: dyn_permille=%d dyn_rounds=%d", dyn_permille, dyn_rounds);
    // Work-list slots: the first NW are the CTAs' own lists; with a dynamic tail (BALANCED only) they
    // are followed by dyn_rounds rounds of NW smaller lists that the CTAs claim in order at run time.
    const bool tail = mode == TANGRAM_MODE_BALANCED && dyn_rounds > 0;
    const int32_t W = tail ? NW * (1 + dyn_rounds) : NW;
    if (mode != TANGRAM_MODE_BALANCED && mode != TANGRAM_MODE_SPLITMAP && mode != TANGRAM_MODE_STATIC_EVEN)
        return fail(TANGRAM_ERR_INVALID_ARG, "plan_partitions: mode=%d", mode);
    for (int32_t r = 0; r < R; ++r)
        for (int32_t h = 0; h < H; ++h) {
            const int64_t row = (int64_t)r * C + t->cluster_of[h];
            const int64_t cap_tokens = (t->tbl_indptr[row + 1] - t->tbl_indptr[row]) * (int64_t)P;
            const int32_t n = kv_len[(size_t)r * H + h];
            if (n < 0 || n > cap_tokens)
                return fail(TANGRAM_ERR_INVALID_ARG, "plan_partitions: kv_len[%d][%d]=%d exceeds its table (%lld tokens)",
                            r, h, n, (long long)cap_tokens);
        }

    std::vector<int32_t> S(C);
    algorithm1(B, t->perm, H, Hp, NW, S.data());
    std::vector<RawItem> raw;
    const int64_t n_seq = (int64_t)R * H;
    raw.reserve((size_t)(n_seq + W));

    if (mode == TANGRAM_MODE_BALANCED) {
        // Lay the sequences end to end on a cost axis (granules, plus c0 per non-empty sequence) and
        // cut the axis at b_k = floor(k T / W).
        int64_t T = 0;
        for (int32_t r = 0; r < R; ++r)
            for (int32_t h = 0; h < H; ++h) {
                const int64_t u = (kv_len[(size_t)r * H + h] + (int64_t)g - 1) / g;
                T += u + (u > 0 ? c0 : 0);
            }
        // Relative size of list k: (1000 - dyn) 2^(J-1) for the NW static lists; dyn 2^(J-1-j) for the
        // lists of round j = 1..J-1 and dyn for the last round J (each round hands out half of what is
        // left, the last one all of it).  b_k = floor(T cumw_k / cumw_W).
        std::vector<int64_t> cumw((size_t)W + 1, 0);
        for (int32_t k = 0; k < W; ++k) {
            int64_t w = 1;
            if (tail) {
                const int32_t J = dyn_rounds, round = k / NW;  // 0 = static
                if (round == 0) w = (int64_t)(1000 - dyn_permille) << (J - 1);
                else if (round < J) w = (int64_t)dyn_permille << (J - 1 - round);
                else w = dyn_permille;
            }
            cumw[(size_t)k + 1] = cumw[(size_t)k] + w;
        }
        const int64_t totw = cumw[(size_t)W];
        auto cut = [&](int64_t k) { return (int64_t)(((__int128)T * cumw[(size_t)k]) / totw); };
        int64_t pos = 0;   // cost position where the current sequence starts
        int64_t k = 0;     // current worker
        for (int32_t r = 0; r < R; ++r)
            for (int32_t j = 0; j < H; ++j) {
                const int32_t h = t->perm[j];
                const int32_t n = kv_len[(size_t)r * H + h];
                const int64_t u = (n + (int64_t)g - 1) / g;
                if (u == 0) continue;
                const int64_t first = pos + c0, last = first + u;  // granule positions [first, last)
                int64_t p = first;
                while (p < last) {
                    while (cut(k + 1) <= p) ++k;
                    const int64_t stop = std::min(last, cut(k + 1));
                    const int64_t tb = (p - first) * g;
                    const int64_t te = std::min<int64_t>(n, (stop - first) * g);
                    raw.push_back({(int32_t)k, r, h, (int32_t)tb, (int32_t)te});
                    p = stop;
                }
                pos = last;
            }
    } else {
        int32_t s_even = static_splits;
        if (mode == TANGRAM_MODE_STATIC_EVEN) {
            if (s_even <= 0) s_even = (int32_t)std::max<int64_t>(1, (W + n_seq - 1) / n_seq);
            std::fill(S.begin(), S.end(), s_even);
        }
        int64_t dealt = 0;
        for (int32_t r = 0; r < R; ++r)
            for (int32_t j = 0; j < H; ++j) {
                const int32_t h = t->perm[j];
                const int32_t n = kv_len[(size_t)r * H + h];
                const int64_t u = (n + (int64_t)g - 1) / g;
                const int64_t Sc = S[t->cluster_of[h]];
                for (int64_t c = 0; c < Sc; ++c) {
                    const int64_t lo = (c * u) / Sc, hi = ((c + 1) * u) / Sc;
                    const int64_t tb = lo * g, te = std::min<int64_t>(n, hi * g);
                    if (te <= tb) continue;
                    raw.push_back({(int32_t)(dealt % W), r, h, (int32_t)tb, (int32_t)te});
                    ++dealt;
                }
            }
    }

    out->W = W, out->n_static = NW, out->mode = mode;
    out->n_items = (int64_t)raw.size();
    out->n_part_slots = (int64_t)raw.size();
    if (out->split_map) std::copy(S.begin(), S.end(), out->split_map);
    if (!out->items) return TANGRAM_OK;  // query
    if (!out->worker_indptr || !out->part_indptr || !out->split_map)
        return fail(TANGRAM_ERR_INVALID_ARG, "plan_partitions: NULL output array");
    if (out->items_cap < out->n_items)
        return fail(TANGRAM_ERR_BUFFER_TOO_SMALL, "plan_partitions: items_cap %lld < %lld", (long long)out->items_cap,
                    (long long)out->n_items);

    // parts per sequence; raw is already in token order inside every sequence
    std::vector<int64_t> cnt((size_t)n_seq, 0);
    for (const RawItem& it : raw) ++cnt[(size_t)it.r * H + it.h];
    out->part_indptr[0] = 0;
    for (int64_t s = 0; s < n_seq; ++s) out->part_indptr[s + 1] = out->part_indptr[s] + cnt[(size_t)s];
    std::vector<int64_t> wcount((size_t)W + 1, 0);
    for (const RawItem& it : raw) ++wcount[(size_t)it.worker + 1];
    for (int32_t w = 0; w < W; ++w) wcount[(size_t)w + 1] += wcount[(size_t)w];
    std::copy(wcount.begin(), wcount.end(), out->worker_indptr);
    std::vector<int64_t> wcur(wcount.begin(), wcount.end() - 1);
    std::vector<int64_t> ord((size_t)n_seq, 0);
    for (const RawItem& it : raw) {
        const size_t s = (size_t)it.r * H + it.h;
        tangram_item& o = out->items[wcur[(size_t)it.worker]++];
        o.req = it.r, o.kv_head = it.h, o.cluster = t->cluster_of[it.h], o.slot = t->slot_of[it.h];
        o.tok_begin = it.tb, o.tok_end = it.te;
        o.part_slot = (int32_t)(out->part_indptr[s] + ord[s]++);
        o.n_parts = (int32_t)cnt[s];
    }
    return TANGRAM_OK;
}

// ---- NEXT-3: page accounting under a grouping policy (Fig. 7 :168, :190, Fig. 15 :316-320)
extern "C" int tangram_account_pages(const double* B, const int32_t* reserved, const int32_t* ctx_len, int32_t R,
                                     int32_t H, int32_t heads_per_page, int32_t page_size, int32_t policy,
                                     tangram_page_account* out) {
    if (!B || !reserved || !ctx_len || !out) return fail(TANGRAM_ERR_INVALID_ARG, "account_pages: NULL argument");
    const int32_t Hp = heads_per_page, P = page_size;
    if (R < 1 || H < 1 || Hp < 1 || H % Hp != 0 || P < 1)
        return fail(TANGRAM_ERR_INVALID_ARG, "account_pages: R=%d H=%d heads_per_page=%d page_size=%d", R, H, Hp, P);
    if (policy != TANGRAM_GROUP_CLUSTERED && policy != TANGRAM_GROUP_ADJACENT)
        return fail(TANGRAM_ERR_INVALID_ARG, "account_pages: policy=%d", policy);
    std::vector<int32_t> order(H);
    std::iota(order.begin(), order.end(), 0);
    if (policy == TANGRAM_GROUP_CLUSTERED)  // the same stable sort as the table builder (:227-233)
        std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return B[a] < B[b]; });
    int64_t pages = 0, exact = 0, full = 0, used = 0;
    for (int32_t r = 0; r < R; ++r) {
        if (ctx_len[r] < 1) return fail(TANGRAM_ERR_INVALID_ARG, "account_pages: ctx_len[%d]=%d < 1", r, ctx_len[r]);
        const int32_t* row = reserved + (size_t)r * H;
        for (int32_t h = 0; h < H; ++h) {
            if (row[h] < 0) return fail(TANGRAM_ERR_INVALID_ARG, "account_pages: reserved[%d][%d] < 0", r, h);
            exact += (int64_t)P * ((row[h] + (int64_t)P - 1) / P);
            used += row[h];
        }
        for (int32_t g = 0; g < H / Hp; ++g) {
            int32_t longest = 0;
            for (int32_t j = 0; j < Hp; ++j) longest = std::max(longest, row[order[g * Hp + j]]);
            pages += (longest + (int64_t)P - 1) / P;
        }
        full += (int64_t)H * P * ((ctx_len[r] + (int64_t)P - 1) / P);
    }
    const int64_t alloc = (int64_t)Hp * P * pages;
    out->pages_alloc = pages, out->slots_alloc = alloc, out->slots_exact = exact, out->slots_full = full;
    out->slots_used = used, out->tables = (int64_t)R * (H / Hp);
    out->reclaimed_frac = 1.0 - static_cast<double>(alloc) / static_cast<double>(full);
    out->fragmentation = alloc > 0 ? static_cast<double>(alloc - used) / static_cast<double>(alloc) : 0.0;
    return TANGRAM_OK;
}

// ---- NEXT-4: Budget Calibration (:156-158, Eq. 5); population sigma, sums in sample order
extern "C" int tangram_calibrate_budgets(const double* ratios, int32_t n_samples, int32_t H, double alpha,
                                         double* mu_out, double* sigma_out, double* B_out) {
    if (!ratios || !mu_out || !sigma_out) return fail(TANGRAM_ERR_INVALID_ARG, "calibrate_budgets: NULL argument");
    if (n_samples < 1 || H < 1) return fail(TANGRAM_ERR_INVALID_ARG, "calibrate_budgets: n_samples=%d H=%d", n_samples, H);
    for (size_t i = 0; i < (size_t)n_samples * H; ++i)
        if (!std::isfinite(ratios[i])) return fail(TANGRAM_ERR_INVALID_ARG, "calibrate_budgets: ratio %zu is not finite", i);
    const double n = static_cast<double>(n_samples);
    for (int32_t h = 0; h < H; ++h) {
        double acc = 0.0;
        for (int32_t i = 0; i < n_samples; ++i) acc = acc + ratios[(size_t)i * H + h];
        const double m = acc / n;
        double acc2 = 0.0;
        for (int32_t i = 0; i < n_samples; ++i) {
            const double dlt = ratios[(size_t)i * H + h] - m;
            const double sq = dlt * dlt;
            acc2 = acc2 + sq;
        }
        const double sd = std::sqrt(acc2 / n);
        mu_out[h] = m, sigma_out[h] = sd;
        if (B_out) {
            const double margin = alpha * sd;
            B_out[h] = std::min(1.0, m + margin);  // Eq. 5
        }
    }
    return TANGRAM_OK;
}

// ---- default dynamic tail of the BALANCED plan (measured tuning rule, reading A32)
extern "C" int tangram_default_dynamic_tail(const int32_t* kv_len, int32_t R, int32_t H, int32_t n_workers,
                                            int32_t granule_tokens, int32_t overhead_granules,
                                            int32_t* dyn_permille_out, int32_t* dyn_rounds_out) {
    if (!kv_len || !dyn_permille_out || !dyn_rounds_out || R < 1 || H < 1 || n_workers < 1 || granule_tokens < 1 ||
        overhead_granules < 0)
        return fail(TANGRAM_ERR_INVALID_ARG, "default_dynamic_tail: bad argument");
    int64_t total = 0;
    for (int64_t i = 0; i < (int64_t)R * H; ++i) {
        if (kv_len[i] < 0) return fail(TANGRAM_ERR_INVALID_ARG, "default_dynamic_tail: kv_len < 0");
        const int64_t u = (kv_len[i] + (int64_t)granule_tokens - 1) / granule_tokens;
        total += u + (u > 0 ? overhead_granules : 0);
    }
    // fewer than 48 cost units per worker: static; up to 384: half of the axis in 4 rounds; above: in 6 rounds
    if (total < (int64_t)48 * n_workers) *dyn_permille_out = 0, *dyn_rounds_out = 0;
    else if (total < (int64_t)384 * n_workers) *dyn_permille_out = 500, *dyn_rounds_out = 4;
    else *dyn_permille_out = 500, *dyn_rounds_out = 6;
    return TANGRAM_OK;
}
