/*
 * TEST INFRASTRUCTURE -- fp64 CPU oracle for Tangram decode attention (O1 of DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with the CUDA path (paper_2606_06302_b200/csrc) and is the plain
 * definition written out: for one request r and one query head j, gather the retained tokens of
 * KV head h = floor(j / G) through that head's cluster page table (Ragged Paging, PAPER.md:190
 * "a page holds H_p x 2 x P x d elements for the H_p heads of one group in one layer"; Eq. 1,
 * PAPER.md:57-58, K~ = K[I,:], V~ = V[I,:]) and evaluate softmax(q K~^T / sqrt(d)) V~ in fp64.
 * The paper never writes softmax attention out; the softmax scale (1/sqrt(d) unless the caller
 * gives another one, as tangram_decode_attention's sm_scale argument does) and natural-log LSE are
 * DESIGN.md readings A19/A20/A21.  Element order inside a page is reading A4:
 * pool[page][slot][kv][token][d], kv 0 = K, 1 = V, bf16.
 *
 * No blocking, no online softmax, no reordering: three plain passes (scores, max+sum, PV).
 * Pins: tests/test_oracle_pins.py (dense library attention, brute force, closed forms,
 * split/merge identity, page-permutation invariance).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16; /* bf16 is the upper half of an IEEE binary32 */
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

typedef struct {
    const uint16_t* q;          /* [R][Hq][d] bf16 */
    const uint16_t* pool;       /* [n_pages][Hp][2][P][d] bf16 */
    const int64_t* tbl_indptr;  /* [R*C+1], row = r*C + c */
    const int32_t* tbl_pages;   /* page ids */
    const int32_t* cluster_of;  /* [H] */
    const int32_t* slot_of;     /* [H] */
    int32_t R, H, Hq, C, Hp, P, d;
    double scale;               /* softmax scale: x_t = (q . k_t) * scale; <= 0 means 1/sqrt(d) (reading A19) */
} oracle_ctx;

/* Attention of query head j of request r over tokens [t0, t1) of its KV head.
 * out[d] is normalised within the range; *lse = log sum_t exp(x_t).  Empty range: out = 0,
 * lse = -inf. */
static void attend_range(const oracle_ctx* c, int r, int j, int t0, int t1, double* out,
                         double* lse) {
    const int G = c->Hq / c->H;
    const int h = j / G;
    const int cl = c->cluster_of[h];
    const int s = c->slot_of[h];
    const int d = c->d, P = c->P;
    const int n = t1 - t0;
    for (int e = 0; e < d; ++e) out[e] = 0.0;
    if (n <= 0) {
        *lse = -INFINITY;
        return;
    }
    const uint16_t* qv = c->q + ((size_t)r * c->Hq + j) * d;
    const int32_t* row = c->tbl_pages + c->tbl_indptr[(size_t)r * c->C + cl];
    const size_t page_elems = (size_t)c->Hp * 2 * P * d;
    double* x = (double*)malloc(sizeof(double) * (size_t)n);
    const double scale = c->scale > 0.0 ? c->scale : 1.0 / sqrt((double)d);
    /* pass 1: x_t = (q . k_t) * scale   (scale = 1/sqrt(d) by default) */
    for (int t = t0; t < t1; ++t) {
        const size_t page = (size_t)row[t / P];
        const uint16_t* k = c->pool + page * page_elems + (((size_t)s * 2 + 0) * P + (t % P)) * d;
        double acc = 0.0;
        for (int e = 0; e < d; ++e) acc += bf16_to_f64(qv[e]) * bf16_to_f64(k[e]);
        x[t - t0] = acc * scale;
    }
    /* pass 2: m = max x, l = sum exp(x - m) */
    double m = x[0];
    for (int i = 1; i < n; ++i)
        if (x[i] > m) m = x[i];
    double l = 0.0;
    for (int i = 0; i < n; ++i) l += exp(x[i] - m);
    /* pass 3: out = sum exp(x - m) v_t / l */
    for (int t = t0; t < t1; ++t) {
        const size_t page = (size_t)row[t / P];
        const uint16_t* v = c->pool + page * page_elems + (((size_t)s * 2 + 1) * P + (t % P)) * d;
        const double p = exp(x[t - t0] - m);
        for (int e = 0; e < d; ++e) out[e] += p * bf16_to_f64(v[e]);
    }
    for (int e = 0; e < d; ++e) out[e] /= l;
    *lse = m + log(l);
    free(x);
}

void tangram_oracle_attend_range(const uint16_t* q, const uint16_t* pool, const int64_t* tbl_indptr,
                                 const int32_t* tbl_pages, const int32_t* cluster_of,
                                 const int32_t* slot_of, int32_t R, int32_t H, int32_t Hq, int32_t C,
                                 int32_t Hp, int32_t P, int32_t d, int32_t r, int32_t j, int32_t t0,
                                 int32_t t1, double scale, double* out, double* lse) {
    oracle_ctx c = {q, pool, tbl_indptr, tbl_pages, cluster_of, slot_of, R, H, Hq, C, Hp, P, d, scale};
    attend_range(&c, r, j, t0, t1, out, lse);
}

/* Attention for a list of (request, query head) pairs: pairs[2*i] = r, pairs[2*i+1] = j.
 * out [n_pairs][d], lse [n_pairs].  kv_len [R][H].  A plain `parallel for` over the pairs
 * (each pair is independent); n_threads <= 0 keeps the OpenMP default; scale <= 0 means 1/sqrt(d).
 * Returns the number of threads used. */
int tangram_oracle_attention_pairs(const uint16_t* q, const uint16_t* pool,
                                   const int64_t* tbl_indptr, const int32_t* tbl_pages,
                                   const int32_t* cluster_of, const int32_t* slot_of,
                                   const int32_t* kv_len, int32_t R, int32_t H, int32_t Hq,
                                   int32_t C, int32_t Hp, int32_t P, int32_t d,
                                   const int32_t* pairs, int64_t n_pairs, double scale, double* out,
                                   double* lse, int32_t n_threads) {
    oracle_ctx c = {q, pool, tbl_indptr, tbl_pages, cluster_of, slot_of, R, H, Hq, C, Hp, P, d, scale};
    const int G = Hq / H;
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int64_t i = 0; i < n_pairs; ++i) {
        const int r = pairs[2 * i], j = pairs[2 * i + 1];
        const int n = kv_len[(size_t)r * H + j / G];
        attend_range(&c, r, j, 0, n, out + (size_t)i * d, lse + i);
    }
    return used;
}
