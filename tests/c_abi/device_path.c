/* Plain C caller of the whole path on the device (include/tangram.h + the CUDA runtime C API only, no Python, no
 * torch): reserve -> tables -> plan -> upload -> tangram_decode_attention, checked against closed forms
 * (SURVEY.md §8(c) pins): q = 0 and V_h == h + 1  =>  out_j = floor(j / G) + 1 exactly, lse_j = ln(kv_len);
 * everything in the pool that is not a retained row is NaN and must never reach the result.
 * Built and run by tests/test_gpu_parity.py::test_whole_path_from_plain_c. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "tangram.h"

#define CHECK(cond)                                                                  \
    do {                                                                             \
        if (!(cond)) {                                                               \
            fprintf(stderr, "FAILED %s:%d: %s (%s)\n", __FILE__, __LINE__, #cond, tangram_last_error()); \
            return 1;                                                                \
        }                                                                            \
    } while (0)

enum { R = 3, H = 2, HQ = 6, G = 3, D = 64, P = 16, C = 2, HP = 1 };

static float bf16_to_float(uint16_t b) {
    uint32_t u = (uint32_t)b << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

int main(void) {
    const double mu[H] = {1.0, 0.25}, sigma[H] = {0.0, 0.0};
    const int32_t ctx[R] = {1000, 37, 4096};
    double B[H];
    int32_t reserved[R * H], kv_len[R * H];
    int32_t perm[H], cluster_of[H], slot_of[H], *tbl_pages, *free_pages, split_map[C];
    int64_t tbl_indptr[R * C + 1], part_indptr[R * H + 1], *worker_indptr;
    tangram_tables t;
    tangram_plan p;
    tangram_device_plan dp;
    int32_t n_cta = 0;
    int64_t n_pool, i;
    int r, h, tok, e, j;

    CHECK(tangram_reserve_budgets(mu, sigma, 2.0, H, ctx, R, NULL, B, reserved, kv_len) == TANGRAM_OK);
    memset(&t, 0, sizeof t);
    CHECK(tangram_build_ragged_tables(B, reserved, R, H, C, P, NULL, 0, 0u, NULL, &t) == TANGRAM_ERR_OUT_OF_PAGES);
    n_pool = t.n_pages_used + 7;
    free_pages = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_pool);
    tbl_pages = (int32_t*)malloc(sizeof(int32_t) * (size_t)n_pool);
    for (i = 0; i < n_pool; ++i) free_pages[i] = (int32_t)((i * 7919) % n_pool); /* 7919 is prime: a permutation */
    if (n_pool % 7919 == 0) return 2;
    t.perm = perm, t.cluster_of = cluster_of, t.slot_of = slot_of, t.tbl_indptr = tbl_indptr, t.tbl_pages = tbl_pages;
    t.tbl_pages_cap = n_pool;
    CHECK(tangram_build_ragged_tables(B, reserved, R, H, C, P, free_pages, n_pool, 0u, NULL, &t) == TANGRAM_OK);

    CHECK(tangram_query_max_ctas(0, D, G, &n_cta) == TANGRAM_OK && n_cta > 0);
    memset(&p, 0, sizeof p);
    p.split_map = split_map;
    CHECK(tangram_plan_partitions(&t, B, kv_len, n_cta, 64, 1, TANGRAM_MODE_BALANCED, 0, 500, 6, &p) == TANGRAM_OK);
    p.items = (tangram_item*)malloc(sizeof(tangram_item) * (size_t)(p.n_items + 1));
    p.items_cap = p.n_items + 1;
    worker_indptr = (int64_t*)malloc(sizeof(int64_t) * (size_t)(p.W + 1));
    p.worker_indptr = worker_indptr, p.part_indptr = part_indptr;
    CHECK(tangram_plan_partitions(&t, B, kv_len, n_cta, 64, 1, TANGRAM_MODE_BALANCED, 0, 500, 6, &p) == TANGRAM_OK);

    {
        /* pool[page][slot][kv][token][d] bf16: NaN everywhere, K rows = 0.5 and V rows = h + 1 on retained tokens */
        const size_t page_elems = (size_t)HP * 2 * P * D, pool_elems = (size_t)n_pool * page_elems;
        uint16_t* pool = (uint16_t*)malloc(pool_elems * 2);
        uint16_t *q_h = (uint16_t*)calloc((size_t)R * HQ * D, 2), *out_h = (uint16_t*)malloc((size_t)R * HQ * D * 2);
        float* lse_h = (float*)malloc(sizeof(float) * R * HQ);
        void *d_blob, *d_q, *d_pool, *d_out, *d_lse, *d_ws;
        const size_t blob_bytes = tangram_blob_bytes(&t, &p), ws_bytes = tangram_workspace_bytes(p.n_part_slots, G, D);
        for (i = 0; i < (int64_t)pool_elems; ++i) pool[i] = 0x7FC0; /* NaN */
        for (r = 0; r < R; ++r)
            for (h = 0; h < H; ++h) {
                const int64_t row0 = tbl_indptr[r * C + cluster_of[h]];
                const uint16_t vbits = h == 0 ? 0x3F80 /* 1.0 */ : 0x4000 /* 2.0 */;
                for (tok = 0; tok < kv_len[r * H + h]; ++tok) {
                    uint16_t* pg = pool + (size_t)tbl_pages[row0 + tok / P] * page_elems + (size_t)slot_of[h] * 2 * P * D;
                    for (e = 0; e < D; ++e) {
                        pg[(0 * P + tok % P) * D + e] = 0x3F00; /* K = 0.5 */
                        pg[(1 * P + tok % P) * D + e] = vbits;
                    }
                }
            }
        CHECK(cudaMalloc(&d_blob, blob_bytes) == cudaSuccess && cudaMalloc(&d_q, (size_t)R * HQ * D * 2) == cudaSuccess);
        CHECK(cudaMalloc(&d_pool, pool_elems * 2) == cudaSuccess && cudaMalloc(&d_out, (size_t)R * HQ * D * 2) == cudaSuccess);
        CHECK(cudaMalloc(&d_lse, sizeof(float) * R * HQ) == cudaSuccess && cudaMalloc(&d_ws, ws_bytes + 256) == cudaSuccess);
        CHECK(cudaMemcpy(d_q, q_h, (size_t)R * HQ * D * 2, cudaMemcpyHostToDevice) == cudaSuccess);
        CHECK(cudaMemcpy(d_pool, pool, pool_elems * 2, cudaMemcpyHostToDevice) == cudaSuccess);
        CHECK(tangram_upload(&t, &p, d_blob, blob_bytes, NULL, &dp) == TANGRAM_OK);
        for (j = 0; j < 2; ++j) { /* twice: the scheduler counters re-arm themselves */
            CHECK(cudaMemset(d_out, 0xFF, (size_t)R * HQ * D * 2) == cudaSuccess);
            CHECK(tangram_decode_attention(&dp, d_q, d_pool, n_pool, NULL, HQ, D, 0.f, d_out, (float*)d_lse, d_ws, ws_bytes + 256,
                                           NULL, NULL) == TANGRAM_OK);
            CHECK(cudaDeviceSynchronize() == cudaSuccess);
            CHECK(cudaMemcpy(out_h, d_out, (size_t)R * HQ * D * 2, cudaMemcpyDeviceToHost) == cudaSuccess);
            CHECK(cudaMemcpy(lse_h, d_lse, sizeof(float) * R * HQ, cudaMemcpyDeviceToHost) == cudaSuccess);
            for (r = 0; r < R; ++r)
                for (h = 0; h < HQ; ++h) {
                    const float want = (float)(h / G + 1), want_lse = logf((float)kv_len[r * H + h / G]);
                    for (e = 0; e < D; ++e) CHECK(bf16_to_float(out_h[((size_t)r * HQ + h) * D + e]) == want);
                    CHECK(fabsf(lse_h[r * HQ + h] - want_lse) <= 1e-3f);
                }
        }
        /* error contract from C: a workspace that is too small, a head_dim the kernels do not have */
        if (p.n_part_slots > 0)
            CHECK(tangram_decode_attention(&dp, d_q, d_pool, n_pool, NULL, HQ, D, 0.f, d_out, (float*)d_lse, d_ws, 16, NULL,
                                           NULL) == TANGRAM_ERR_BUFFER_TOO_SMALL);
        CHECK(tangram_decode_attention(&dp, d_q, d_pool, n_pool, NULL, HQ, 96, 0.f, d_out, (float*)d_lse, d_ws, ws_bytes, NULL,
                                       NULL) == TANGRAM_ERR_INVALID_ARG);
    }
    printf("c_abi device path ok (W=%d, items=%lld, lists=%d)\n", (int)p.n_static, (long long)p.n_items, (int)dp.W);
    return 0;
}
