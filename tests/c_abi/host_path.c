/* Plain C99 caller of the C ABI (include/tangram.h): Budget Reservation -> Ragged Paging tables -> AoT plan ->
 * page accounting -> calibration, host side only (no CUDA device needed).  Built and run by
 * tests/test_host_vs_oracle.py::test_header_is_plain_c_and_host_path_runs_from_c with -std=c99 -pedantic -Werror;
 * the values checked are the hand-evaluated fixtures of tests/golden/hand_examples.json / SURVEY.md §8(c). */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "tangram.h"

#define CHECK(cond)                                                                  \
    do {                                                                             \
        if (!(cond)) {                                                               \
            fprintf(stderr, "FAILED %s:%d: %s (%s)\n", __FILE__, __LINE__, #cond, tangram_last_error()); \
            return 1;                                                                \
        }                                                                            \
    } while (0)

int main(void) {
    /* a1: mu = .25, sigma = .0625, alpha = 2 -> B = .375; N = 1000 -> 375, N = 1001 -> 376 (dyadic closed form) */
    const double mu[2] = {0.25, 0.9375}, sigma[2] = {0.0625, 0.0625};
    const int32_t ctx[2] = {1000, 1001};
    double B[2];
    int32_t reserved[4], kv_len[4];
    CHECK(tangram_reserve_budgets(mu, sigma, 2.0, 2, ctx, 2, NULL, B, reserved, kv_len) == TANGRAM_OK);
    CHECK(B[0] == 0.375 && B[1] == 1.0);
    CHECK(reserved[0] == 375 && reserved[1] == 1000 && reserved[2] == 376 && reserved[3] == 1001);
    CHECK(memcmp(reserved, kv_len, sizeof reserved) == 0);

    /* a2: two clusters of one head, P = 16 */
    int32_t free_pages[200], perm[2], cluster_of[2], slot_of[2], tbl_pages[200];
    int64_t tbl_indptr[5];
    tangram_tables t;
    int i;
    for (i = 0; i < 200; ++i) free_pages[i] = 199 - i;
    memset(&t, 0, sizeof t);
    CHECK(tangram_build_ragged_tables(B, reserved, 2, 2, 2, 16, free_pages, 200, 0u, NULL, &t) == TANGRAM_OK);
    CHECK(t.n_pages_used == 24 + 63 + 24 + 63); /* ceil(375/16), ceil(1000/16), ceil(376/16), ceil(1001/16) */
    t.perm = perm, t.cluster_of = cluster_of, t.slot_of = slot_of, t.tbl_indptr = tbl_indptr, t.tbl_pages = tbl_pages;
    t.tbl_pages_cap = 200;
    CHECK(tangram_build_ragged_tables(B, reserved, 2, 2, 2, 16, free_pages, 200, 0u, NULL, &t) == TANGRAM_OK);
    CHECK(perm[0] == 0 && perm[1] == 1 && tbl_indptr[1] == 24 && tbl_indptr[4] == 174 && tbl_pages[0] == 199);
    CHECK(tangram_build_ragged_tables(B, reserved, 2, 2, 2, 16, free_pages, 100, 0u, NULL, &t) == TANGRAM_ERR_OUT_OF_PAGES);

    /* a3: Algorithm 1 on the tables' budgets with N_CTA = 11: Phi / tau = [3, 8] */
    {
        int32_t split_map[2];
        int64_t worker_indptr[12], part_indptr[5];
        tangram_plan p;
        tangram_item* items;
        memset(&p, 0, sizeof p);
        p.split_map = split_map;
        CHECK(tangram_plan_partitions(&t, B, kv_len, 11, 64, 1, TANGRAM_MODE_SPLITMAP, 0, 0, 0, &p) == TANGRAM_OK);
        CHECK(split_map[0] == 3 && split_map[1] == 8 && p.n_items == 2 * (3 + 8));
        items = (tangram_item*)malloc(sizeof(tangram_item) * (size_t)p.n_items);
        p.items = items, p.items_cap = p.n_items, p.worker_indptr = worker_indptr, p.part_indptr = part_indptr;
        CHECK(tangram_plan_partitions(&t, B, kv_len, 11, 64, 1, TANGRAM_MODE_SPLITMAP, 0, 0, 0, &p) == TANGRAM_OK);
        CHECK(worker_indptr[11] == p.n_items && part_indptr[4] == p.n_part_slots);
        CHECK(tangram_plan_partitions(&t, B, kv_len, 11, 65, 1, TANGRAM_MODE_BALANCED, 0, 0, 0, &p) == TANGRAM_ERR_INVALID_ARG);
        free(items);
    }

    /* NEXT-3: Fig. 7 in numbers */
    {
        const double Bf[6] = {0.25, 1.0, 0.25, 0.25, 1.0, 0.25};
        const int32_t res[6] = {16, 64, 16, 16, 64, 16}, n64[1] = {64};
        tangram_page_account a;
        CHECK(tangram_account_pages(Bf, res, n64, 1, 6, 3, 16, TANGRAM_GROUP_ADJACENT, &a) == TANGRAM_OK);
        CHECK(a.slots_alloc == 384 && a.reclaimed_frac == 0.0);
        CHECK(tangram_account_pages(Bf, res, n64, 1, 6, 3, 16, TANGRAM_GROUP_CLUSTERED, &a) == TANGRAM_OK);
        CHECK(a.slots_alloc == 240 && a.reclaimed_frac == 1.0 - 240.0 / 384.0 && a.tables == 2);
    }

    /* NEXT-4: {1/4, 3/4} -> mu = 1/2, population sigma = 1/4, B = 3/4 at alpha = 1 */
    {
        const double x[2] = {0.25, 0.75};
        double m, sd, b;
        CHECK(tangram_calibrate_budgets(x, 2, 1, 1.0, &m, &sd, &b) == TANGRAM_OK);
        CHECK(m == 0.5 && sd == 0.25 && b == 0.75);
    }
    /* NEXT-4 (block tables): the hand-evaluated growth example of tests/golden/hand_examples.json "extend_tables":
     * B = [.9,.2,.6,.3] -> clusters {1,3} and {2,0}; 2 growth slots per row; 7 pages built, 4 more handed out */
    {
        const double Bg[4] = {0.9, 0.2, 0.6, 0.3};
        const int32_t res[8] = {40, 10, 33, 16, 16, 5, 20, 7};
        const int32_t fl[11] = {50, 7, 23, 41, 8, 15, 16, 42, 4, 99, 3};
        const int32_t kv1[8] = {40, 10, 33, 16, 16, 5, 20, 7}, kv2[8] = {48, 10, 33, 32, 16, 16, 32, 7};
        const int32_t want1[15] = {50, 42, -1, 7, 23, 41, -1, -1, 8, -1, -1, 15, 16, -1, -1};
        const int32_t want2[15] = {50, 42, 4, 7, 23, 41, 99, -1, 8, 3, -1, 15, 16, -1, -1};
        int32_t pm[4], co[4], so[4], pages[15], rows[4];
        int64_t ip[5], ext = -1, starved = -1;
        tangram_tables g;
        memset(&g, 0, sizeof g);
        g.perm = pm, g.cluster_of = co, g.slot_of = so, g.tbl_indptr = ip, g.tbl_pages = pages, g.tbl_pages_cap = 15;
        g.headroom_pages = 2, g.row_pages = rows;
        CHECK(tangram_build_ragged_tables(Bg, res, 2, 4, 2, 16, fl, 11, 0u, NULL, &g) == TANGRAM_OK);
        CHECK(g.n_pages_used == 7 && g.n_slots == 15 && ip[4] == 15 && rows[0] == 1 && rows[1] == 3 && rows[3] == 2);
        CHECK(tangram_extend_tables(&g, kv1, fl, 11, 1, &ext, &starved) == TANGRAM_OK);
        CHECK(ext == 1 && starved == 0 && g.n_pages_used == 8 && memcmp(pages, want1, sizeof want1) == 0);
        CHECK(tangram_extend_tables(&g, kv2, fl, 11, 0, &ext, &starved) == TANGRAM_OK);
        CHECK(ext == 3 && starved == 1 && g.n_pages_used == 11 && memcmp(pages, want2, sizeof want2) == 0);
        CHECK(rows[0] == 3 && rows[1] == 4 && rows[2] == 2 && rows[3] == 2);
        g.row_pages = NULL;
        CHECK(tangram_extend_tables(&g, kv2, fl, 11, 0, NULL, NULL) == TANGRAM_ERR_INVALID_ARG);
    }
    printf("c_abi host path ok\n");
    return 0;
}
