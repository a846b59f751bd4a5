/* abi_host_check.c -- plain C99 client of include/hadpsgd.h (proves the header is C, not C++) that
 * exercises the host-only entry points: allocator (a0), pairing scheduler (a1), shard split and
 * the LR recipe.  tests/test_host_runtime_c.py builds it twice: against libhadpsgd.so, and
 * together with the host sources under -fsanitize=address,undefined.  Prints "ok" or aborts. */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "hadpsgd.h"

#define CHECK(c) do { if (!(c)) { fprintf(stderr, "FAILED %s:%d: %s\n", __FILE__, __LINE__, #c); return 1; } } while (0)

int main(void) {
    /* a1: every even S up to the maximum, both parities: a perfect matching of ring neighbours */
    static int32_t partner[HADPSGD_MAX_S];
    int S, s;
    uint64_t k;
    for (S = 2; S <= HADPSGD_MAX_S; S += 2) {
        for (k = 0; k < 4; ++k) {
            CHECK(hadpsgd_pairing(S, k, partner) == HADPSGD_OK);
            for (s = 0; s < S; ++s) {
                int p = partner[s], d = ((p - s) % S + S) % S;
                CHECK(p >= 0 && p < S && p != s && partner[p] == s);
                CHECK(d == 1 || d == S - 1);
                if (k % 2 == 0) CHECK(p == (s ^ 1));
            }
        }
    }
    CHECK(hadpsgd_pairing(1, 0, partner) == HADPSGD_OK && partner[0] == 0);
    CHECK(hadpsgd_pairing(3, 0, partner) == HADPSGD_INVALID_ARG);
    CHECK(hadpsgd_pairing(0, 0, partner) == HADPSGD_INVALID_ARG);
    CHECK(hadpsgd_pairing(4, 0, NULL) == HADPSGD_INVALID_ARG);

    /* a0: a ragged table; offsets aligned and non-overlapping, regions ordered and aligned */
    {
        enum { N = 9 };
        const int64_t seg[N] = {1, 63, 64, 65, 1000003, 7, 4096, 129, 2};
        int64_t off[N], P = 0, expect = 0;
        size_t w = 0, v = 0, g = 0, wb = 0, need = 0, need_emit = 0;
        hadpsgd_dtypes dt;
        int i;
        memset(&dt, 0, sizeof dt);
        dt.grad_dtype = HADPSGD_BF16;
        CHECK(hadpsgd_layout(6, 3, seg, N, dt, off, &P, &w, &v, &g, &wb) == HADPSGD_OK);
        for (i = 0; i < N; ++i) {
            CHECK(off[i] == expect && off[i] % HADPSGD_SEG_ALIGN_ELEMS == 0);
            expect += (seg[i] + HADPSGD_SEG_ALIGN_ELEMS - 1) / HADPSGD_SEG_ALIGN_ELEMS * HADPSGD_SEG_ALIGN_ELEMS;
        }
        CHECK(P == expect);
        CHECK(w == 0 && v >= (size_t)6 * P * 4 && g >= v + (size_t)6 * P * 4 && v % 256 == 0 && g % 256 == 0);
        CHECK(hadpsgd_required_bytes(6, 3, seg, N, dt, &need) == HADPSGD_OK);
        CHECK(need >= g + (size_t)18 * P * 2);
        dt.working_dtype = HADPSGD_BF16;
        CHECK(hadpsgd_required_bytes(6, 3, seg, N, dt, &need_emit) == HADPSGD_OK);
        CHECK(need_emit >= need + (size_t)6 * P * 2 && need_emit < need + (size_t)6 * P * 2 + 512);
        CHECK(hadpsgd_layout(6, 3, seg, N, dt, NULL, NULL, NULL, NULL, NULL, &wb) == HADPSGD_OK);
        CHECK(wb >= g + (size_t)18 * P * 2 && wb % 256 == 0);
        dt.master_dtype = HADPSGD_BF16;
        CHECK(hadpsgd_required_bytes(6, 3, seg, N, dt, &need) == HADPSGD_INVALID_ARG);
        dt.master_dtype = HADPSGD_F32;
        CHECK(hadpsgd_required_bytes(6, 3, seg, 0, dt, &need) == HADPSGD_INVALID_ARG);
        CHECK(hadpsgd_required_bytes(6, 3, NULL, N, dt, &need) == HADPSGD_INVALID_ARG);
        CHECK(hadpsgd_required_bytes(6, 3, seg, N, dt, NULL) == HADPSGD_INVALID_ARG);
    }

    /* f4: stage buffers of the super-learner partition sit right behind the S weight buffers */
    {
        const int64_t seg[2] = {1000, 77};
        size_t w = 0, v = 0, v_peer = 0, need = 0, need_peer = 0;
        int64_t P = 0;
        hadpsgd_dtypes dt;
        memset(&dt, 0, sizeof dt);
        CHECK(hadpsgd_layout(4, 2, seg, 2, dt, NULL, &P, &w, &v, NULL, NULL) == HADPSGD_OK);
        CHECK(hadpsgd_required_bytes(4, 2, seg, 2, dt, &need) == HADPSGD_OK);
        dt.peer_stage = 1;
        CHECK(hadpsgd_layout(4, 2, seg, 2, dt, NULL, NULL, &w, &v_peer, NULL, NULL) == HADPSGD_OK);
        CHECK(hadpsgd_required_bytes(4, 2, seg, 2, dt, &need_peer) == HADPSGD_OK);
        CHECK(w == 0 && v >= (size_t)4 * P * 4 && v_peer >= (size_t)12 * P * 4);
        CHECK(need_peer >= need + (size_t)8 * P * 4 && need_peer < need + (size_t)8 * P * 4 + 512);
        dt.working_dtype = HADPSGD_BF16;
        CHECK(hadpsgd_required_bytes(4, 2, seg, 2, dt, &need) == HADPSGD_INVALID_ARG);
        dt.working_dtype = HADPSGD_F32; dt.peer_stage = 2;
        CHECK(hadpsgd_required_bytes(4, 2, seg, 2, dt, &need) == HADPSGD_INVALID_ARG);
    }

    /* f4: the peer planner over 4 ranks of 2 (the paper's 8 x 2 in small), ring schedule: odd steps leave
     * every member pending on its neighbour, even steps resolve both members of the local pair */
    {
        const int32_t rank_begin[5] = {0, 2, 4, 6, 8};
        int32_t partner[8], pending[2] = {-1, -1}, kind[2], mate[2], rd[2], wr[2], peer[2];
        int rank;
        uint64_t epoch;
        for (rank = 0; rank < 4; ++rank) {
            pending[0] = pending[1] = -1;
            for (epoch = 0; epoch < 6; ++epoch) {
                CHECK(hadpsgd_pairing(8, epoch, partner) == HADPSGD_OK);
                CHECK(hadpsgd_plan_peer(4, rank, rank_begin, partner, epoch, pending, kind, mate, rd, wr, peer) == HADPSGD_OK);
                if (epoch % 2 == 0) {
                    CHECK(kind[0] == 0 && kind[1] == 0 && mate[0] == 1 && mate[1] == 0 && wr[0] == 0 && wr[1] == 1);
                    CHECK(pending[0] == -1 && pending[1] == -1);
                    CHECK(epoch == 0 ? (peer[0] == -1 && rd[0] == 0) : (peer[0] >= 8 && rd[0] == 4 && rd[1] == 5));
                } else {
                    CHECK(kind[0] == 2 && kind[1] == 2 && wr[0] == 4 && wr[1] == 5 && rd[0] == 0 && peer[0] == -1);
                    CHECK(pending[0] == (2 * rank + 7) % 8 && pending[1] == (2 * rank + 2) % 8);
                }
            }
        }
        partner[0] = 0; partner[1] = 0;                      /* not a matching */
        CHECK(hadpsgd_plan_peer(4, 0, rank_begin, partner, 0, pending, kind, mate, rd, wr, peer) == HADPSGD_INVALID_ARG);
        CHECK(hadpsgd_plan_peer(4, 4, rank_begin, partner, 0, pending, kind, mate, rd, wr, peer) == HADPSGD_INVALID_ARG);
    }

    /* shared pair slots: the ring schedule becomes periodic after the first step */
    {
        int32_t partner[8], slot[8], rd[8], wr[8], cs[8], cd[8], n = 0, first[8];
        int s, k;
        for (s = 0; s < 8; ++s) slot[s] = s;
        for (k = 0; k < 7; ++k) {
            CHECK(hadpsgd_pairing(8, (uint64_t)k, partner) == HADPSGD_OK);
            CHECK(hadpsgd_plan_slots(8, partner, 1, slot, rd, wr, cs, cd, &n) == HADPSGD_OK && n == 0);
            for (s = 0; s < 8; ++s) CHECK(slot[s] == slot[partner[s]] && wr[s] == slot[s]);
            if (k == 1) memcpy(first, slot, sizeof first);
            if (k == 3 || k == 5) CHECK(memcmp(first, slot, sizeof first) == 0);
        }
    }

    /* f4: shard ranges tile the buffer for every world size */
    {
        int world, r;
        for (world = 1; world <= 16; ++world) {
            int64_t P = 64 * 1000003LL, prev = 0, lo, hi;
            for (r = 0; r < world; ++r) {
                CHECK(hadpsgd_shard_range(P, world, r, &lo, &hi) == HADPSGD_OK);
                CHECK(lo == prev && hi >= lo && lo % 64 == 0);
                prev = hi;
            }
            CHECK(prev == P);
        }
    }

    /* f3: PAPER.md:70 example, 0.1 -> 1.0 over 10 epochs for batch 256 -> 2560 */
    {
        double lr = 0;
        int e;
        for (e = 1; e <= 10; ++e) {
            CHECK(hadpsgd_lr_schedule(0.1, 256, 2560, 10, e, &lr) == HADPSGD_OK);
            CHECK(lr > 0.1 * e - 1e-12 && lr < 0.1 * e + 1e-12);
        }
        CHECK(hadpsgd_lr_schedule(0.1, 256, 2560, 10, 12, &lr) == HADPSGD_OK && lr > 0.5 - 1e-12 && lr < 0.5 + 1e-12);
        CHECK(hadpsgd_lr_schedule(0.1, 256, 2560, 10, 0, &lr) == HADPSGD_INVALID_ARG);
    }
    CHECK(strcmp(hadpsgd_error_string(HADPSGD_OK), "ok") == 0);
    printf("ok\n");
    return 0;
}
