// scheduler.cpp -- a1, the deterministic pairing scheduler (host only).
//
// Stands in for the asynchronous ADPSGD ring: every step each
// super-learner averages with its left or right ring neighbour.  Even step_k pairs
// (2i, 2i+1); odd step_k pairs (2i+1, (2i+2) mod S) (north_star (b)).  The matching is
// perfect, so T_k has exactly two 0.5s in every row and column; S odd > 1
// admits no perfect matching and is rejected (R8).
#include "internal.h"

namespace hadpsgd {

int ring_partner(int S, uint64_t step_k, int32_t* partner) {
    if (S < 1 || !partner) return HADPSGD_INVALID_ARG;
    if (S == 1) { partner[0] = 0; return HADPSGD_OK; }
    if (S & 1) return HADPSGD_INVALID_ARG;
    const int shift = static_cast<int>(step_k & 1);  // 0: (2i,2i+1)   1: (2i+1,2i+2)
    for (int i = 0; i < S / 2; ++i) {
        int a = (2 * i + shift) % S, b = (2 * i + 1 + shift) % S;
        partner[a] = b;
        partner[b] = a;
    }
    return HADPSGD_OK;
}

int validate_matching(int S, const int32_t* partner) {
    if (S < 1 || !partner) return HADPSGD_INVALID_ARG;
    for (int s = 0; s < S; ++s) {
        int p = partner[s];
        if (p < 0 || p >= S || partner[p] != s) return HADPSGD_INVALID_ARG;
    }
    return HADPSGD_OK;
}

void plan_unshare(int S, std::vector<int32_t>* w_slot, std::vector<SlotCopy>* copies) {
    std::vector<int> refs(S, 0);
    for (int s = 0; s < S; ++s) refs[(*w_slot)[s]]++;
    int next_free = 0;
    std::vector<char> seen(S, 0);
    for (int s = 0; s < S; ++s) {
        const int x = (*w_slot)[s];
        if (!seen[x]) { seen[x] = 1; continue; }      // the first member keeps the slot
        while (refs[next_free] != 0) ++next_free;       // exists: #free == #extra references
        copies->push_back({x, next_free});
        refs[next_free] = 1;
        (*w_slot)[s] = next_free;
    }
}

void plan_step(int S, const int32_t* partner, bool share, std::vector<int32_t>* w_slot,
               std::vector<WorkItem>* pairs, std::vector<WorkItem>* singles,
               std::vector<SlotCopy>* copies) {
    pairs->clear();
    singles->clear();
    copies->clear();
    if (!share) {
        for (int s = 0; s < S; ++s) {
            const int p = partner[s];
            if (p == s) singles->push_back({s, s, s, s, s, s, 0, 0});
            else if (s < p) pairs->push_back({s, p, s, p, s, p, 0, 0});
        }
        return;
    }
    bool has_single = false;
    for (int s = 0; s < S; ++s) has_single = has_single || partner[s] == s;
    if (has_single) plan_unshare(S, w_slot, copies);   // an unmixed member needs a slot of its own

    std::vector<int> refs(S, 0);
    for (int s = 0; s < S; ++s) refs[(*w_slot)[s]]++;
    std::vector<char> free_at_start(S, 0);
    for (int x = 0; x < S; ++x) free_at_start[x] = refs[x] == 0;
    int next_free = 0;
    std::vector<int32_t> after(*w_slot);
    for (int s = 0; s < S; ++s) {
        const int p = partner[s];
        const int xs = (*w_slot)[s];
        if (p == s) { singles->push_back({s, s, xs, xs, xs, xs, 0, 0}); continue; }
        if (p < s) continue;
        const int xp = (*w_slot)[p];
        // references to a slot from outside this pair
        const int outside_s = refs[xs] - 1 - (xp == xs ? 1 : 0);
        const int outside_p = refs[xp] - 1 - (xp == xs ? 1 : 0);
        int out;
        if (outside_s == 0) out = xs;
        else if (outside_p == 0) out = xp;
        else {
            while (!free_at_start[next_free]) ++next_free;
            out = next_free++;
        }
        pairs->push_back({s, p, xs, xp, out, out, 0, 0});
        after[s] = after[p] = out;
    }
    *w_slot = after;
}

int plan_peer_step(int world, int rank, const int32_t* rank_begin, const int32_t* partner, uint64_t epoch,
                   std::vector<int32_t>* pending, std::vector<WorkItem>* pairs, std::vector<WorkItem>* singles) {
    if (world < 1 || rank < 0 || rank >= world || !rank_begin || !partner || !pending) return HADPSGD_INVALID_ARG;
    const int S_g = rank_begin[world], lo = rank_begin[rank], hi = rank_begin[rank + 1];
    const int S_l = hi - lo;
    if (rank_begin[0] != 0 || S_l < 1 || static_cast<int>(pending->size()) != S_l) return HADPSGD_INVALID_ARG;
    if (validate_matching(S_g, partner) != HADPSGD_OK) return HADPSGD_INVALID_ARG;
    pairs->clear();
    singles->clear();
    const int rd = static_cast<int>((epoch + 1) & 1), wr = static_cast<int>(epoch & 1);   // stage parities
    auto read_of = [&](int sl, int32_t* a, int32_t* b) {
        const int32_t pend = (*pending)[sl];
        if (pend >= 0) { *a = S_l * (1 + rd) + sl; *b = 1 + rd * S_g + pend; }   // w = 1/2 (own stage + partner's)
        else { *a = sl; *b = 0; }
    };
    std::vector<int32_t> next(S_l, -1);
    for (int sl = 0; sl < S_l; ++sl) {
        const int sg = lo + sl, pg = partner[sg];
        int32_t a_s, b_s;
        read_of(sl, &a_s, &b_s);
        if (pg == sg) {                                   // unmixed: T_ss = 1
            singles->push_back({sl, sl, a_s, a_s, sl, sl, b_s, b_s});
        } else if (pg >= lo && pg < hi) {                 // both members live here: an ordinary pair
            if (pg < sg) continue;
            const int pl = pg - lo;
            int32_t a_p, b_p;
            read_of(pl, &a_p, &b_p);
            pairs->push_back({sl, pl, a_s, a_p, sl, pl, b_s, b_p});
        } else {                                          // partner in another arena: publish u, mix next step
            const int32_t o = S_l * (1 + wr) + sl;
            singles->push_back({sl, sl, a_s, a_s, o, o, b_s, b_s});
            next[sl] = pg;
        }
    }
    *pending = next;
    return HADPSGD_OK;
}

}  // namespace hadpsgd

// The peer plan of one step as a pure host function (what a peer-mode handle does internally), so the
// multi-rank data flow can be checked without GPUs.  Outputs, all [S_local] and indexed by the LOCAL
// member: kind (0 pair member, 1 unmixed, 2 straddling: publishes u), mate (local index of the pair
// mate, or -1), read_buf / write_buf (weight buffer index: main s, stage (e, s) = S_local (1 + e) + s),
// read_peer (-1, or e * S_global + global partner: the stage buffer averaged with read_buf first).
extern "C" int hadpsgd_plan_peer(int world, int rank, const int32_t* rank_begin, const int32_t* partner,
                                 uint64_t epoch, int32_t* pending, int32_t* kind, int32_t* mate,
                                 int32_t* read_buf, int32_t* write_buf, int32_t* read_peer) {
    using namespace hadpsgd;
    if (world < 1 || rank < 0 || rank >= world || !rank_begin || !partner || !pending || !kind || !mate || !read_buf ||
        !write_buf || !read_peer)
        return HADPSGD_INVALID_ARG;
    for (int r = 0; r < world; ++r) if (rank_begin[r + 1] <= rank_begin[r]) return HADPSGD_INVALID_ARG;
    const int S_l = rank_begin[rank + 1] - rank_begin[rank];
    std::vector<int32_t> pend(pending, pending + S_l);
    std::vector<WorkItem> pairs, singles;
    int rc = plan_peer_step(world, rank, rank_begin, partner, epoch, &pend, &pairs, &singles);
    if (rc != HADPSGD_OK) return rc;
    for (const WorkItem& it : pairs) {
        kind[it.s] = kind[it.p] = 0; mate[it.s] = it.p; mate[it.p] = it.s;
        read_buf[it.s] = it.ws; read_buf[it.p] = it.wp; write_buf[it.s] = it.wo_s; write_buf[it.p] = it.wo_p;
        read_peer[it.s] = it.b_s - 1; read_peer[it.p] = it.b_p - 1;
    }
    for (const WorkItem& it : singles) {
        kind[it.s] = pend[it.s] >= 0 ? 2 : 1; mate[it.s] = -1;
        read_buf[it.s] = it.ws; write_buf[it.s] = it.wo_s; read_peer[it.s] = it.b_s - 1;
    }
    for (int s = 0; s < S_l; ++s) pending[s] = pend[s];
    return HADPSGD_OK;
}

extern "C" int hadpsgd_plan_slots(int S, const int32_t* partner, int share, int32_t* w_slot, int32_t* read_slot,
                                  int32_t* write_slot, int32_t* copy_src, int32_t* copy_dst, int32_t* n_copies) {
    using namespace hadpsgd;
    if (S < 1 || S > HADPSGD_MAX_S || !partner || !w_slot || !read_slot || !write_slot || !copy_src || !copy_dst ||
        !n_copies || validate_matching(S, partner) != HADPSGD_OK)
        return HADPSGD_INVALID_ARG;
    for (int s = 0; s < S; ++s) if (w_slot[s] < 0 || w_slot[s] >= S) return HADPSGD_INVALID_ARG;
    std::vector<int32_t> slot(w_slot, w_slot + S);
    std::vector<WorkItem> pairs, singles;
    std::vector<SlotCopy> copies;
    plan_step(S, partner, share != 0, &slot, &pairs, &singles, &copies);
    for (const WorkItem& it : pairs) {
        read_slot[it.s] = it.ws; read_slot[it.p] = it.wp; write_slot[it.s] = it.wo_s; write_slot[it.p] = it.wo_p;
    }
    for (const WorkItem& it : singles) { read_slot[it.s] = it.ws; write_slot[it.s] = it.wo_s; }
    *n_copies = static_cast<int32_t>(copies.size());
    for (size_t i = 0; i < copies.size(); ++i) { copy_src[i] = copies[i].src; copy_dst[i] = copies[i].dst; }
    for (int s = 0; s < S; ++s) w_slot[s] = slot[s];
    return HADPSGD_OK;
}

extern "C" int hadpsgd_pairing(int S, uint64_t step_k, int32_t* partner_out) {
    return hadpsgd::ring_partner(S, step_k, partner_out);
}
