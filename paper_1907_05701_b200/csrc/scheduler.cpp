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
            if (p == s) singles->push_back({s, s, s, s, s, s});
            else if (s < p) pairs->push_back({s, p, s, p, s, p});
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
        if (p == s) { singles->push_back({s, s, xs, xs, xs, xs}); continue; }
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
        pairs->push_back({s, p, xs, xp, out, out});
        after[s] = after[p] = out;
    }
    *w_slot = after;
}

}  // namespace hadpsgd

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
