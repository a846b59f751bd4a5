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

void matching_to_work(int S, const int32_t* partner, std::vector<WorkItem>* pairs,
                      std::vector<WorkItem>* singles) {
    pairs->clear();
    singles->clear();
    for (int s = 0; s < S; ++s) {
        if (partner[s] == s) singles->push_back({s, s});
        else if (s < partner[s]) pairs->push_back({s, partner[s]});
    }
}

}  // namespace hadpsgd

extern "C" int hadpsgd_pairing(int S, uint64_t step_k, int32_t* partner_out) {
    return hadpsgd::ring_partner(S, step_k, partner_out);
}
