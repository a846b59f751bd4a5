"""Host logic of HADPSGD_SHARE_PAIR_WEIGHTS (no GPU): the slot planner behind hadpsgd_step*.

Both members of a pair end a step with identical weights (R3), so they may share one
of the S weight buffers.  The planner must guarantee, for ANY sequence of matchings, that
  * no buffer written in a step is read by a different work item of that step (the kernel runs
    all items concurrently and updates in place),
  * different items write different buffers,
  * reading through the slots gives exactly what per-learner buffers would give.
The last point is checked by simulating the storage with tokens instead of weights."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def H():
    from paper_1907_05701_b200 import build as b
    b.build()
    import paper_1907_05701_b200 as m
    return m


def simulate(H, S, matchings, share=True):
    """Run the planner over a sequence of matchings.  `ref[s]` is the token learner s would hold
    with one private buffer each; `store[x]` is what slot x holds; they must always agree."""
    slot = list(range(S))
    store = [("init", s) for s in range(S)]
    ref = [("init", s) for s in range(S)]
    for k, partner in enumerate(matchings):
        slot_after, rd, wr, copies = H.hadpsgd_plan_slots(partner, slot, share)
        for src, dst in copies:                                  # un-sharing copies run first
            assert dst not in slot, "copy target is still in use"
            store[dst] = store[src]
        # after the copies the planner's own view of "where w_s is" is rd[s]
        for s in range(S):
            assert store[rd[s]] == ref[s], (k, s)
        items = {}
        for s in range(S):
            items.setdefault(frozenset((s, partner[s])), []).append(s)
        writes = {}
        for members in items.values():
            outs = {wr[s] for s in members}
            for x in outs:
                assert x not in writes, "two items write the same buffer"
                writes[x] = members
        for x, members in writes.items():                        # in-place safety
            readers = [s for s in range(S) if rd[s] == x and s not in members]
            assert not readers, (k, x, members, readers)
        new_store = list(store)
        for members in items.values():
            if len(members) == 2:
                a, b = sorted(members)
                tok = ("mix", k, ref[a], ref[b])
                assert wr[a] == wr[b] or not share
            else:
                a = members[0]
                tok = ("upd", k, ref[a])
            for s in members:
                new_store[wr[s]] = tok
                ref[s] = tok
        store = new_store
        slot = slot_after
        assert all(slot[s] == wr[s] for s in range(S))
        for s in range(S):
            assert store[slot[s]] == ref[s]
    return slot


def ring(H, S, k):
    return H.hadpsgd_pairing(S, k)


@pytest.mark.parametrize("S", [2, 4, 6, 8, 16, 64, 512])
def test_ring_schedule_is_periodic_and_safe(H, S):
    slots = []
    slot = list(range(S))
    for k in range(6):
        slot, rd, wr, copies = H.hadpsgd_plan_slots(ring(H, S, k), slot)
        assert not copies
        slots.append(list(slot))
    assert slots[0] == slots[2] == slots[4] and slots[1] == slots[3] == slots[5]   # period 2 from step 0 on
    simulate(H, S, [ring(H, S, k) for k in range(7)])
    simulate(H, S, [ring(H, S, k) for k in (0, 0, 1, 1, 1, 0, 3, 2)])               # replayed parities


def test_identity_without_sharing(H):
    S = 8
    slot, rd, wr, copies = H.hadpsgd_plan_slots(ring(H, S, 1), list(range(S)), share=False)
    assert slot == rd == wr == list(range(S)) and not copies


def test_random_matchings_including_unpaired_members(H):
    from hypothesis import given, settings, strategies as st

    @st.composite
    def matching_seq(draw):
        S = draw(st.integers(1, 24))
        seq = []
        for _ in range(draw(st.integers(1, 8))):
            perm = draw(st.permutations(list(range(S))))
            n_pairs = draw(st.integers(0, S // 2))
            partner = list(range(S))
            for i in range(n_pairs):
                a, b = perm[2 * i], perm[2 * i + 1]
                partner[a], partner[b] = b, a
            seq.append(partner)
        return S, seq

    @settings(max_examples=300, deadline=None)
    @given(matching_seq())
    def check(arg):
        S, seq = arg
        simulate(H, S, seq)

    check()


def test_plan_slots_rejects_bad_input(H):
    with pytest.raises(H.HadpsgdError):
        H.hadpsgd_plan_slots([1, 2, 0], [0, 1, 2])          # not a matching
    with pytest.raises(H.HadpsgdError):
        H.hadpsgd_plan_slots([1, 0], [0, 5])                # slot out of range
