"""Super-learner partition (row f4; Fig. 3) without GPUs.

The product's peer planner (hadpsgd_plan_peer, a pure host function of libhadpsgd.so) decides, for
every rank and step, which weight buffer each local member reads, which partner stage buffer it
averages in first, and where it writes.  Here the DATA FLOW it prescribes is executed on numpy
buffers -- one set of buffers per rank, a member may only touch its own rank's buffers plus the stage
buffers of other ranks it is told to read -- with the per-member arithmetic taken from the oracle
(S = 1 / S = 2 oracle calls), and the result is compared with the oracle run on all S_global
super-learners at once.  That checks planning and pointer exchange: the stage parities, that nobody
reads a buffer that is being written in the same epoch, that both owners of a straddling pair resolve
the same mix, that flush materialises it.

The second test does the same across two real processes over gloo (world_size 2): stage buffers
travel by send/recv where the GPUs would read each other's memory.
"""
import os
import socket

import numpy as np
import pytest

LR, MU = 0.1, 0.9
G, P = 2, 257


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


@pytest.fixture(scope="module")
def H():
    from paper_1907_05701_b200 import build as b
    b.build()
    import paper_1907_05701_b200 as m
    return m


class Rank:
    """One rank's buffers: main weights, momentum, 2 x S_l stage buffers, pending table."""

    def __init__(self, r, rank_begin, w, v):
        self.r, self.lo, self.hi = r, rank_begin[r], rank_begin[r + 1]
        self.S_l = self.hi - self.lo
        self.main = w[self.lo:self.hi].copy()
        self.v = v[self.lo:self.hi].copy()
        self.stage = np.full((2, self.S_l, w.shape[1]), np.nan, np.float32)    # NaN: must be written before read
        self.pending = [-1] * self.S_l
        self.writing = set()                 # (parity, local s) written in the current epoch

    def buf(self, idx):
        if idx < self.S_l:
            return self.main[idx]
        e, s = divmod(idx - self.S_l, self.S_l)
        return self.stage[e, s]


def run_epoch(H, oracle_mod, ranks, rank_begin, partner, epoch, grads, read_remote):
    """One step of every rank, following hadpsgd_plan_peer.  read_remote(r, e, s_global) returns the
    stage buffer of a member owned by another rank AS IT WAS AT THE EPOCH BARRIER."""
    world, S_g = len(ranks), rank_begin[-1]
    snap = [rk.stage.copy() for rk in ranks]            # what a peer read sees: the state at the barrier
    for rk in ranks:
        rk.writing = set()
        plan = H.hadpsgd_plan_peer(world, rk.r, rank_begin, partner, epoch, rk.pending)
        new_main, new_stage = rk.main.copy(), rk.stage.copy()
        w_in = []
        for s in range(rk.S_l):                         # resolve what every member's weights ARE
            a = rk.buf(plan["read_buf"][s]).copy()
            if plan["read_buf"][s] >= rk.S_l:           # own stage: must be the parity written last epoch
                e = (plan["read_buf"][s] - rk.S_l) // rk.S_l
                assert e == (epoch + 1) % 2
            if plan["read_peer"][s] >= 0:
                e, sg = divmod(plan["read_peer"][s], S_g)
                assert e == (epoch + 1) % 2 and not (rk.lo <= sg < rk.hi) and sg == rk.pending[s]
                b = read_remote(rk.r, e, sg, snap)
                a = np.float32(0.5) * (a + b)           # the pending mix (fp32 add, exact halving)
            else:
                assert rk.pending[s] < 0
            assert not np.isnan(a).any(), "read a stage buffer nobody wrote"
            w_in.append(a)
        done = set()
        for s in range(rk.S_l):
            if s in done:
                continue
            kind, mate = plan["kind"][s], plan["mate"][s]
            members = [s, mate] if kind == 0 else [s]
            w = np.stack([w_in[m] for m in members])
            v = np.stack([rk.v[m] for m in members])
            g = np.ascontiguousarray(np.stack([grads[rk.lo + m] for m in members]))
            oracle_mod.step(g, w, v, LR, MU, 0)          # S = 2: one pair; S = 1: u = w - lr v'
            for i, m in enumerate(members):
                rk.v[m] = v[i]
                wb = plan["write_buf"][m]
                if kind == 2:
                    e, ss = divmod(wb - rk.S_l, rk.S_l)
                    assert wb >= rk.S_l and e == epoch % 2 and ss == m
                    new_stage[e, ss] = w[i]
                    rk.writing.add((e, ss))
                else:
                    assert wb == m
                    new_main[m] = w[i]
                done.add(m)
        rk.main, rk.stage, rk.pending = new_main, new_stage, plan["pending"]


def flush(ranks, rank_begin, epoch):
    S_g = rank_begin[-1]
    snap = [rk.stage.copy() for rk in ranks]
    rd = (epoch + 1) % 2
    for rk in ranks:
        for s in range(rk.S_l):
            if rk.pending[s] >= 0:
                sg = rk.pending[s]
                owner = next(r for r in range(len(ranks)) if rank_begin[r] <= sg < rank_begin[r + 1])
                b = snap[owner][rd, sg - rank_begin[owner]]
                rk.main[s] = np.float32(0.5) * (rk.stage[rd, s] + b)
                rk.pending[s] = -1


def local_read(ranks, rank_begin):
    def read(r, e, sg, snap):
        owner = next(q for q in range(len(ranks)) if rank_begin[q] <= sg < rank_begin[q + 1])
        assert owner != r
        return snap[owner][e, sg - rank_begin[owner]]
    return read


def ring(S, k):
    p = [0] * S
    sh = k % 2
    for i in range(S // 2):
        a, b = (2 * i + sh) % S, (2 * i + 1 + sh) % S
        p[a], p[b] = b, a
    return p


SPLITS = [[0, 2, 4, 6, 8], [0, 1, 2, 3, 4], [0, 3, 5, 8], [0, 8], [0, 1, 8], [0, 4, 8]]


@pytest.mark.parametrize("rank_begin", SPLITS)
def test_ring_schedule_over_ranks_equals_single_arena_oracle(H, oracle_mod, rank_begin):
    S = rank_begin[-1]
    rng = np.random.default_rng(S + len(rank_begin))
    w = (rng.standard_normal((S, P)) * 0.05).astype(np.float32)
    v = (rng.standard_normal((S, P)) * 0.01).astype(np.float32)
    ranks = [Rank(r, rank_begin, w, v) for r in range(len(rank_begin) - 1)]
    ow, ov = w.copy(), v.copy()
    for k in range(7):
        g = (rng.standard_normal((S, G, P)) * 1e-3).astype(np.float32)
        run_epoch(H, oracle_mod, ranks, rank_begin, ring(S, k), k, g, local_read(ranks, rank_begin))
        oracle_mod.step(g, ow, ov, LR, MU, k)
        gv = np.concatenate([rk.v for rk in ranks])
        assert np.array_equal(bits(gv), bits(ov)), k
        # members whose mix is not pending already hold the oracle's weights
        for rk in ranks:
            for s in range(rk.S_l):
                if rk.pending[s] < 0:
                    assert np.array_equal(bits(rk.main[s]), bits(ow[rk.lo + s])), (k, rk.r, s)
    flush(ranks, rank_begin, 7)
    gw = np.concatenate([rk.main for rk in ranks])
    assert np.array_equal(bits(gw), bits(ow))
    assert all(p < 0 for rk in ranks for p in rk.pending)


def test_custom_matchings_unmixed_members_and_mid_run_flush(H, oracle_mod):
    rank_begin = [0, 3, 4, 7]                      # uneven ranks, odd S_global
    S = 7
    matchings = [[3, 1, 5, 0, 4, 2, 6], [1, 0, 3, 2, 5, 4, 6], [6, 2, 1, 4, 3, 5, 0], [0, 1, 2, 3, 4, 5, 6],
                 [4, 5, 6, 3, 0, 1, 2], [4, 5, 6, 3, 0, 1, 2], [1, 0, 2, 6, 5, 4, 3]]
    rng = np.random.default_rng(5)
    w = (rng.standard_normal((S, P)) * 0.05).astype(np.float32)
    v = np.zeros((S, P), np.float32)
    ranks = [Rank(r, rank_begin, w, v) for r in range(3)]
    ow, ov = w.copy(), v.copy()
    epoch = 0
    for k, partner in enumerate(matchings):
        g = (rng.standard_normal((S, G, P)) * 1e-3).astype(np.float32)
        run_epoch(H, oracle_mod, ranks, rank_begin, partner, epoch, g, local_read(ranks, rank_begin))
        epoch += 1
        oracle_mod.step(g, ow, ov, LR, MU, k, partner=partner)
        if k in (2, 4):                            # a flush between steps does not advance the epoch
            flush(ranks, rank_begin, epoch)
            assert np.array_equal(bits(np.concatenate([rk.main for rk in ranks])), bits(ow)), k
    flush(ranks, rank_begin, epoch)
    assert np.array_equal(bits(np.concatenate([rk.main for rk in ranks])), bits(ow))
    assert np.array_equal(bits(np.concatenate([rk.v for rk in ranks])), bits(ov))


def test_plan_peer_structure_and_errors(H):
    rank_begin = [0, 2, 4, 6, 8]
    # odd ring step: every member's partner lives next door -> all straddle, all publish into stage[e & 1]
    for epoch in (0, 1, 6):
        d = H.hadpsgd_plan_peer(4, 1, rank_begin, ring(8, 1), epoch, [-1, -1])
        assert d["kind"] == [2, 2] and d["pending"] == [1, 4] and d["mate"] == [-1, -1]
        assert d["read_buf"] == [0, 1] and d["read_peer"] == [-1, -1]
        assert d["write_buf"] == [2 * (1 + epoch % 2) + 0, 2 * (1 + epoch % 2) + 1]
    # the even step after it: a local pair whose two members first resolve their pending mixes
    d = H.hadpsgd_plan_peer(4, 1, rank_begin, ring(8, 0), 1, [1, 4])
    assert d["kind"] == [0, 0] and d["mate"] == [1, 0] and d["pending"] == [-1, -1]
    assert d["read_buf"] == [2, 3] and d["write_buf"] == [0, 1]            # stage parity 0, then main
    assert d["read_peer"] == [0 * 8 + 1, 0 * 8 + 4]
    # one rank holding everything never straddles
    d = H.hadpsgd_plan_peer(1, 0, [0, 8], ring(8, 1), 3, [-1] * 8)
    assert set(d["kind"]) == {0} and d["pending"] == [-1] * 8 and d["read_peer"] == [-1] * 8
    for bad in (dict(world=4, rank=4), dict(partner=[1, 2, 0, 3, 4, 5, 6, 7]), dict(rank_begin=[0, 2, 2, 6, 8]),
                dict(rank_begin=[1, 2, 4, 6, 8])):
        args = dict(world=4, rank=1, rank_begin=rank_begin, partner=ring(8, 1))
        args.update(bad)
        with pytest.raises(H.HadpsgdError):
            H.hadpsgd_plan_peer(args["world"], args["rank"], args["rank_begin"], args["partner"], 0, [-1, -1])


# ------------------------------------------------------------------ two processes over gloo

def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _gloo_worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    import oracle
    import paper_1907_05701_b200 as Hm
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        S, steps = 8, 6
        rank_begin = [0, 4, 8] if world == 2 else [0, 8]
        rng = np.random.default_rng(99)                      # every rank draws the same global problem
        w = (rng.standard_normal((S, P)) * 0.05).astype(np.float32)
        v = np.zeros((S, P), np.float32)
        me = Rank(rank, rank_begin, w, v)
        other = 1 - rank
        for k in range(steps):
            g = (rng.standard_normal((S, G, P)) * 1e-3).astype(np.float32)
            # EPOCH BARRIER + exchange: each rank hands the other a copy of its stage region (what a peer
            # read over NVLink would see after the barrier)
            mine = torch.from_numpy(me.stage.copy())
            theirs = torch.empty_like(mine)
            reqs = [dist.isend(mine, other), dist.irecv(theirs, other)]
            for q in reqs:
                q.wait()
            remote = theirs.numpy()

            def read(r, e, sg, snap):
                assert rank_begin[other] <= sg < rank_begin[other + 1]
                return remote[e, sg - rank_begin[other]]
            run_epoch(Hm, oracle, _one(me, world), rank_begin, ring(S, k), k, g, read)
        # final flush needs the partner's stage once more
        mine = torch.from_numpy(me.stage.copy())
        theirs = torch.empty_like(mine)
        for q in [dist.isend(mine, other), dist.irecv(theirs, other)]:
            q.wait()
        rd = (steps + 1) % 2
        for s in range(me.S_l):
            if me.pending[s] >= 0:
                me.main[s] = np.float32(0.5) * (me.stage[rd, s] + theirs.numpy()[rd, me.pending[s] - rank_begin[other]])
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), w=me.main, v=me.v)
    finally:
        dist.destroy_process_group()


class _one(list):
    """run_epoch iterates over `ranks` and takes len(ranks) as the world size: a list that yields only
    this process's rank but reports the real world size."""

    def __init__(self, rk, world):
        super().__init__([rk])
        self.world = world

    def __len__(self):
        return self.world


@pytest.mark.timeout(300)
def test_two_processes_over_gloo_equal_single_arena_oracle(tmp_path, oracle_mod, H):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_gloo_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    S, steps = 8, 6
    rng = np.random.default_rng(99)
    ow = (rng.standard_normal((S, P)) * 0.05).astype(np.float32)
    ov = np.zeros((S, P), np.float32)
    for k in range(steps):
        g = (rng.standard_normal((S, G, P)) * 1e-3).astype(np.float32)
        oracle_mod.step(g, ow, ov, LR, MU, k)
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert np.array_equal(bits(np.concatenate([p["w"] for p in parts])), bits(ow))
    assert np.array_equal(bits(np.concatenate([p["v"] for p in parts])), bits(ov))
