"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  All tests here need a B200 (-m gpu).

Bars (north_star):  DETERMINISTIC mode -> w and v bit-exact.  Default mode ->
|d| <= 1e-6 + 1e-5 |x| per element.  Diagnostics -> relative 1e-4 (reduction order is free).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

LR, MU = 0.1, 0.9


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def H(torch_cuda):
    import paper_1907_05701_b200 as m
    m.lib()                      # fail loudly if the extension is missing
    return m


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


def run_both(H, oracle_mod, S, G, seg_len, steps, *, bf16=False, flags=0, seed=11, dist="normal",
             matching=None, lr=LR, mu=MU, check_diag=True, v0_sd=0.0, blocks_per_sm=0):
    """Run `steps` steps on the GPU and in the oracle over the WHOLE (small) problem and return
    (gpu_w, gpu_v, ora_w, ora_v) in natural order; asserts diagnostics on the way."""
    import torch
    from fixtures import generator as gen
    from fixtures import problem
    exact = bool(flags & H.DETERMINISTIC)
    h = H.Hadpsgd(S, G, seg_len, H.BF16 if bf16 else H.F32, flags)
    if blocks_per_sm:
        h.hadpsgd_set_launch(blocks_per_sm)
    P = int(sum(seg_len))
    problem.fill_weights(h, seed)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    nat = torch.from_numpy(h.natural_index()).cuda()
    if v0_sd:
        for s in range(S):
            v0 = gen.normal_f32(gen.stream_key(seed, gen.STREAM_MOMENTUM, 0, s, 0), 0, P, v0_sd)
            ov[s] = v0
            h.hadpsgd_momentum(s)[nat] = torch.from_numpy(v0).cuda()
    oflags = 0
    if flags & H.NO_MIX: oflags |= oracle_mod.NO_MIX
    if flags & H.EQ7_LITERAL: oflags |= oracle_mod.EQ7_LITERAL
    for k in range(steps):
        problem.fill_grads(h, seed, k, dist)
        og = problem.host_grads(seed, k, S, G, 0, P, dist, bf16=bf16)
        if matching is not None:
            h.hadpsgd_step_matching(lr, mu, k, matching(k))
            od = oracle_mod.step(og, ow, ov, lr, mu, k, flags=oflags & ~oracle_mod.NO_MIX, diag=True, partner=matching(k))
        else:
            h.hadpsgd_step(lr, mu, k)
            od = oracle_mod.step(og, ow, ov, lr, mu, k, flags=oflags, diag=True)
        if check_diag and not (flags & H.NO_DIAG):
            assert_diag(h.hadpsgd_diagnostics(), od, k)
    torch.cuda.synchronize()
    gw = np.stack([h.hadpsgd_weights(s)[nat].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[nat].cpu().numpy() for s in range(S)])
    # padding must still be zero
    if h.P_padded != P:
        mask = torch.ones(h.P_padded, dtype=torch.bool, device="cuda"); mask[nat] = False
        for s in range(S):
            assert not h.hadpsgd_weights(s)[mask].any() and not h.hadpsgd_momentum(s)[mask].any()
    h.close()
    return gw, gv, ow, ov


def assert_diag(gd, od, k=0):
    """a5 against the oracle's double accumulators (R14, R16): relative 1e-4; a gap the
    oracle reports as exactly 0 (unmixed member) must be exactly 0 on the GPU too."""
    for name in ("gsq", "wsq", "gap"):
        assert np.allclose(gd[name], od[name], rtol=1e-4, atol=1e-30), (name, k, gd[name], od[name])
    assert np.array_equal(gd["gap"] == 0.0, od["gap"] == 0.0), (k, gd["gap"], od["gap"])


def assert_parity(gw, gv, ow, ov, exact):
    if exact:
        assert np.array_equal(bits(gw), bits(ow)), f"w differs in {np.sum(bits(gw) != bits(ow))} elements"
        assert np.array_equal(bits(gv), bits(ov)), f"v differs in {np.sum(bits(gv) != bits(ov))} elements"
    else:
        assert np.all(np.abs(gw - ow) <= 1e-6 + 1e-5 * np.abs(ow)), np.max(np.abs(gw - ow))
        assert np.all(np.abs(gv - ov) <= 1e-6 + 1e-5 * np.abs(ov)), np.max(np.abs(gv - ov))


# ------------------------------------------------------------------------------- fixtures

def test_device_generator_matches_host(torch_cuda):
    torch = torch_cuda
    from fixtures import device, generator as gen
    key = gen.stream_key(5, gen.STREAM_GRAD, 3, 2, 1)
    n, off = 100_003, 1_234_567_891
    for dist, scale in (("normal", 1e-3), ("uniform", 1e-3), ("normal", 0.05)):
        t = torch.empty(n, dtype=torch.float32, device="cuda")
        device.fill(t, key, dist, scale, elem_offset=off)
        ref = gen.normal_f32(key, off, n, scale) if dist == "normal" else gen.uniform_f32(key, off, n, scale)
        assert np.array_equal(bits(t.cpu().numpy()), bits(ref))
    tb = torch.empty(n, dtype=torch.bfloat16, device="cuda")
    device.fill(tb, key, "normal", 1e-3, elem_offset=off)
    assert np.array_equal(tb.view(torch.int16).cpu().numpy().view(np.uint16), gen.normal_bf16(key, off, n, 1e-3))


# ------------------------------------------------------------------------------- config 0: Tiny

@pytest.mark.parametrize("exact", [True, False])
def test_tiny_config_full(H, oracle_mod, exact):
    """BASELINE.json configs[0]: S=2, G=2, flat 1,000,000 fp32, lr 0.1, mu 0.9, 10 steps."""
    flags = H.DETERMINISTIC if exact else 0
    gw, gv, ow, ov = run_both(H, oracle_mod, 2, 2, [1_000_000], 10, flags=flags, seed=1)
    assert_parity(gw, gv, ow, ov, exact)


# ------------------------------------------------------------------------------- shapes / edge cases

ODD_TABLE = [1, 3, 7, 1025, 64, 63, 65, 4099, 2, 100_001]      # adversarial ragged table


@pytest.mark.parametrize("S,G", [(1, 1), (2, 1), (2, 2), (4, 3), (4, 4), (6, 5), (8, 8), (16, 4), (2, 16), (2, 13)])
@pytest.mark.parametrize("bf16", [False, True])
def test_small_shapes_bit_exact(H, oracle_mod, S, G, bf16):
    """Templated G in {1,2,4,8} and the runtime-G kernel (3,5,13,16); several tiles plus a
    ragged tail (P = 70,001 is not a multiple of anything); deterministic => bit-exact."""
    gw, gv, ow, ov = run_both(H, oracle_mod, S, G, [70_001], 3, bf16=bf16, flags=H.DETERMINISTIC, seed=S * 100 + G,
                              v0_sd=0.01)
    assert_parity(gw, gv, ow, ov, True)


@pytest.mark.parametrize("bf16", [False, True])
@pytest.mark.parametrize("exact", [True, False])
def test_ragged_table_equals_flat(H, oracle_mod, bf16, exact):
    """Odd-length segment table: padded layout, padding stays zero, results equal the oracle on
    the concatenated (flat) data."""
    flags = H.DETERMINISTIC if exact else 0
    gw, gv, ow, ov = run_both(H, oracle_mod, 4, 2, ODD_TABLE, 4, bf16=bf16, flags=flags, seed=21)
    assert_parity(gw, gv, ow, ov, exact)
    if exact:   # and the flat layout gives the very same bits
        fw, fv, _, _ = run_both(H, oracle_mod, 4, 2, [sum(ODD_TABLE)], 4, bf16=bf16, flags=flags, seed=21)
        assert np.array_equal(bits(fw), bits(gw)) and np.array_equal(bits(fv), bits(gv))


@pytest.mark.parametrize("P", [1, 3, 4, 5, 63, 64, 65, 1023, 1024, 1025])
def test_tiny_lengths(H, oracle_mod, P):
    gw, gv, ow, ov = run_both(H, oracle_mod, 2, 2, [P], 2, flags=H.DETERMINISTIC, seed=P)
    assert_parity(gw, gv, ow, ov, True)


@pytest.mark.parametrize("flagname", ["NO_MIX", "EQ7_LITERAL", "NO_DIAG"])
@pytest.mark.parametrize("bf16", [False, True])
def test_flags(H, oracle_mod, flagname, bf16):
    flags = H.DETERMINISTIC | getattr(H, flagname)
    gw, gv, ow, ov = run_both(H, oracle_mod, 4, 4, [33_333], 3, bf16=bf16, flags=flags, seed=31, v0_sd=0.01)
    assert_parity(gw, gv, ow, ov, True)
    gw, gv, ow, ov = run_both(H, oracle_mod, 4, 4, [33_333], 3, bf16=bf16, flags=getattr(H, flagname), seed=31)
    assert_parity(gw, gv, ow, ov, False)


def test_odd_S_without_mixing(H, oracle_mod):
    gw, gv, ow, ov = run_both(H, oracle_mod, 3, 2, [10_000], 2, flags=H.DETERMINISTIC | H.NO_MIX, seed=41)
    assert_parity(gw, gv, ow, ov, True)


def test_max_S(H, oracle_mod):
    """S = HADPSGD_MAX_S = 512 super-learners (256 pairs: eight launches of 32 work items)."""
    gw, gv, ow, ov = run_both(H, oracle_mod, 512, 1, [2_000], 2, flags=H.DETERMINISTIC, seed=51)
    assert_parity(gw, gv, ow, ov, True)


def test_default_mode_tolerance_20_steps(H, oracle_mod):
    gw, gv, ow, ov = run_both(H, oracle_mod, 16, 4, [50_000], 20, seed=61)
    assert_parity(gw, gv, ow, ov, False)


def test_forced_grid_sizes(H, oracle_mod):
    """Same bits whatever the persistent grid (1 block/SM ... 8 blocks/SM)."""
    ref = None
    for bps in (1, 2, 8):
        gw, gv, ow, ov = run_both(H, oracle_mod, 4, 4, [300_007], 2, flags=H.DETERMINISTIC, seed=71, blocks_per_sm=bps)
        assert_parity(gw, gv, ow, ov, True)


def test_uniform_sweep_points(H, oracle_mod):
    """BASELINE.json configs[4] (bandwidth sweep) sample points small enough for a full
    oracle run: flat fp32, uniform grads in [-1e-3, 1e-3]."""
    for P, S, G in ((1 << 10, 2, 2), (1 << 12, 16, 8), (1 << 14, 4, 4), (1 << 16, 8, 2), (1 << 18, 2, 8)):
        for exact in (True, False):                        # deterministic: bits; default (FMA): tolerance
            gw, gv, ow, ov = run_both(H, oracle_mod, S, G, [P], 3, flags=H.DETERMINISTIC if exact else 0,
                                      seed=P + S + G, dist="uniform")
            assert_parity(gw, gv, ow, ov, exact)


# ------------------------------------------------------------------------------- shared pair storage

@pytest.mark.parametrize("S,G,bf16", [(2, 2, False), (4, 4, False), (16, 4, False), (8, 8, True), (6, 3, False), (1, 2, False),
                                      (8, 1, False), (8, 8, False), (6, 1, True)])
@pytest.mark.parametrize("exact", [True, False])
def test_share_pair_weights_equals_oracle(H, oracle_mod, S, G, bf16, exact):
    """HADPSGD_SHARE_PAIR_WEIGHTS: one weight buffer per pair, tile-major walk -- same arithmetic, so
    the same bits as the oracle (ragged table, 5 steps = both parities, steady state reached)."""
    flags = H.SHARE_PAIR_WEIGHTS | (H.DETERMINISTIC if exact else 0)
    gw, gv, ow, ov = run_both(H, oracle_mod, S, G, ODD_TABLE, 5, bf16=bf16, flags=flags, seed=300 + S + G, v0_sd=0.01)
    assert_parity(gw, gv, ow, ov, exact)


def test_share_pair_weights_pointers_unshare_and_consensus(H, oracle_mod, torch_cuda):
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed = 8, 2, 100_003, 141
    h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC | H.SHARE_PAIR_WEIGHTS, working_dtype=H.BF16)
    problem.fill_weights(h, seed)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    ptr0 = [h.hadpsgd_weights(s).data_ptr() for s in range(S)]
    assert len(set(ptr0)) == S                                     # before the first step: one buffer each
    for k in range(3):
        problem.fill_grads(h, seed, k)
        h.hadpsgd_step(LR, MU, k)
        oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k)
        partner = H.hadpsgd_pairing(S, k)
        ptr = [h.hadpsgd_weights(s).data_ptr() for s in range(S)]
        assert all(ptr[s] == ptr[partner[s]] for s in range(S)) and len(set(ptr)) == S // 2
        assert h.hadpsgd_consensus() == pytest.approx(oracle_mod.consensus_distance(ow), rel=1e-10)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    assert np.array_equal(bits(gw), bits(ow))
    gb = np.stack([h.hadpsgd_weights_bf16(s).view(torch.int16)[:P].cpu().numpy().view(np.uint16) for s in range(S)])
    assert np.array_equal(gb, oracle_mod.round_bf16(ow))
    h.hadpsgd_unshare()                                            # every learner gets its own buffer back
    ptr = [h.hadpsgd_weights(s).data_ptr() for s in range(S)]
    assert len(set(ptr)) == S
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gb = np.stack([h.hadpsgd_weights_bf16(s).view(torch.int16)[:P].cpu().numpy().view(np.uint16) for s in range(S)])
    assert np.array_equal(bits(gw), bits(ow)) and np.array_equal(gb, oracle_mod.round_bf16(ow))
    h.hadpsgd_weights(3)[:P] += 1.0                                # now safe: nobody shares buffer 3
    ow[3] += np.float32(1.0)
    problem.fill_grads(h, seed, 3)
    h.hadpsgd_step(LR, MU, 3)
    oracle_mod.step(problem.host_grads(seed, 3, S, G, 0, P), ow, ov, LR, MU, 3)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    assert np.array_equal(bits(gw), bits(ow))
    h.close()
    for bad in (H.NO_MIX, H.EQ7_LITERAL):
        with pytest.raises(H.HadpsgdError):
            H.Hadpsgd(4, 2, [100], H.F32, H.SHARE_PAIR_WEIGHTS | bad)


def test_share_pair_weights_with_custom_matchings_and_unpaired_members(H, oracle_mod, torch_cuda):
    """Ring steps interleaved with caller-supplied matchings that leave members unmixed (odd S):
    the shared buffers must be split again before an unmixed member updates in place."""
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed = 7, 2, 30_011, 151
    matchings = [[1, 0, 3, 2, 5, 4, 6], [0, 2, 1, 4, 3, 6, 5], [6, 1, 2, 3, 4, 5, 0], [1, 0, 3, 2, 5, 4, 6],
                 [0, 1, 2, 3, 4, 5, 6], [2, 3, 0, 1, 6, 5, 4]]
    h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC | H.SHARE_PAIR_WEIGHTS)
    problem.fill_weights(h, seed)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    for k, partner in enumerate(matchings):
        problem.fill_grads(h, seed, k)
        h.hadpsgd_step_matching(LR, MU, k, partner)
        od = oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k, diag=True, partner=partner)
        assert_diag(h.hadpsgd_diagnostics(), od, k)
        gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
        gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
        assert np.array_equal(bits(gw), bits(ow)) and np.array_equal(bits(gv), bits(ov)), k
    h.close()


def test_share_pair_weights_graph_replay_from_steady_state(H, oracle_mod, torch_cuda):
    """With shared buffers the launch parameters depend on which buffer holds what; the pattern is
    periodic with period 2 once one step has run, so an (odd, even) pair captured after one eager
    step replays correctly."""
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed = 4, 2, 123_457, 161
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC | H.SHARE_PAIR_WEIGHTS, stream=side)
        problem.fill_weights(h, seed)
        problem.fill_grads(h, seed, 0)
        h.hadpsgd_step(LR, MU, 0)                                  # eager: reaches the periodic state
    side.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        h.hadpsgd_step(LR, MU, 1)
        h.hadpsgd_step(LR, MU, 2)
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    og = problem.host_grads(seed, 0, S, G, 0, P)
    for k in range(7):
        oracle_mod.step(og, ow, ov, LR, MU, k)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    assert_parity(gw, gv, ow, ov, True)
    h.close()


# ------------------------------------------------------------------------------- super-learner partition (f4)

def _ring(S, k):
    p = [0] * S
    for i in range(S // 2):
        a, b = (2 * i + k % 2) % S, (2 * i + 1 + k % 2) % S
        p[a], p[b] = b, a
    return p


def run_peer_group(H, oracle_mod, rank_begin, G, seg_len, matchings, *, bf16=False, exact=True, seed=401,
                   flush_at=(), no_diag=False):
    """R = len(rank_begin)-1 HADPSGD_PEER handles on ONE GPU and one stream stand in for R ranks (a
    same-device pointer is a valid peer pointer; one stream is the epoch barrier).  Every step is
    compared with the oracle on all S_global super-learners: momentum and gsq at once; weights, wsq and
    gap at once for members whose mix completed inside the step, and one step later (pend_wsq /
    pend_gap, or after hadpsgd_peer_flush) for members whose partner lives in another arena."""
    import torch
    from fixtures import device, generator as gen
    world, S = len(rank_begin) - 1, rank_begin[-1]
    P = int(sum(seg_len))
    flags = H.PEER | (H.DETERMINISTIC if exact else 0) | (H.NO_DIAG if no_diag else 0)
    hs = [H.Hadpsgd(rank_begin[r + 1] - rank_begin[r], G, seg_len, H.BF16 if bf16 else H.F32, flags) for r in range(world)]
    for r, h in enumerate(hs):
        h.hadpsgd_peer_init(r, world, rank_begin)
    for r, h in enumerate(hs):
        for q, other in enumerate(hs):
            if q != r:
                h.hadpsgd_peer_attach(q, other.hadpsgd_peer_stage())
    nat_off = np.concatenate([[0], np.cumsum(seg_len)])

    def fill(buf, h, key, dist, scale):
        for k, n in enumerate(seg_len):
            off, _ = h.hadpsgd_segment(k)
            device.fill(buf[off:off + n], key, dist, scale, elem_offset=int(nat_off[k]))

    owner = lambda sg: next(r for r in range(world) if rank_begin[r] <= sg < rank_begin[r + 1])
    for sg in range(S):
        h = hs[owner(sg)]
        fill(h.hadpsgd_weights(sg - rank_begin[owner(sg)]), h, gen.stream_key(seed, gen.STREAM_WEIGHT, 0, sg, 0), "normal", 0.05)
    from fixtures import problem
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    nat = torch.from_numpy(hs[0].natural_index()).cuda()
    prev = None                                       # (oracle diag, pending flags) of the step before
    for k, partner in enumerate(matchings):
        for sg in range(S):
            h, sl = hs[owner(sg)], sg - rank_begin[owner(sg)]
            for g in range(G):
                fill(h.hadpsgd_grads(sl, g), h, gen.stream_key(seed, gen.STREAM_GRAD, k, sg, g), "normal", 1e-3)
        for h in hs:                                  # same stream: launch order is the epoch barrier
            if partner is None:
                h.hadpsgd_step(LR, MU, k)
            else:
                h.hadpsgd_step_matching(LR, MU, k, partner)
        og = problem.host_grads(seed, k, S, G, 0, P, bf16=bf16)
        od = oracle_mod.step(og, ow, ov, LR, MU, k, diag=True, partner=partner if partner is not None else _ring(S, k))
        pend_now = np.zeros(S, bool)
        for r, h in enumerate(hs):
            lo, hi = rank_begin[r], rank_begin[r + 1]
            gv = np.stack([h.hadpsgd_momentum(s)[nat].cpu().numpy() for s in range(hi - lo)])
            if exact:
                assert np.array_equal(bits(gv), bits(ov[lo:hi])), (k, r)
            else:
                assert np.all(np.abs(gv - ov[lo:hi]) <= 1e-6 + 1e-5 * np.abs(ov[lo:hi]))
            if no_diag:
                continue
            d = h.hadpsgd_diagnostics()
            pend_now[lo:hi] = d["pending"] == 1
            assert np.allclose(d["gsq"], od["gsq"][lo:hi], rtol=1e-4, atol=1e-30), (k, r)
            done = ~pend_now[lo:hi]
            assert np.allclose(d["wsq"][done], od["wsq"][lo:hi][done], rtol=1e-4, atol=1e-30), (k, r)
            assert np.allclose(d["gap"][done], od["gap"][lo:hi][done], rtol=1e-4, atol=1e-30), (k, r)
            assert np.array_equal(d["gap"][done] == 0, od["gap"][lo:hi][done] == 0)
            if prev is not None:                      # what the step before still owed
                was = prev[1][lo:hi]
                assert np.allclose(d["pend_wsq"][was], prev[0]["wsq"][lo:hi][was], rtol=1e-4), (k, r)
                assert np.allclose(d["pend_gap"][was], prev[0]["gap"][lo:hi][was], rtol=1e-4), (k, r)
                assert not d["pend_wsq"][~was].any() and not d["pend_gap"][~was].any()
        prev = (od, pend_now)
        if k in flush_at:
            for r, h in enumerate(hs):
                h.hadpsgd_peer_flush()
                if not no_diag:
                    d = h.hadpsgd_diagnostics()
                    lo, hi = rank_begin[r], rank_begin[r + 1]
                    was = pend_now[lo:hi]
                    assert np.allclose(d["pend_wsq"][was], od["wsq"][lo:hi][was], rtol=1e-4)
                    assert np.allclose(d["pend_gap"][was], od["gap"][lo:hi][was], rtol=1e-4)
                    assert not d["pending"].any()
            prev = None
            gw = np.concatenate([np.stack([h.hadpsgd_weights(s)[nat].cpu().numpy() for s in range(h.S)]) for h in hs])
            assert_parity(gw, gw * 0, ow, ow * 0, exact)
    for h in hs:
        h.hadpsgd_peer_flush()
    torch.cuda.synchronize()
    gw = np.concatenate([np.stack([h.hadpsgd_weights(s)[nat].cpu().numpy() for s in range(h.S)]) for h in hs])
    gv = np.concatenate([np.stack([h.hadpsgd_momentum(s)[nat].cpu().numpy() for s in range(h.S)]) for h in hs])
    launches = [h.hadpsgd_launch_count() for h in hs]
    if sum(seg_len) != hs[0].P_padded:                # padding of main and stage buffers stays zero
        mask = torch.ones(hs[0].P_padded, dtype=torch.bool, device="cuda"); mask[nat] = False
        for h in hs:
            stage = h._view(h.hadpsgd_peer_stage(), 2 * h.S * h.P_padded, torch.float32).view(2 * h.S, h.P_padded)
            assert not stage[:, mask].any()
    for h in hs:
        h.close()
    assert_parity(gw, gv, ow, ov, exact)
    return launches


@pytest.mark.parametrize("rank_begin", [[0, 2, 4, 6, 8], [0, 1, 2, 3, 4], [0, 3, 5, 8], [0, 8], [0, 4, 8]])
@pytest.mark.parametrize("exact", [True, False])
def test_peer_partition_ring_multi_arena(H, oracle_mod, rank_begin, exact):
    """Ring schedule over R arenas (2 super-learners per 'GPU' is the paper's 16x4 on 8 nodes in small):
    on odd steps EVERY pair straddles two arenas.  Ragged table, 7 steps, a flush in the middle."""
    run_peer_group(H, oracle_mod, rank_begin, 4, ODD_TABLE, [None] * 7, exact=exact, flush_at=(3,))


def test_peer_partition_custom_matchings_odd_S(H, oracle_mod):
    rank_begin = [0, 3, 4, 7]
    matchings = [[3, 1, 5, 0, 4, 2, 6], [1, 0, 3, 2, 5, 4, 6], [6, 2, 1, 4, 3, 5, 0], [0, 1, 2, 3, 4, 5, 6],
                 [4, 5, 6, 3, 0, 1, 2], [4, 5, 6, 3, 0, 1, 2], [1, 0, 2, 6, 5, 4, 3]]
    run_peer_group(H, oracle_mod, rank_begin, 2, [50_003], matchings, flush_at=(2, 4))


@pytest.mark.parametrize("G,bf16", [(8, True), (3, False), (8, False), (1, True)])
def test_peer_partition_other_kernels(H, oracle_mod, G, bf16):
    """bf16 gradients, G = 8 and the runtime-G kernel in peer mode; one launch per step per rank when a
    rank's work is all pairs or all singles."""
    launches = run_peer_group(H, oracle_mod, [0, 2, 4], G, [70_001], [None] * 4, bf16=bf16)
    assert launches == [4 + 1, 4 + 1]                  # 4 steps + the final flush (S = 4: both members pending)
    run_peer_group(H, oracle_mod, [0, 2, 4], G, [3_001], [None] * 3, bf16=bf16, no_diag=True)


def test_peer_errors(H):
    h = H.Hadpsgd(2, 2, [1000], H.F32, H.PEER)
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_step(LR, MU, 0)                       # not initialised
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_peer_init(0, 2, [0, 3, 4])            # S mismatch
    h.hadpsgd_peer_init(0, 2, [0, 2, 4])
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_step(LR, MU, 1)                       # rank 1 not attached
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_peer_attach(0, h.hadpsgd_peer_stage())   # own rank
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_consensus()
    h.close()
    for bad in (H.SHARE_PAIR_WEIGHTS, H.EQ7_LITERAL):
        with pytest.raises(H.HadpsgdError):
            H.Hadpsgd(2, 2, [1000], H.F32, H.PEER | bad)
    with pytest.raises(H.HadpsgdError):
        H.Hadpsgd(2, 2, [1000], H.F32, H.PEER, working_dtype=H.BF16)
    plain = H.Hadpsgd(2, 2, [1000])
    with pytest.raises(H.HadpsgdError):
        plain.hadpsgd_peer_init(0, 1, [0, 2])
    plain.close()


def _ipc_worker(rank, world, port, out_dir):
    """One process per rank, BOTH ON GPU 0: stage regions are exchanged as CUDA IPC handles (gloo carries
    the 64 bytes).  Between steps there is NO synchronize and NO barrier: the library's neighbour-only epoch
    handshake (stream waits on the partner's epoch word, through the IPC mapping) orders the two
    processes; rank 1 is delayed on purpose so that rank 0 runs ahead and must block.  No kernel waits on
    another."""
    import os
    import torch
    import torch.distributed as dist
    import paper_1907_05701_b200 as Hm
    from fixtures import device, generator as gen
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        S, G, P, seed, steps = 8, 2, 200_003, 431, 5
        rank_begin = [0, 4, 8]
        lo = rank_begin[rank]
        h = Hm.Hadpsgd(4, G, [P], Hm.F32, Hm.PEER | Hm.DETERMINISTIC, own_arena=(rank == 0))   # one of each arena kind
        h.hadpsgd_peer_init(rank, world, rank_begin)
        ipc, off = h.hadpsgd_peer_ipc_export()
        mine = torch.tensor(list(ipc) + list(off.to_bytes(8, "little")), dtype=torch.uint8)
        got = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(got, mine)
        for r in range(world):
            if r != rank:
                raw = bytes(got[r].tolist())
                h.hadpsgd_peer_ipc_attach(r, raw[:64], int.from_bytes(raw[64:], "little"))
                h.hadpsgd_peer_ipc_attach(r, raw[:64], int.from_bytes(raw[64:], "little"))   # re-attach: the old mapping is closed
        for s in range(4):
            device.fill(h.hadpsgd_weights(s)[:P], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, lo + s, 0), "normal", 0.05)
        for k in range(steps):
            for s in range(4):
                for g in range(G):
                    device.fill(h.hadpsgd_grads(s, g)[:P], gen.stream_key(seed, gen.STREAM_GRAD, k, lo + s, g), "normal", 1e-3)
            if rank == 1 and k in (1, 3):
                torch.cuda._sleep(400_000_000)          # ~0.2 s: the other process gets two steps ahead of this one
            h.hadpsgd_step(0.1, 0.9, k)                 # no synchronize, no barrier: the epoch handshake orders the ranks
        h.hadpsgd_peer_flush()
        torch.cuda.synchronize()
        dist.barrier()                                  # nobody tears its stage region down before all have read it
        w = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(4)])
        v = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(4)])
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), w=w, v=v)
        dist.barrier()
        h.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_peer_partition_two_processes_cuda_ipc(H, oracle_mod, tmp_path):
    """The cross-process plumbing of bench.py --partition superlearner, on one GPU: two processes, each
    owning 4 of 8 super-learners, read each other's stage buffers through cudaIpcOpenMemHandle
    mappings inside the fused kernel.  Bit-exact against the oracle on all 8."""
    import socket
    import torch.multiprocessing as mp
    from fixtures import problem
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    mp.spawn(_ipc_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    S, G, P, seed, steps = 8, 2, 200_003, 431, 5
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    for k in range(steps):
        oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k)
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(2)]
    assert np.array_equal(bits(np.concatenate([p["w"] for p in parts])), bits(ow))
    assert np.array_equal(bits(np.concatenate([p["v"] for p in parts])), bits(ov))


def test_range_partition_shards_equal_the_unsharded_model(H, oracle_mod, torch_cuda):
    """bench.py --partition range: rank r owns hadpsgd_shard_range(P, N, r) of every buffer of ONE model.
    Three shard handles on one GPU, filled from the GLOBAL element index, must reproduce the unsharded
    handle bit for bit, and their diagnostics must add up to its diagnostics (the all-reduce)."""
    torch = torch_cuda
    from fixtures import device, generator as gen, problem
    S, G, P, seed, world = 4, 2, 64 * 3001, 501, 3
    full = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC)
    problem.fill_weights(full, seed)
    shards = []
    for r in range(world):
        lo, hi = H.hadpsgd_shard_range(P, world, r)
        h = H.Hadpsgd(S, G, [hi - lo], H.F32, H.DETERMINISTIC)
        for s in range(S):
            device.fill(h.hadpsgd_weights(s)[:hi - lo], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, s, 0), "normal", 0.05, elem_offset=lo)
        shards.append((lo, hi, h))
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    for k in range(3):
        problem.fill_grads(full, seed, k)
        full.hadpsgd_step(LR, MU, k)
        od = oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k, diag=True)
        tot = {n: np.zeros(S) for n in ("gsq", "wsq", "gap")}
        for lo, hi, h in shards:
            for s in range(S):
                for g in range(G):
                    device.fill(h.hadpsgd_grads(s, g)[:hi - lo], gen.stream_key(seed, gen.STREAM_GRAD, k, s, g), "normal", 1e-3,
                                elem_offset=lo)
            h.hadpsgd_step(LR, MU, k)
            d = h.hadpsgd_diagnostics()
            for n in tot:
                tot[n] += d[n]
        assert_diag(tot, od, k)
    torch.cuda.synchronize()
    for lo, hi, h in shards:
        for s in range(S):
            assert torch.equal(h.hadpsgd_weights(s)[:hi - lo], full.hadpsgd_weights(s)[lo:hi])
            assert torch.equal(h.hadpsgd_momentum(s)[:hi - lo], full.hadpsgd_momentum(s)[lo:hi])
        h.close()
    gw = np.stack([full.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    assert np.array_equal(bits(gw), bits(ow))
    full.close()


# ------------------------------------------------------------------------------- API behaviour

def test_custom_matching_and_unpaired(H, oracle_mod):
    """hadpsgd_step_matching (row f1): caller-supplied matching, including unpaired members, against
    the oracle's own matching entry (weights, momentum and all three diagnostics; two launches --
    pairs then singles -- feed one diagnostics record)."""
    import torch
    from fixtures import problem
    S, G, P, seed = 7, 2, 20_000, 81                  # odd S: only possible with unpaired members
    partner = [3, 1, 5, 0, 4, 2, 6]                   # pairs (0,3), (2,5); 1, 4 and 6 unmixed (T_ii = 1)
    h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC)
    problem.fill_weights(h, seed)
    problem.fill_grads(h, seed, 0)
    h.hadpsgd_step_matching(LR, MU, 0, partner)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    od = oracle_mod.step(problem.host_grads(seed, 0, S, G, 0, P), ow, ov, LR, MU, 0, diag=True, partner=partner)
    assert_diag(h.hadpsgd_diagnostics(), od)
    torch.cuda.synchronize()
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    assert_parity(gw, gv, ow, ov, True)
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_step_matching(LR, MU, 0, [1, 2, 0, 3, 4, 5, 6])  # not an involution
    h.close()


MATCHING_SEQ = [[3, 1, 5, 0, 4, 2, 6], [1, 0, 3, 2, 5, 4, 6], [0, 1, 2, 3, 4, 5, 6], [6, 2, 1, 4, 3, 5, 0]]


@pytest.mark.parametrize("flagname", [None, "EQ7_LITERAL"])
@pytest.mark.parametrize("bf16", [False, True])
@pytest.mark.parametrize("exact", [True, False])
def test_matching_sequences_with_diagnostics(H, oracle_mod, flagname, bf16, exact):
    """Caller-supplied matchings over several steps (odd S, non-neighbour pairs, unmixed members, the
    identity), default and eq.-(7)-literal: w, v and every step's diagnostics against the oracle's
    matching entry."""
    flags = (H.DETERMINISTIC if exact else 0) | (getattr(H, flagname) if flagname else 0)
    gw, gv, ow, ov = run_both(H, oracle_mod, 7, 3, ODD_TABLE, len(MATCHING_SEQ), bf16=bf16, flags=flags, seed=171,
                              v0_sd=0.01, matching=lambda k: MATCHING_SEQ[k])
    assert_parity(gw, gv, ow, ov, exact)


def test_max_S_unmixed_diagnostics_span_several_launches(H, oracle_mod):
    """S = 512 unmixed super-learners = 512 single items, 32 per launch: sixteen launches feed one
    diagnostics record (gap exactly 0 everywhere)."""
    gw, gv, ow, ov = run_both(H, oracle_mod, 512, 2, [3_001], 2, flags=H.DETERMINISTIC | H.NO_MIX, seed=52)
    assert_parity(gw, gv, ow, ov, True)


def test_diagnostics_stress_large_grids(H, oracle_mod):
    """Many work items (S = 32: 16 pairs, so several warps write block partials), the largest
    persistent grid (16 blocks/SM), many steps: diagnostics must equal the oracle's every step and be
    bitwise identical between two runs (the collectors add the tagged block partials in a fixed order)."""
    from fixtures import problem
    S, G, P, seed, steps = 32, 2, 40_003, 181, 12
    runs = []
    for rep in range(2):
        h = H.Hadpsgd(S, G, [P], H.F32, 0)
        h.hadpsgd_set_launch(16)
        problem.fill_weights(h, seed)
        ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
        rec = []
        for k in range(steps):
            problem.fill_grads(h, seed, k)
            h.hadpsgd_step(LR, MU, k)
            gd = h.hadpsgd_diagnostics()
            if rep == 0:
                assert_diag(gd, oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k, diag=True), k)
            rec.append(np.concatenate([gd["gsq"], gd["wsq"], gd["gap"]]))
        runs.append(np.stack(rec))
        h.close()
    assert np.array_equal(runs[0], runs[1])


def test_diagnostics_under_graph_replay_with_fresh_gradients(H, oracle_mod, torch_cuda):
    """A replayed graph re-launches the step with the SAME tag on its block partials.  The gradients
    are refilled between replays, so a collector that picked up a partial of an earlier replay (a slot
    it failed to zero) would report that replay's sums: every replay's diagnostics must equal the
    oracle's for that step.  Several blocks per item and several items per collector-less block."""
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed = 8, 2, 300_011, 77
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC, stream=side)
        problem.fill_weights(h, seed)
        problem.fill_grads(h, seed, 0)
    side.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        h.hadpsgd_step(LR, MU, 0)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    for rep in range(6):
        with torch.cuda.stream(side):
            problem.fill_grads(h, seed, rep)
            graph.replay()
            gd = h.hadpsgd_diagnostics()
        od = oracle_mod.step(problem.host_grads(seed, rep, S, G, 0, P), ow, ov, LR, MU, 0, diag=True)
        assert_diag(gd, od, rep)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    assert_parity(gw, gv, ow, ov, True)
    h.close()


def test_diagnostics_with_the_launch_shape_changing_every_step(H, oracle_mod):
    """One handle, the grid and the number of work items changing from step to step (blocks per SM 1,
    16, 3, default; matchings with 3, 1, 0 and 2 pairs): the block partials of one launch must never
    be taken for those of another (different rows per block, different contributors per item)."""
    from fixtures import problem
    S, G, P, seed = 7, 3, 150_001, 191
    seqs = [[1, 0, 3, 2, 5, 4, 6], [0, 1, 6, 3, 4, 5, 2], list(range(7)), [4, 1, 5, 3, 0, 2, 6]]
    bps = [1, 16, 3, 0]
    h = H.Hadpsgd(S, G, [P], H.F32, 0)
    problem.fill_weights(h, seed)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    for k in range(12):
        m = np.asarray(seqs[k % 4], np.int32)
        h.hadpsgd_set_launch(bps[(k // 4 + k) % 4])
        problem.fill_grads(h, seed, k)
        h.hadpsgd_step_matching(LR, MU, k, m)
        od = oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k, diag=True, partner=m)
        assert_diag(h.hadpsgd_diagnostics(), od, k)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    assert_parity(gw, gv, ow, ov, False)
    h.close()


def test_handles_stepping_concurrently_on_their_own_streams(H, torch_cuda):
    """Four handles of different shapes (one with the largest grid, 16 blocks/SM) enqueue 60 steps each
    on four streams at once, so their grids share the SMs and no grid is resident as a whole all the time:
    the collectors of the diagnostics still get every block partial (they wait for blocks that are
    running or queued, never for one that cannot run), and weights and diagnostics equal, bit for bit,
    those of the same handles stepped one after the other."""
    torch = torch_cuda
    from fixtures import problem
    shapes = [(16, 4, 300_011), (8, 8, 200_003), (4, 2, 1_000_003), (32, 2, 40_003)]

    def run(concurrent, steps=60):
        streams = [torch.cuda.Stream() for _ in shapes]
        hs = []
        for i, (S, G, P) in enumerate(shapes):
            with torch.cuda.stream(streams[i]):
                h = H.Hadpsgd(S, G, [P], H.F32, 0, stream=streams[i])
                if i == 3:
                    h.hadpsgd_set_launch(16)
                problem.fill_weights(h, 50 + i)
                problem.fill_grads(h, 50 + i, 0)
            hs.append(h)
        torch.cuda.synchronize()
        recs = [[] for _ in hs]

        def look(i):
            d = hs[i].hadpsgd_diagnostics()
            recs[i].append(np.concatenate([d["gsq"], d["wsq"], d["gap"]]))
        if concurrent:
            for k in range(steps):
                for h in hs:
                    h.hadpsgd_step(LR, MU, k)
                if k % 20 == 19:
                    for i in range(len(hs)):
                        look(i)
        else:
            for i, h in enumerate(hs):
                for k in range(steps):
                    h.hadpsgd_step(LR, MU, k)
                    if k % 20 == 19:
                        look(i)
        torch.cuda.synchronize()
        out = [(np.stack(r), torch.stack([h.hadpsgd_weights(s) for s in range(h.S)]).cpu().numpy()) for r, h in zip(recs, hs)]
        for h in hs:
            h.close()
        return out

    serial, together = run(False), run(True)
    for (d0, w0), (d1, w1) in zip(serial, together):
        assert not np.isnan(d0).any() and np.array_equal(d0, d1)
        assert np.array_equal(bits(w0), bits(w1))


@pytest.mark.parametrize("share", [False, True])
def test_host_gradient_path_equals_resident_path(H, oracle_mod, share):
    """hadpsgd_step_host (the e2e entry): chunked H2D + kernel on element sub-ranges must give
    the same bits and the same diagnostics as the resident-gradient step.  P spans 3 chunks."""
    import torch
    from fixtures import problem
    S, G, seed = 4, 2, 91
    P = (8 << 20) * 2 + 12_345 * 64
    outs = []
    for path in ("resident", "host"):
        h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC | (H.SHARE_PAIR_WEIGHTS if share else 0))
        problem.fill_weights(h, seed)
        for k in range(2):
            problem.fill_grads(h, seed, k)
            if path == "resident":
                h.hadpsgd_step(LR, MU, k)
                d = h.hadpsgd_diagnostics()
            else:
                host = [h.hadpsgd_grads(s, g).cpu().pin_memory() for s in range(S) for g in range(G)]
                for s in range(S):
                    for g in range(G):
                        h.hadpsgd_grads(s, g).zero_()          # the copy must really happen
                d = h.hadpsgd_step_host([t.data_ptr() for t in host], LR, MU, k)
        torch.cuda.synchronize()
        outs.append((torch.stack([h.hadpsgd_weights(s) for s in range(S)]).cpu().numpy(),
                     torch.stack([h.hadpsgd_momentum(s) for s in range(S)]).cpu().numpy(), d))
        h.close()
    assert np.array_equal(bits(outs[0][0]), bits(outs[1][0])) and np.array_equal(bits(outs[0][1]), bits(outs[1][1]))
    for name in ("gsq", "wsq", "gap"):
        assert np.allclose(outs[0][2][name], outs[1][2][name], rtol=1e-12)
    # against the oracle: windows around every chunk boundary of the host path (8 Mi elements), the
    # start, the ragged end and two interior stretches -- 1.3 M elements per buffer in all
    chunk = 8 << 20
    wins = [(0, 200_000), (chunk - 100_000, chunk + 100_000), (2 * chunk - 100_000, 2 * chunk + 100_000),
            (P - 200_000, P), (3_000_000, 3_250_000), (12_000_000, 12_250_000)]
    for lo, hi in wins:
        ow, ov = problem.host_weights(seed, S, lo, hi), np.zeros((S, hi - lo), np.float32)
        for k in range(2):
            oracle_mod.step(problem.host_grads(seed, k, S, G, lo, hi), ow, ov, LR, MU, k)
        assert np.array_equal(bits(outs[1][0][:, lo:hi]), bits(ow)) and np.array_equal(bits(outs[1][1][:, lo:hi]), bits(ov))


@pytest.mark.parametrize("exact", [True, False])
def test_special_values_propagate_like_ieee(H, oracle_mod, torch_cuda, exact):
    """DESIGN.md R17: no flush-to-zero, Inf/NaN propagate.  Subnormal weights, momenta and gradients,
    huge values whose pair sum overflows, Inf and NaN are planted in both sides' inputs; finite
    results must match (bit for bit in deterministic mode), NaN and Inf must land in the same
    places."""
    torch = torch_cuda
    S, G, P = 4, 2, 4096
    rng = np.random.default_rng(7)
    w = (rng.standard_normal((S, P)) * 0.05).astype(np.float32)
    v = (rng.standard_normal((S, P)) * 0.01).astype(np.float32)
    g = (rng.standard_normal((S, G, P)) * 1e-3).astype(np.float32)
    sub = np.float32(1e-45)                                  # smallest subnormal
    w[0, 0:8] = [sub, -sub, 3 * sub, 1e-39, -1e-39, 0.0, -0.0, 1.1754942e-38]
    w[1:, 0:8] = w[0, 0:8]; v[:, 0:8] = 0.0; g[:, :, 0:8] = 0.0      # every pair averages equal subnormals
    g[2, :, 8:16] = sub; v[2, 8:16] = 2 * sub                # subnormal gradient mean and momentum
    w[0, 16], w[1, 16] = 3.0e38, 3.0e38                      # u_s + u_p overflows to +Inf before the 1/2
    w[2, 17] = np.inf; w[3, 18] = -np.inf; w[0, 19] = np.nan; g[1, 0, 20] = np.nan; v[3, 21] = np.inf
    g[2, 1, 22] = np.inf; g[2, 0, 22] = -np.inf             # Inf - Inf in the learner sum -> NaN
    h = H.Hadpsgd(S, G, [P], H.F32, (H.DETERMINISTIC if exact else 0))
    for s in range(S):
        h.hadpsgd_weights(s)[:P] = torch.from_numpy(w[s]).cuda()
        h.hadpsgd_momentum(s)[:P] = torch.from_numpy(v[s]).cuda()
        for k in range(G):
            h.hadpsgd_grads(s, k)[:P] = torch.from_numpy(g[s, k]).cuda()
    ow, ov = w.copy(), v.copy()
    with np.errstate(all="ignore"):
        for k in range(2):
            h.hadpsgd_step(LR, MU, k)
            oracle_mod.step(g, ow, ov, LR, MU, k)
    torch.cuda.synchronize()
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    h.close()
    for got, want in ((gw, ow), (gv, ov)):
        assert np.array_equal(np.isnan(got), np.isnan(want))
        assert np.array_equal(np.isposinf(got), np.isposinf(want)) and np.array_equal(np.isneginf(got), np.isneginf(want))
        fin = np.isfinite(want)
        if exact:
            assert np.array_equal(bits(got)[fin], bits(want)[fin])
        else:
            with np.errstate(all="ignore"):
                assert np.all(np.abs(got[fin] - want[fin]) <= 1e-6 + 1e-5 * np.abs(want[fin]))
    assert np.isnan(ow).sum() >= 3 and np.isinf(ow).sum() >= 3          # the plants did propagate
    # subnormal inputs were not flushed: 1/2 (sub + sub) = sub, 1/2 (3 sub + 3 sub) = 3 sub
    assert gw[0, 0] == sub and gw[0, 2] == 3 * sub and gw[0, 1] == -sub


def test_library_owned_arena_and_two_streams(H, oracle_mod, torch_cuda):
    """opts.arena == NULL: the library cudaMallocs (and frees) its own memory.  Two such handles on
    two different streams run the same problem concurrently and both must match the oracle."""
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed = 4, 2, 200_003, 131
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    hs = []
    for st in streams:
        with torch.cuda.stream(st):
            h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC, stream=st, own_arena=True)
            assert h.arena is None
            problem.fill_weights(h, seed)
            problem.fill_grads(h, seed, 0)
        hs.append(h)
    for k in range(4):
        for h in hs:
            h.hadpsgd_step(LR, MU, k)           # enqueue on both streams back to back
    torch.cuda.synchronize()
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    og = problem.host_grads(seed, 0, S, G, 0, P)
    for k in range(4):
        oracle_mod.step(og, ow, ov, LR, MU, k)
    for h in hs:
        gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
        gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
        assert_parity(gw, gv, ow, ov, True)
        h.close()


def test_diagnostics_can_be_switched_off_for_some_steps(H, oracle_mod):
    """hadpsgd_set_diagnostics: steps without a5 give the same w, v; hadpsgd_diagnostics() keeps returning
    the record of the last step that computed them."""
    from fixtures import problem
    S, G, P, seed = 4, 2, 50_021, 191
    h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC)
    problem.fill_weights(h, seed)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    kept = None
    for k in range(6):
        h.hadpsgd_set_diagnostics(k % 3 == 0)                       # steps 0 and 3 only
        problem.fill_grads(h, seed, k)
        h.hadpsgd_step(LR, MU, k)
        od = oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P), ow, ov, LR, MU, k, diag=True)
        gd = h.hadpsgd_diagnostics()
        if k % 3 == 0:
            kept = od
        assert gd["step_k"] == (k // 3) * 3
        assert_diag(gd, kept, k)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    assert_parity(gw, gv, ow, ov, True)
    h.close()
    nd = H.Hadpsgd(2, 2, [100], H.F32, H.NO_DIAG)
    with pytest.raises(H.HadpsgdError):
        nd.hadpsgd_set_diagnostics(True)
    nd.hadpsgd_set_diagnostics(False)
    nd.close()


def test_diagnostics_are_run_to_run_deterministic(H):
    from fixtures import problem
    res = []
    for _ in range(3):
        h = H.Hadpsgd(4, 4, [1_000_003], H.F32, 0)
        problem.fill_weights(h, 5)
        problem.fill_grads(h, 5, 0)
        h.hadpsgd_step(LR, MU, 1)
        d = h.hadpsgd_diagnostics()
        res.append(np.concatenate([d["gsq"], d["wsq"], d["gap"]]))
        h.close()
    assert np.array_equal(res[0], res[1]) and np.array_equal(res[0], res[2])


def test_error_codes(H, torch_cuda):
    torch = torch_cuda
    odd = H.Hadpsgd(3, 2, [100])                                 # odd S > 1: no ring matching (R8) ...
    with pytest.raises(H.HadpsgdError) as e:
        odd.hadpsgd_step(LR, MU, 0)
    assert e.value.code == -1 and odd.hadpsgd_launch_count() == 0
    odd.hadpsgd_step_matching(LR, MU, 0, [1, 0, 2])              # ... but a matching with T_22 = 1 is fine
    odd.close()
    with pytest.raises(H.HadpsgdError):
        H.Hadpsgd(2, 0, [100])
    with pytest.raises(H.HadpsgdError):
        H.Hadpsgd(2, 2, [100, 0])
    h = H.Hadpsgd(2, 2, [100])
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_weights(2)
    with pytest.raises(H.HadpsgdError):
        h.hadpsgd_grads(0, 2)
    assert h.hadpsgd_launch_count() == 0
    h.hadpsgd_step(LR, MU, 0)
    assert h.hadpsgd_launch_count() == 1                         # ONE kernel per step
    h.close()
    # arena too small
    import ctypes
    from paper_1907_05701_b200 import binding as b
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    opts = b.hadpsgd_opts(small.data_ptr(), 1024, None, 0, 0)
    arr = (ctypes.c_int64 * 1)(100_000)
    hh = ctypes.c_void_p()
    rc = b.lib().hadpsgd_create(2, 2, arr, 1, b.hadpsgd_dtypes(0, 0), ctypes.byref(opts), ctypes.byref(hh))
    assert rc == b.OUT_OF_MEMORY and not hh


@pytest.mark.parametrize("bf16_grads,S,G,flagname", [(False, 4, 4, None), (True, 4, 8, None), (False, 2, 3, None),
                                                     (True, 3, 2, "NO_MIX"), (False, 4, 2, "EQ7_LITERAL")])
def test_bf16_working_copy(H, oracle_mod, torch_cuda, bf16_grads, S, G, flagname):
    """dtypes.working_dtype = BF16 (row f2): every step also writes bf16(w') round-to-nearest-even.
    Deterministic mode: the copy equals the oracle's rounding of the oracle's weights, bit for bit;
    default mode: it is the correct rounding of the weights the GPU itself produced.  Ragged table,
    so the copy's padding must stay zero too."""
    torch = torch_cuda
    from fixtures import problem
    seg, seed, steps = ODD_TABLE, 111, 3
    P = sum(seg)
    extra = getattr(H, flagname) if flagname else 0
    oflags = getattr(oracle_mod, flagname) if flagname in ("NO_MIX", "EQ7_LITERAL") else 0
    for exact in (True, False):
        h = H.Hadpsgd(S, G, seg, H.BF16 if bf16_grads else H.F32, (H.DETERMINISTIC if exact else 0) | extra,
                      working_dtype=H.BF16)
        problem.fill_weights(h, seed)
        ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
        assert not h.hadpsgd_weights_bf16(0).view(torch.int16).any()          # zero until the first step
        for k in range(steps):
            problem.fill_grads(h, seed, k)
            h.hadpsgd_step(LR, MU, k)
            oracle_mod.step(problem.host_grads(seed, k, S, G, 0, P, bf16=bf16_grads), ow, ov, LR, MU, k, flags=oflags)
        torch.cuda.synchronize()
        nat = torch.from_numpy(h.natural_index()).cuda()
        gw = np.stack([h.hadpsgd_weights(s)[nat].cpu().numpy() for s in range(S)])
        gb = np.stack([h.hadpsgd_weights_bf16(s).view(torch.int16)[nat].cpu().numpy().view(np.uint16) for s in range(S)])
        assert np.array_equal(gb, oracle_mod.round_bf16(gw))                  # correct rounding of the GPU's own w'
        if exact:
            assert np.array_equal(bits(gw), bits(ow))
            assert np.array_equal(gb, oracle_mod.round_bf16(ow))
        mask = torch.ones(h.P_padded, dtype=torch.bool, device="cuda"); mask[nat] = False
        for s in range(S):
            assert not h.hadpsgd_weights_bf16(s).view(torch.int16)[mask].any()
        h.close()
    plain = H.Hadpsgd(2, 2, [100])
    with pytest.raises(H.HadpsgdError):
        plain.hadpsgd_weights_bf16(0)
    plain.close()


def test_consensus_distance_and_variance_identity(H, oracle_mod, torch_cuda):
    """hadpsgd_consensus: D = sum_s |w_s - wbar|^2 against the oracle, and -- with zero
    gradients, so u = w -- the invariant D(before) - D(after) = 1/2 sum_pairs gap that ties the a5
    pair-gap diagnostic to consensus, and the contraction of D under repeated mixing."""
    torch = torch_cuda
    from fixtures import problem
    S, G, seg, seed = 8, 2, ODD_TABLE, 121
    P = sum(seg)
    h = H.Hadpsgd(S, G, seg, H.F32, H.DETERMINISTIC)
    problem.fill_weights(h, seed)                       # gradients and momentum stay zero
    ow = problem.host_weights(seed, S, 0, P)
    ov = np.zeros((S, P), np.float32)
    og = np.zeros((S, G, P), np.float32)
    D = [h.hadpsgd_consensus()]
    assert D[0] == pytest.approx(oracle_mod.consensus_distance(ow), rel=1e-10)
    for k in range(6):
        h.hadpsgd_step(LR, MU, k)
        d = h.hadpsgd_diagnostics()
        oracle_mod.step(og, ow, ov, LR, MU, k)
        D.append(h.hadpsgd_consensus())
        assert D[-1] == pytest.approx(oracle_mod.consensus_distance(ow), rel=1e-10)
        partner = H.hadpsgd_pairing(S, k)
        half_gap = 0.5 * sum(d["gap"][s] for s in range(S) if s < partner[s])
        assert D[-2] - D[-1] == pytest.approx(half_gap, rel=1e-5)
        assert D[-1] < D[-2]
    assert h.hadpsgd_consensus() == D[-1]               # run-to-run deterministic
    h.close()


def test_cuda_graph_capture_and_replay(H, oracle_mod, torch_cuda):
    """hadpsgd_step only enqueues on its stream, so an (even, odd) step pair can be captured into a
    CUDA graph and replayed; 3 replays = 6 steps must equal 6 oracle steps bit for bit."""
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed = 4, 2, 123_457, 101
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC, stream=side)
        problem.fill_weights(h, seed)
        problem.fill_grads(h, seed, 0)
    side.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        h.hadpsgd_step(LR, MU, 0)
        h.hadpsgd_step(LR, MU, 1)
    assert h.hadpsgd_launch_count() == 2
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    og = problem.host_grads(seed, 0, S, G, 0, P)
    for k in range(6):
        oracle_mod.step(og, ow, ov, LR, MU, k)
    gw = np.stack([h.hadpsgd_weights(s)[:P].cpu().numpy() for s in range(S)])
    gv = np.stack([h.hadpsgd_momentum(s)[:P].cpu().numpy() for s in range(S)])
    assert_parity(gw, gv, ow, ov, True)
    d = h.hadpsgd_diagnostics()
    assert d["step_k"] == 1 and np.all(d["gsq"] > 0)
    h.close()


# ------------------------------------------------------------------------------- full-size configs

def windows_for(P, seg_len, n_win, width, seed):
    """Element windows (natural index): the very start, the very end (ragged tail), segment
    boundaries, and seeded random places."""
    rng = np.random.default_rng(seed)
    wins = [(0, width), (P - width, P)]
    nat = np.concatenate([[0], np.cumsum(seg_len)])
    for b in nat[1:-1][:: max(1, (len(nat) - 2) // 3)][:3]:
        wins.append((int(b) - width // 2, int(b) + width // 2))
    while len(wins) < n_win:
        lo = int(rng.integers(0, P - width))
        wins.append((lo, lo + width))
    return wins[:n_win]


def full_size_parity(H, oracle_mod, name, *, exact, n_win=6, width=8192, extra_flags=0):
    """BASELINE.json full sizes, in the launch configuration bench.py times (default grid,
    diagnostics on): run all steps on the GPU with per-step regenerated gradients, then check
    sampled element windows against the oracle, which re-runs every step on each window with
    inputs regenerated from (seed, step, s, g, i)."""
    import torch
    from fixtures import problem, shapes
    cfg = shapes.CONFIGS[name]
    S, G, seg_len, steps = cfg["S"], cfg["G"], cfg["seg_len"], cfg["steps"]
    bf16 = cfg["grad"] == "bf16"
    seed = 1000 + len(name)
    P = int(sum(seg_len))
    h = H.Hadpsgd(S, G, seg_len, H.BF16 if bf16 else H.F32, (H.DETERMINISTIC if exact else 0) | extra_flags)
    problem.fill_weights(h, seed)
    diags = []
    for k in range(steps):
        problem.fill_grads(h, seed, k, cfg["dist"])
        h.hadpsgd_step(LR, MU, k)
        diags.append(h.hadpsgd_diagnostics())
    torch.cuda.synchronize()
    assert h.hadpsgd_launch_count() == steps
    for lo, hi in windows_for(P, seg_len, n_win, width, seed):
        idx = torch.from_numpy(problem.padded_index(seg_len, h.layout["seg_offset"], lo, hi)).cuda()
        gw = np.stack([h.hadpsgd_weights(s)[idx].cpu().numpy() for s in range(S)])
        gv = np.stack([h.hadpsgd_momentum(s)[idx].cpu().numpy() for s in range(S)])
        ow, ov = problem.host_weights(seed, S, lo, hi), np.zeros((S, hi - lo), np.float32)
        for k in range(steps):
            oracle_mod.step(problem.host_grads(seed, k, S, G, lo, hi, cfg["dist"], bf16=bf16), ow, ov, LR, MU, k)
        assert_parity(gw, gv, ow, ov, exact)
    # properties that hold at any size: both members of the last step's pairs hold the same
    # bits (R3), and gsq ~ P * sigma^2 / G for i.i.d. gradients of std sigma
    partner = H.hadpsgd_pairing(S, steps - 1)
    for s in range(S):
        if s < partner[s]:
            assert torch.equal(h.hadpsgd_weights(s), h.hadpsgd_weights(partner[s]))
    for d in diags:
        assert np.allclose(d["gsq"], P * 1e-6 / G, rtol=5e-3)
        assert np.all(d["gap"] > 0) and np.all(d["wsq"] > 0)
    h.close()
    torch.cuda.empty_cache()


def test_config1_swb300_full_size(H, oracle_mod):
    """configs[1]: 94,797,312 params flat fp32, S=16, G=4, 20 steps (36.4 GB resident)."""
    full_size_parity(H, oracle_mod, "swb300", exact=True)
    full_size_parity(H, oracle_mod, "swb300", exact=False, n_win=3)      # default (FMA) mode: tolerance


def test_config2_swb2000_full_size_exact(H, oracle_mod):
    """configs[2] (headline): 145,145,344 params flat fp32, S=16, G=4, 20 steps (55.7 GB)."""
    full_size_parity(H, oracle_mod, "swb2000", exact=True)


def test_config2_swb2000_whole_buffer_every_element(H, oracle_mod, torch_cuda):
    """configs[2] (headline), launch configuration of bench.py, deterministic mode: EVERY element of
    every weight and momentum buffer after 2 steps (both ring parities) against the oracle, bit for
    bit.  The oracle stays single-threaded; it is run on disjoint 1 Mi-element windows by one host
    thread per core (the C call releases the GIL).  Oracle inputs come from the device twin of the
    seeded generator (bit-compared with the numpy one in test_device_generator_matches_host),
    generated per window and copied down -- 100 GB of numpy hashing would take minutes."""
    import os
    import threading
    from concurrent.futures import ThreadPoolExecutor
    torch = torch_cuda
    diag_lock = threading.Lock()
    from fixtures import device, generator as gen, problem, shapes
    cfg = shapes.CONFIGS["swb2000"]
    S, G, P, steps, seed = cfg["S"], cfg["G"], int(sum(cfg["seg_len"])), 2, 4242
    h = H.Hadpsgd(S, G, cfg["seg_len"], H.F32, H.DETERMINISTIC)
    assert h.P_padded == P
    problem.fill_weights(h, seed)
    gdiag = []
    for k in range(steps):
        problem.fill_grads(h, seed, k)
        h.hadpsgd_step(LR, MU, k)
        gdiag.append(h.hadpsgd_diagnostics())
    torch.cuda.synchronize()
    assert h.hadpsgd_launch_count() == steps
    n_threads = os.cpu_count() or 1
    W = 1 << 20
    compared = {"w": 0, "v": 0}
    odiag = [{q: np.zeros(S) for q in ("gsq", "wsq", "gap")} for _ in range(steps)]   # the oracle's a5, summed over windows

    def check(lo, hi, w0, grads, gw, gv):
        ow, ov = w0, np.zeros((S, hi - lo), np.float32)
        for k in range(steps):
            d = oracle_mod.step(grads[k], ow, ov, LR, MU, k, diag=True)
            with diag_lock:
                for q in odiag[k]:
                    odiag[k][q] += d[q]
        bad_w, bad_v = int(np.sum(bits(gw) != bits(ow))), int(np.sum(bits(gv) != bits(ov)))
        return lo, hi, bad_w, bad_v

    dev_w0 = torch.empty((S, W), dtype=torch.float32, device="cuda")
    dev_g = torch.empty((steps, S, G, W), dtype=torch.float32, device="cuda")
    futures = []
    with ThreadPoolExecutor(max_workers=n_threads) as pool:
        for lo in range(0, P, W):
            hi = min(lo + W, P)
            n = hi - lo
            for s in range(S):
                device.fill(dev_w0[s], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, s, 0), "normal", 0.05, elem_offset=lo, n=n)
                for k in range(steps):
                    for g in range(G):
                        device.fill(dev_g[k, s, g], gen.stream_key(seed, gen.STREAM_GRAD, k, s, g), "normal", 1e-3,
                                    elem_offset=lo, n=n)
            w0 = np.ascontiguousarray(dev_w0[:, :n].cpu().numpy())
            grads = [np.ascontiguousarray(dev_g[k, :, :, :n].cpu().numpy()) for k in range(steps)]
            gw = np.stack([h.hadpsgd_weights(s)[lo:hi].cpu().numpy() for s in range(S)])
            gv = np.stack([h.hadpsgd_momentum(s)[lo:hi].cpu().numpy() for s in range(S)])
            futures.append(pool.submit(check, lo, hi, w0, grads, gw, gv))
            while len(futures) > 2 * n_threads:           # bound the host memory in flight
                lo_, hi_, bw, bv = futures.pop(0).result()
                assert bw == 0 and bv == 0, (lo_, hi_, bw, bv)
                compared["w"] += S * (hi_ - lo_); compared["v"] += S * (hi_ - lo_)
        for f in futures:
            lo_, hi_, bw, bv = f.result()
            assert bw == 0 and bv == 0, (lo_, hi_, bw, bv)
            compared["w"] += S * (hi_ - lo_); compared["v"] += S * (hi_ - lo_)
    assert compared["w"] == S * P and compared["v"] == S * P       # every element of every buffer
    for k in range(steps):          # a5 at full size against the oracle's double accumulators (Q16: relative 1e-4)
        for q in ("gsq", "wsq", "gap"):
            assert np.allclose(gdiag[k][q], odiag[k][q], rtol=1e-4, atol=0), (k, q, gdiag[k][q], odiag[k][q])
    h.close()
    del dev_w0, dev_g
    torch.cuda.empty_cache()


def test_config2_swb2000_full_size_default_mode(H, oracle_mod):
    full_size_parity(H, oracle_mod, "swb2000", exact=False, n_win=4)


def test_config2_and_3_full_size_shared_pair_weights(H, oracle_mod):
    """The headline config and the ragged bf16 config with HADPSGD_SHARE_PAIR_WEIGHTS (the launch
    configuration bench.py --flags share times)."""
    full_size_parity(H, oracle_mod, "swb2000", exact=True, extra_flags=H.SHARE_PAIR_WEIGHTS)
    full_size_parity(H, oracle_mod, "swb2000", exact=False, n_win=3, extra_flags=H.SHARE_PAIR_WEIGHTS)
    full_size_parity(H, oracle_mod, "swb2000_ragged_bf16", exact=True, n_win=4, extra_flags=H.SHARE_PAIR_WEIGHTS)


def test_config3_ragged_bf16_full_size(H, oracle_mod):
    """configs[3]: same 145M shape as a 40-segment ragged table, bf16 grads, S=8, G=8."""
    full_size_parity(H, oracle_mod, "swb2000_ragged_bf16", exact=True)
    full_size_parity(H, oracle_mod, "swb2000_ragged_bf16", exact=False, n_win=3)


def test_largest_sweep_point_windows(H, oracle_mod, torch_cuda):
    """configs[4] at its maximum size: flat fp32 2^28 params, S=16, G=4 (103 GB resident; byte
    offsets up to 2^36), uniform gradients, 3 steps; sampled windows against the oracle."""
    torch = torch_cuda
    from fixtures import problem
    S, G, P, seed, steps = 16, 4, 1 << 28, 77, 3
    free, _ = torch.cuda.mem_get_info()
    assert free > H.hadpsgd_required_bytes(S, G, [P]), "needs ~103 GB of free HBM"
    h = H.Hadpsgd(S, G, [P], H.F32, H.DETERMINISTIC)
    problem.fill_weights(h, seed)
    for k in range(steps):
        problem.fill_grads(h, seed, k, "uniform")
        h.hadpsgd_step(LR, MU, k)
    torch.cuda.synchronize()
    for lo, hi in windows_for(P, [P], 5, 4096, seed):
        gw = np.stack([h.hadpsgd_weights(s)[lo:hi].cpu().numpy() for s in range(S)])
        gv = np.stack([h.hadpsgd_momentum(s)[lo:hi].cpu().numpy() for s in range(S)])
        ow, ov = problem.host_weights(seed, S, lo, hi), np.zeros((S, hi - lo), np.float32)
        for k in range(steps):
            oracle_mod.step(problem.host_grads(seed, k, S, G, lo, hi, "uniform"), ow, ov, LR, MU, k)
        assert_parity(gw, gv, ow, ov, True)
    h.close()
    torch.cuda.empty_cache()


def test_paper_literal_shape(H, oracle_mod):
    """PAPER.md:106 model (43,130,368 params, '165MB') at 8 super-learners x 8 learners."""
    full_size_parity(H, oracle_mod, "paper_literal", exact=True, n_win=4)
