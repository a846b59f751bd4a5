"""GPU parity, round 3: (1) IEEE edge values (R17) through the kernels the
round-2 special-value test did not reach -- bf16 gradients (both bf16 store forms of the working copy),
the shared-slot CHAIN walk, and a two-arena HADPSGD_PEER group (resolve_pending) -- and (2) EVERY element
of every buffer, plus the a5 diagnostics against the oracle's double accumulators, at BASELINE.json's
full sizes for each distinct kernel family.
All tests need a B200 (-m gpu) and call through the C ABI."""
import os
from concurrent.futures import ThreadPoolExecutor

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


# ------------------------------------------------------------------ the timeout flag of a5

def test_diagnostics_timeout_flag_is_reported_once(H, torch_cuda):
    """A collector that gave up sets a word behind the device results; hadpsgd_diagnostics must turn it
    into HADPSGD_DIAG_TIMEOUT exactly once.  Provoking a real one-minute stall is not a test, so the word
    (the first spare one behind the 5 x S result doubles, at the very end of the arena) is set by hand."""
    torch = torch_cuda
    S = 4
    h = H.Hadpsgd(S, 2, [5000], H.F32, H.DETERMINISTIC)
    h.hadpsgd_step(LR, MU, 0)
    assert h.hadpsgd_diagnostics()["gsq"].shape == (S,)
    tail = (5 * S * 8 + 256 + 255) // 256 * 256                     # allocator: results + 256 spare bytes, rounded
    flag = h.arena[h.arena_bytes - tail + 5 * S * 8: h.arena_bytes - tail + 5 * S * 8 + 4].view(torch.int32)
    assert int(flag.item()) == 0
    flag.fill_(1)
    with pytest.raises(H.HadpsgdError) as e:
        h.hadpsgd_diagnostics()
    assert e.value.code == H.binding.DIAG_TIMEOUT and "timed out" in str(e.value)
    assert h.hadpsgd_diagnostics()["gsq"].shape == (S,)             # reported once; the flag is clear again
    assert int(flag.item()) == 0
    h.close()


# ------------------------------------------------------------------ edge values

def _edge_inputs(S, G, P, bf16):
    """Config-like random inputs with edge values planted.  Returns w, v (fp32 [S,P]) and g ([S,G,P] fp32,
    or uint16 bf16 bit patterns)."""
    rng = np.random.default_rng(17)
    w = (rng.standard_normal((S, P)) * 0.05).astype(np.float32)
    v = (rng.standard_normal((S, P)) * 0.01).astype(np.float32)
    gf = (rng.standard_normal((S, G, P)) * 1e-3).astype(np.float32)
    sub = np.float32(1e-45)
    w[:, 0:8] = np.array([sub, -sub, 3 * sub, 1e-39, -1e-39, 0.0, -0.0, 1.1754942e-38], np.float32)
    v[:, 0:8] = 0.0
    w[0, 16], w[1, 16] = 3.0e38, 3.0e38                      # u_s + u_p overflows before the 1/2
    w[2, 17] = np.inf; w[3, 18] = -np.inf; w[0, 19] = np.nan; v[3, 21] = np.inf
    w[2, 24:28] = np.array([3.3965e38, -3.3965e38, 3.3895e38, 3.39e38], np.float32)   # around the largest bf16 (unmixed member 2)
    v[2, 24:28] = 0.0
    w[1, 30] = np.float32(np.uint32(0x7F800001).view(np.float32))            # a NaN whose upper mantissa bits are zero
    if bf16:
        from fixtures import generator as gen
        g = gen.f32_to_bf16_bits(gf)
        g[:, :, 0:8] = 0
        g[:, :, 24:28] = 0
        g[2, :, 8:12] = np.array([0x0001, 0x007F, 0x8001, 0x0080], np.uint16)   # subnormal bf16 gradients, all learners
        v[2, 8:12] = 0.0
        g[0, 0, 12:16] = np.array([0x0001, 0x8001, 0x007F, 0x0002], np.uint16)  # ... and in one learner only
        g[0, 1:, 12:16] = 0
        g[1, 0, 20] = 0x7FC0                                  # NaN
        g[2, 1, 22], g[2, 0, 22] = 0x7F80, 0xFF80             # Inf - Inf in the learner sum -> NaN
        g[3, 0, 23] = 0x7F7F                                  # largest finite bf16
    else:
        g = gf
        g[:, :, 0:8] = 0.0
        g[:, :, 24:28] = 0.0
        g[2, :, 8:16] = sub
        g[1, 0, 20] = np.nan
        g[2, 1, 22], g[2, 0, 22] = np.inf, -np.inf
    return w, v, g


def _same_special(got, want, exact, what):
    assert np.array_equal(np.isnan(got), np.isnan(want)), what
    assert np.array_equal(np.isposinf(got), np.isposinf(want)) and np.array_equal(np.isneginf(got), np.isneginf(want)), what
    fin = np.isfinite(want)
    if exact:
        assert np.array_equal(bits(got)[fin], bits(want)[fin]), what
    else:
        with np.errstate(all="ignore"):
            assert np.all(np.abs(got[fin] - want[fin]) <= 1e-6 + 1e-5 * np.abs(want[fin])), what


@pytest.mark.parametrize("variant", ["bf16_grads", "emit_f32_grads", "emit_bf16_grads", "share", "share_bf16_grads", "peer", "peer_bf16_grads"])
@pytest.mark.parametrize("exact", [True, False])
def test_edge_values_through_every_kernel_family(H, oracle_mod, torch_cuda, variant, exact):
    """Subnormal / zero / huge / Inf / NaN weights, momenta and (fp32 or bf16) gradients through: the bf16
    gradient loads, the bf16 working copy (16-element store with bf16 gradients, shuffle-paired 8-element
    store with fp32 gradients; pair AND single kernels), the shared-slot walk (CHAIN carry / kSlots), and a
    two-arena peer group whose cross-arena mixes are resolved one step late (resolve_pending) or by
    hadpsgd_peer_flush.  Three steps (four in peer mode), so that every special value also travels through a SECOND mix.  NaN
    and +-Inf must land where the oracle puts them; everything finite matches bit for bit in deterministic
    mode.  A NaN is any NaN (R17), also in the bf16 copy; the copy never turns a NaN into an Inf."""
    torch = torch_cuda
    bf16 = "bf16_grads" in variant
    emit, share, peer = variant.startswith("emit"), variant.startswith("share"), variant.startswith("peer")
    # peer, ring: step 0 mixes inside the arenas, step 1 across them (left pending), step 2 resolves those
    # inside the fused kernel (resolve_pending), step 3 is pending again and is resolved by the flush
    S, G, P, steps = 4, 2, 4096, (4 if peer else 3)
    w, v, g = _edge_inputs(S, G, P, bf16)
    base = H.DETERMINISTIC if exact else 0
    gd = H.BF16 if bf16 else H.F32
    if peer:
        rank_begin = [0, 2, 4]
        hs = [H.Hadpsgd(2, G, [P], gd, base | H.PEER) for _ in range(2)]
        for r, h in enumerate(hs):
            h.hadpsgd_peer_init(r, 2, rank_begin)
        for r, h in enumerate(hs):
            h.hadpsgd_peer_attach(1 - r, hs[1 - r].hadpsgd_peer_stage())
        where = lambda sg: (hs[sg // 2], sg % 2)
    else:
        hs = [H.Hadpsgd(S, G, [P], gd, base | (H.SHARE_PAIR_WEIGHTS if share else 0),
                        working_dtype=H.BF16 if emit else H.F32)]
        where = lambda sg: (hs[0], sg)
    # emit: members 2 and 3 stay unmixed (the single kernel, and huge weights that only overflow in bf16)
    matching = (lambda k: [1, 0, 2, 3]) if emit else (lambda k: None)
    for sg in range(S):
        h, s = where(sg)
        h.hadpsgd_weights(s)[:P] = torch.from_numpy(w[sg]).cuda()
        h.hadpsgd_momentum(s)[:P] = torch.from_numpy(v[sg]).cuda()
        for k in range(G):
            if bf16:
                h.hadpsgd_grads(s, k)[:P].view(torch.int16).copy_(torch.from_numpy(g[sg, k].view(np.int16)).cuda())
            else:
                h.hadpsgd_grads(s, k)[:P] = torch.from_numpy(g[sg, k]).cuda()
    ow, ov = w.copy(), v.copy()
    with np.errstate(all="ignore"):
        for k in range(steps):
            m = matching(k)
            for h in hs:
                if m is None:
                    h.hadpsgd_step(LR, MU, k)
                else:
                    h.hadpsgd_step_matching(LR, MU, k, m)
            oracle_mod.step(g, ow, ov, LR, MU, k, partner=m)
    for h in hs:
        if peer:
            h.hadpsgd_peer_flush()
    torch.cuda.synchronize()
    gw = np.stack([where(sg)[0].hadpsgd_weights(where(sg)[1])[:P].cpu().numpy() for sg in range(S)])
    gv = np.stack([where(sg)[0].hadpsgd_momentum(where(sg)[1])[:P].cpu().numpy() for sg in range(S)])
    _same_special(gw, ow, exact, "weights")
    _same_special(gv, ov, exact, "momentum")
    assert np.isnan(ow).sum() >= 3 and np.isinf(ow).sum() >= 3          # the plants did propagate
    sub = np.float32(1e-45)
    assert gw[0, 0] == sub and gw[0, 2] == 3 * sub and gw[0, 1] == -sub  # subnormal weights were not flushed
    if bf16:                                                             # nor were subnormal bf16 gradients
        assert np.all(gv[2, 8:12] != 0) and np.all(np.abs(gv[2, 8:12]) < 1e-37)
    if emit:
        h = hs[0]
        gb = np.stack([h.hadpsgd_weights_bf16(s).view(torch.int16)[:P].cpu().numpy().view(np.uint16) for s in range(S)])
        is_nan = lambda b: ((b & 0x7F80) == 0x7F80) & ((b & 0x007F) != 0)
        assert np.array_equal(is_nan(gb), np.isnan(gw))                  # a NaN weight gives a NaN copy, never an Inf
        want_b = oracle_mod.round_bf16(gw)                               # correct rounding of the GPU's own w'
        ok = ~np.isnan(gw)
        assert np.array_equal(gb[ok], want_b[ok])
        if exact:
            assert np.array_equal(gb[ok], oracle_mod.round_bf16(ow)[ok])
        # member 2 is unmixed with zero gradients and momentum: its huge weights are unchanged in fp32 ...
        assert np.array_equal(bits(gw[2, 24:28]), bits(w[2, 24:28]))
        # ... and round to +Inf, -Inf, the largest bf16, the largest bf16 in the copy
        assert [int(x) for x in gb[2, 24:28]] == [0x7F80, 0xFF80, 0x7F7F, 0x7F7F]
    for h in hs:
        h.close()


# ------------------------------------------------------------------ every element at full size

def every_element(H, oracle_mod, torch, name, *, exact=True, flags=0, emit=False, steps=2, seed=4343):
    """One BASELINE.json config at full size in the launch configuration bench.py times (default grid,
    diagnostics on): after `steps` steps EVERY element of every weight and momentum buffer (and of the bf16
    working copy) is compared with the oracle, and the three a5 sums of every step with the oracle's double
    accumulators added up over the windows.  The oracle stays single-threaded per call; disjoint windows
    run on one host thread per core.  Oracle inputs come from the device twin of the seeded generator
    (bit-compared with the numpy one in test_device_generator_matches_host).  Returns the element count."""
    from fixtures import device, generator as gen, problem, shapes
    cfg = shapes.CONFIGS[name]
    S, G, seg_len = cfg["S"], cfg["G"], cfg["seg_len"]
    bf16 = cfg["grad"] == "bf16"
    P = int(sum(seg_len))
    h = H.Hadpsgd(S, G, seg_len, H.BF16 if bf16 else H.F32, (H.DETERMINISTIC if exact else 0) | flags,
                  working_dtype=H.BF16 if emit else H.F32)
    flat = h.P_padded == P
    problem.fill_weights(h, seed)
    gdiag = []
    for k in range(steps):
        problem.fill_grads(h, seed, k, cfg["dist"])
        h.hadpsgd_step(LR, MU, k)
        gdiag.append(h.hadpsgd_diagnostics())
    torch.cuda.synchronize()
    assert h.hadpsgd_launch_count() == steps
    n_threads = os.cpu_count() or 1
    W = 1 << 20
    odiag = [{q: np.zeros(S) for q in ("gsq", "wsq", "gap")} for _ in range(steps)]
    compared = 0

    def check(lo, hi, w0, grads, gw, gv, gb):
        ow, ov = w0, np.zeros((S, hi - lo), np.float32)
        ds = [oracle_mod.step(grads[k], ow, ov, LR, MU, k, diag=True) for k in range(steps)]
        if exact:
            bad = int(np.sum(bits(gw) != bits(ow))) + int(np.sum(bits(gv) != bits(ov)))
        else:
            bad = int(np.sum(np.abs(gw - ow) > 1e-6 + 1e-5 * np.abs(ow))) + int(np.sum(np.abs(gv - ov) > 1e-6 + 1e-5 * np.abs(ov)))
        if gb is not None:      # the copy is the correct rounding of the GPU's w' (and of the oracle's, when exact)
            bad += int(np.sum(gb != oracle_mod.round_bf16(ow if exact else gw)))
        return lo, hi, bad, ds

    def drain(f):
        nonlocal compared
        lo_, hi_, bad, ds = f.result()
        assert bad == 0, (name, lo_, hi_, bad)
        compared += S * (hi_ - lo_)
        for k in range(steps):
            for q in ("gsq", "wsq", "gap"):
                odiag[k][q] += ds[k][q]

    dev_w0 = torch.empty((S, W), dtype=torch.float32, device="cuda")
    dev_g = torch.empty((steps, S, G, W), dtype=torch.bfloat16 if bf16 else torch.float32, device="cuda")
    futures = []
    with ThreadPoolExecutor(max_workers=n_threads) as pool:
        for lo in range(0, P, W):
            hi = min(lo + W, P)
            n = hi - lo
            for s in range(S):
                device.fill(dev_w0[s], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, s, 0), "normal", 0.05, elem_offset=lo, n=n)
                for k in range(steps):
                    for g in range(G):
                        device.fill(dev_g[k, s, g], gen.stream_key(seed, gen.STREAM_GRAD, k, s, g), cfg["dist"], 1e-3,
                                    elem_offset=lo, n=n)
            w0 = np.ascontiguousarray(dev_w0[:, :n].cpu().numpy())
            if bf16:
                grads = [np.ascontiguousarray(dev_g[k, :, :, :n].view(torch.int16).cpu().numpy().view(np.uint16)) for k in range(steps)]
            else:
                grads = [np.ascontiguousarray(dev_g[k, :, :, :n].cpu().numpy()) for k in range(steps)]
            idx = slice(lo, hi) if flat else torch.from_numpy(problem.padded_index(seg_len, h.layout["seg_offset"], lo, hi)).cuda()
            gw = np.stack([h.hadpsgd_weights(s)[idx].cpu().numpy() for s in range(S)])
            gv = np.stack([h.hadpsgd_momentum(s)[idx].cpu().numpy() for s in range(S)])
            gb = np.stack([h.hadpsgd_weights_bf16(s).view(torch.int16)[idx].cpu().numpy().view(np.uint16) for s in range(S)]) if emit else None
            futures.append(pool.submit(check, lo, hi, w0, grads, gw, gv, gb))
            while len(futures) > 2 * n_threads:           # bound the host memory in flight
                drain(futures.pop(0))
        for f in futures:
            drain(f)
    assert compared == S * P                              # every element of every buffer
    for k in range(steps):                                # a5 against the oracle's double accumulators (Q16: rel 1e-4)
        for q in ("gsq", "wsq", "gap"):
            assert np.allclose(gdiag[k][q], odiag[k][q], rtol=1e-4, atol=0), (name, k, q, gdiag[k][q], odiag[k][q])
        assert np.all(odiag[k]["gap"] > 0)
    if not flat:                                          # padding stays zero in w, v (and the copy)
        nat = torch.from_numpy(h.natural_index()).cuda()
        mask = torch.ones(h.P_padded, dtype=torch.bool, device="cuda"); mask[nat] = False
        for s in range(S):
            assert not h.hadpsgd_weights(s)[mask].any() and not h.hadpsgd_momentum(s)[mask].any()
            if emit:
                assert not h.hadpsgd_weights_bf16(s).view(torch.int16)[mask].any()
    h.close()
    del dev_w0, dev_g
    torch.cuda.empty_cache()
    return compared


def test_every_element_config3_ragged_bf16(H, oracle_mod, torch_cuda):
    """configs[3]: 8 x 8 learners, bf16 gradients, 40 ragged segments -- the 224-thread G = 8 bf16 kernel."""
    assert every_element(H, oracle_mod, torch_cuda, "swb2000_ragged_bf16") == 8 * 145_145_344


def test_every_element_paper_literal(H, oracle_mod, torch_cuda):
    """The paper-literal 43,130,368-parameter model, 8 x 8 fp32 -- the 160-thread G = 8 fp32 kernel."""
    assert every_element(H, oracle_mod, torch_cuda, "paper_literal") == 8 * 43_130_368


def test_every_element_config1_swb300(H, oracle_mod, torch_cuda):
    assert every_element(H, oracle_mod, torch_cuda, "swb300") == 16 * 94_797_312


def test_every_element_swb2000_bf16_working_copy(H, oracle_mod, torch_cuda):
    """Headline shape with the bf16 working copy (row f2; the 192-thread kernel): w, v and the copy."""
    every_element(H, oracle_mod, torch_cuda, "swb2000", emit=True)


def test_every_element_swb2000_shared_pair_weights(H, oracle_mod, torch_cuda):
    """Headline shape with HADPSGD_SHARE_PAIR_WEIGHTS (the CHAIN walk over shared slots)."""
    every_element(H, oracle_mod, torch_cuda, "swb2000", flags=H.SHARE_PAIR_WEIGHTS)


def test_every_element_swb2000_default_mode(H, oracle_mod, torch_cuda):
    """Headline shape in DEFAULT mode (FMA contraction allowed): every element within the stated
    tolerance 1e-6 + 1e-5 |x| (north_star), diagnostics at rel 1e-4 -- the kernel bench.py times."""
    every_element(H, oracle_mod, torch_cuda, "swb2000", exact=False)


# ------------------------------------------------------------------ neighbour-only epoch handshake (row f4)

@pytest.mark.parametrize("delay_rank", [None, 0, 2])
def test_peer_ranks_on_their_own_streams_are_ordered_by_the_epoch_handshake(H, oracle_mod, torch_cuda, delay_rank):
    """Four HADPSGD_PEER handles ("ranks") on ONE GPU, each on a stream of its own, stepped without any
    host synchronisation or shared stream in between: what orders rank r's step e + 1 behind its partners'
    step e is the library's neighbour-only handshake (no global barrier).  Ring steps,
    then custom matchings with far partners and unmixed members; bit-exact against the oracle.  With one
    rank delayed by a ~1 s spin on its stream, its partner is shown to be BLOCKED (stream not idle) while
    the sleeper runs, and the results are still exact -- without the waits the partner would have read a
    stage buffer that had not been written yet."""
    torch = torch_cuda
    from fixtures import device, generator as gen, problem
    rank_begin, G, P, seed = [0, 2, 4, 6, 8], 2, 300_007, 907
    R, S = len(rank_begin) - 1, rank_begin[-1]
    streams = [torch.cuda.Stream() for _ in range(R)]
    hs = [H.Hadpsgd(2, G, [P], H.F32, H.PEER | H.DETERMINISTIC, stream=streams[r]) for r in range(R)]
    for r, h in enumerate(hs):
        h.hadpsgd_peer_init(r, R, rank_begin)
    for r, h in enumerate(hs):
        for q, other in enumerate(hs):
            if q != r:
                h.hadpsgd_peer_attach(q, other.hadpsgd_peer_stage())
    for sg in range(S):                       # ONE set of gradients, reused by every step: nothing to refill in between
        h, s = hs[sg // 2], sg % 2
        device.fill(h.hadpsgd_weights(s)[:P], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, sg, 0), "normal", 0.05)
        for g in range(G):
            device.fill(h.hadpsgd_grads(s, g)[:P], gen.stream_key(seed, gen.STREAM_GRAD, 0, sg, g), "normal", 1e-3)
    torch.cuda.synchronize()
    ring = lambda k: [(s + 1 if s % 2 == 0 else s - 1) if k % 2 == 0 else ((s + 1) % S if s % 2 == 1 else (s - 1) % S) for s in range(S)]
    matchings = [None] * 6 + [[7, 6, 5, 4, 3, 2, 1, 0], [1, 0, 3, 2, 5, 4, 7, 6], [0, 2, 1, 4, 3, 6, 5, 7],
                              [4, 5, 6, 7, 0, 1, 2, 3], None, None]
    for k, m in enumerate(matchings):                      # enqueue everything; the host never waits for the GPU
        if k == 2 and delay_rank is not None:              # (the first step of a handle uploads its peer table and
            with torch.cuda.stream(streams[delay_rank]):   # synchronises its stream once, so the delay comes later)
                torch.cuda._sleep(2_000_000_000)           # about a second
        for h in hs:
            if m is None:
                h.hadpsgd_step(LR, MU, k)
            else:
                h.hadpsgd_step_matching(LR, MU, k, m)
    if delay_rank is not None:
        # step 1 published u across the arenas ((1,2) (3,4) (5,6) (7,0)) into stage parity 1 and step 2
        # resolves it; step 3 publishes into parity 1 again, so the sleeper's ring neighbours are stuck in
        # front of their step 3 until the sleeper has finished ITS step 2 (the reader of what they overwrite)
        assert not streams[delay_rank].query()
        assert not streams[(delay_rank + 1) % R].query() and not streams[(delay_rank - 1) % R].query()
    for h in hs:
        h.hadpsgd_peer_flush()
    torch.cuda.synchronize()
    og = problem.host_grads(seed, 0, S, G, 0, P)
    ow, ov = problem.host_weights(seed, S, 0, P), np.zeros((S, P), np.float32)
    for k, m in enumerate(matchings):
        oracle_mod.step(og, ow, ov, LR, MU, k, partner=m if m is not None else ring(k))
    gw = np.stack([hs[sg // 2].hadpsgd_weights(sg % 2)[:P].cpu().numpy() for sg in range(S)])
    gv = np.stack([hs[sg // 2].hadpsgd_momentum(sg % 2)[:P].cpu().numpy() for sg in range(S)])
    assert np.array_equal(bits(gw), bits(ow)) and np.array_equal(bits(gv), bits(ov))
    for h in hs:
        h.close()


def test_every_element_peer_group_of_8_at_full_size(H, oracle_mod, torch_cuda):
    """The super-learner partition at the headline size, in the shape `bench.py --emulate-ranks 8` times: 8
    HADPSGD_PEER arenas of 2 x 145,145,344 parameters on one GPU (74 GB), ring steps 0..3 (inside the
    arenas, across them, resolve inside the fused kernel, across them again) and a final flush.  EVERY
    element of all 16 weight and momentum buffers against the oracle, bit for bit, and the a5 sums of every
    step against the oracle's double accumulators: gsq at once; wsq / gap at once for members whose mix
    finished inside the step, and as pend_wsq / pend_gap of the NEXT step (or of the flush) for members
    whose partner lives in another arena.  This is the kPeer kernel on a grid that is busy for thousands of
    tiles per block, which the small peer tests never reach."""
    torch = torch_cuda
    from fixtures import device, generator as gen, problem, shapes
    cfg = shapes.CONFIGS["swb2000"]
    S, G, P, R, steps, seed = cfg["S"], cfg["G"], int(sum(cfg["seg_len"])), 8, 4, 5151
    S_l = S // R
    rank_begin = [r * S_l for r in range(R + 1)]
    hs = [H.Hadpsgd(S_l, G, [P], H.F32, H.PEER | H.DETERMINISTIC) for _ in range(R)]
    for r, h in enumerate(hs):
        h.hadpsgd_peer_init(r, R, rank_begin)
    for r, h in enumerate(hs):
        for q, other in enumerate(hs):
            if q != r:
                h.hadpsgd_peer_attach(q, other.hadpsgd_peer_stage())
    where = lambda sg: (hs[sg // S_l], sg % S_l)
    for sg in range(S):
        h, s = where(sg)
        device.fill(h.hadpsgd_weights(s), gen.stream_key(seed, gen.STREAM_WEIGHT, 0, sg, 0), "normal", 0.05)
    gdiag = []                                             # [step][rank] -> diagnostics dict
    for k in range(steps):
        for sg in range(S):
            h, s = where(sg)
            for g in range(G):
                device.fill(h.hadpsgd_grads(s, g), gen.stream_key(seed, gen.STREAM_GRAD, k, sg, g), "normal", 1e-3)
        for h in hs:                                       # one stream, epoch by epoch
            h.hadpsgd_step(LR, MU, k)
        gdiag.append([h.hadpsgd_diagnostics() for h in hs])
    for h in hs:
        h.hadpsgd_peer_flush()
    after_flush = [h.hadpsgd_diagnostics() for h in hs]
    torch.cuda.synchronize()
    launches = sum(h.hadpsgd_launch_count() for h in hs)
    n_threads = os.cpu_count() or 1
    W = 1 << 20
    odiag = [{q: np.zeros(S) for q in ("gsq", "wsq", "gap")} for _ in range(steps)]
    compared = 0

    def check(lo, hi, w0, grads, gw, gv):
        ow, ov = w0, np.zeros((S, hi - lo), np.float32)
        ds = [oracle_mod.step(grads[k], ow, ov, LR, MU, k, diag=True) for k in range(steps)]
        return lo, hi, int(np.sum(bits(gw) != bits(ow))) + int(np.sum(bits(gv) != bits(ov))), ds

    def drain(f):
        nonlocal compared
        lo_, hi_, bad, ds = f.result()
        assert bad == 0, (lo_, hi_, bad)
        compared += S * (hi_ - lo_)
        for k in range(steps):
            for q in ("gsq", "wsq", "gap"):
                odiag[k][q] += ds[k][q]

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
            gw = np.stack([where(sg)[0].hadpsgd_weights(where(sg)[1])[lo:hi].cpu().numpy() for sg in range(S)])
            gv = np.stack([where(sg)[0].hadpsgd_momentum(where(sg)[1])[lo:hi].cpu().numpy() for sg in range(S)])
            futures.append(pool.submit(check, lo, hi, w0, grads, gw, gv))
            while len(futures) > 2 * n_threads:
                drain(futures.pop(0))
        for f in futures:
            drain(f)
    assert compared == S * P
    close = lambda a, b: np.allclose(a, b, rtol=1e-4, atol=0)
    n_pending = 0
    for k in range(steps):
        owed_by = gdiag[k + 1] if k + 1 < steps else after_flush        # who delivers what step k left pending
        for r in range(R):
            lo, hi = rank_begin[r], rank_begin[r + 1]
            d = gdiag[k][r]
            assert close(d["gsq"], odiag[k]["gsq"][lo:hi]), (k, r)
            pend = d["pending"] == 1
            n_pending += int(pend.sum())
            assert close(d["wsq"][~pend], odiag[k]["wsq"][lo:hi][~pend]) and close(d["gap"][~pend], odiag[k]["gap"][lo:hi][~pend]), (k, r)
            assert close(owed_by[r]["pend_wsq"][pend], odiag[k]["wsq"][lo:hi][pend]), (k, r)
            assert close(owed_by[r]["pend_gap"][pend], odiag[k]["gap"][lo:hi][pend]), (k, r)
            assert not owed_by[r]["pend_wsq"][~pend].any() and not owed_by[r]["pend_gap"][~pend].any(), (k, r)
    assert n_pending == 2 * S                              # steps 1 and 3: every member's ring partner is in another arena
    assert not any(d["pending"].any() for d in after_flush)
    # launches: steps 0 and 1 one plain pair / single launch per rank, step 2 one pending-pair launch, step 3
    # one single launch, then one flush (two kernels, counted once)
    assert launches == R * (steps + 1), launches
    for h in hs:
        h.close()
    del dev_w0, dev_g
    torch.cuda.empty_cache()
