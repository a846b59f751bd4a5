"""Pins for the CPU oracle (oracle/) against what the paper and the mathematics fix.

None of these re-types the oracle's loop: each compares it with something independent --
exact rational arithmetic, a closed form, a dense mixing-matrix product, an invariant of
doubly stochastic matrices, or a special case that collapses to eq. (3)/(6) of PAPER.md.
Citations are PAPER.md:<line>.  Runs on CPU (-m "not gpu").
"""
from fractions import Fraction

import numpy as np
import pytest

from fixtures import generator as gen

LR, MU = 0.1, 0.9


def rand(shape, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(shape) * scale).astype(np.float32)


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


# ------------------------------------------------------------------ pairing / T_k

def paper_T(S, step_k):
    """T_k built here from the prose, independently of the oracle: even step pairs
    (2i,2i+1), odd step pairs (2i+1,(2i+2) mod S); averaging a pair puts 0.5 at the four
    positions (a,a),(a,b),(b,a),(b,b)."""
    T = np.zeros((S, S))
    if S == 1:
        T[0, 0] = 1.0
        return T
    for i in range(S // 2):
        a, b = (2 * i, 2 * i + 1) if step_k % 2 == 0 else (2 * i + 1, (2 * i + 2) % S)
        for x in (a, b):
            for y in (a, b):
                T[x, y] = 0.5
    return T


@pytest.mark.parametrize("S", [2, 4, 6, 8, 16, 64])
@pytest.mark.parametrize("step_k", [0, 1, 2, 7])
def test_mixing_matrix_structure(oracle_mod, S, step_k):
    T = oracle_mod.mixing_matrix(S, step_k)
    assert np.array_equal(T, T.T)                       # symmetric
    assert np.array_equal(T.sum(0), np.ones(S))         # doubly stochastic
    assert np.array_equal(T.sum(1), np.ones(S))
    assert set(np.unique(T)) <= {0.0, 0.5}
    assert np.all((T == 0.5).sum(0) == 2) and np.all((T == 0.5).sum(1) == 2)  # "two 0.5s"
    assert np.array_equal(T @ T, T)                     # pair projector: idempotent
    assert np.array_equal(T, paper_T(S, step_k))
    p = oracle_mod.partner(S, step_k)
    assert np.array_equal(p[p], np.arange(S)) and np.all(p != np.arange(S))  # perfect matching
    # ring neighbours only: partner is s+1 or s-1 mod S
    assert np.all(((p - np.arange(S)) % S == 1) | ((p - np.arange(S)) % S == S - 1))


def test_pairing_alternates_and_covers_ring(oracle_mod):
    S = 8
    even, odd = oracle_mod.partner(S, 0), oracle_mod.partner(S, 1)
    assert list(even) == [1, 0, 3, 2, 5, 4, 7, 6]
    assert list(odd) == [7, 2, 1, 4, 3, 6, 5, 0]
    assert np.array_equal(oracle_mod.partner(S, 10), even)
    assert np.array_equal(oracle_mod.partner(S, 11), odd)
    # union of the two matchings is the whole ring (every node talks left and right)
    edges = {frozenset((s, int(even[s]))) for s in range(S)} | {frozenset((s, int(odd[s]))) for s in range(S)}
    assert edges == {frozenset((s, (s + 1) % S)) for s in range(S)}


def test_pairing_degenerate(oracle_mod):
    assert list(oracle_mod.partner(1, 0)) == [0]
    assert list(oracle_mod.partner(2, 0)) == [1, 0]
    assert list(oracle_mod.partner(2, 1)) == [1, 0]      # S=2: odd pair (1,0) is the same pair
    for S in (3, 5, 7):
        with pytest.raises(ValueError):
            oracle_mod.partner(S, 0)                      # reading R8: no perfect matching
    with pytest.raises(ValueError):
        oracle_mod.partner(0, 0)


# ------------------------------------------------------------------ eq. (3): plain SGD

def test_reduces_to_eq3_bit_exact(oracle_mod):
    """S=1, G=1, mu=0: w' = w - lr*g, one fp32 multiply then one fp32 subtract."""
    P = 4099
    w, g = rand((1, P), 1, 0.05), rand((1, 1, P), 2, 1e-3)
    expect_w = w - np.float32(LR) * g[0]          # numpy fp32: mul rounded, then sub rounded
    v = np.zeros((1, P), np.float32)
    oracle_mod.step(g, w, v, LR, 0.0, 0)
    assert np.array_equal(bits(w), bits(expect_w))
    assert np.array_equal(bits(v), bits(g[0]))     # v = 0*0 + g


def test_exact_rational_worked_example(oracle_mod):
    """Hand-checkable case with dyadic inputs where EVERY fp32 operation is exact, so the
    expected result is the exact rational value of
        v' = mu v + (1/G) sum_g g ;  u = w - lr v' ;  w' = (u_s + u_p)/2
    computed with fractions.Fraction.  Catches a dropped term, a wrong sign, a swapped
    index or operand (all four super-learners and both learners carry distinct values)."""
    S, G, P = 4, 2, 3
    F = Fraction
    lr, mu = F(1, 2), F(1, 4)
    w = [[F(s * 8 + i, 16) for i in range(P)] for s in range(S)]
    v = [[F(-(s + 1) * (i + 2), 32) for i in range(P)] for s in range(S)]
    g = [[[F((s * 5 + gg * 3 + i * 7) % 11 - 5, 8) for i in range(P)] for gg in range(G)] for s in range(S)]
    for step_k in (0, 1):
        wn = np.array([[float(x) for x in r] for r in w], np.float32)
        vn = np.array([[float(x) for x in r] for r in v], np.float32)
        gn = np.array([[[float(x) for x in r] for r in q] for q in g], np.float32)
        oracle_mod.step(gn, wn, vn, float(lr), float(mu), step_k)
        v = [[mu * v[s][i] + sum(g[s][gg][i] for gg in range(G)) / G for i in range(P)] for s in range(S)]
        u = [[w[s][i] - lr * v[s][i] for i in range(P)] for s in range(S)]
        pairs = [(0, 1), (2, 3)] if step_k == 0 else [(1, 2), (3, 0)]
        w = [[None] * P for _ in range(S)]
        for a, b in pairs:
            for i in range(P):
                w[a][i] = w[b][i] = (u[a][i] + u[b][i]) / 2
        for s in range(S):
            for i in range(P):
                assert F(float(vn[s, i])) == v[s][i], (step_k, s, i)
                assert F(float(wn[s, i])) == w[s][i], (step_k, s, i)


# ------------------------------------------------------------------ momentum closed form (reading R2)

def test_momentum_closed_form(oracle_mod):
    """Constant gradient g, S=G=1: v_k = g (1-mu^k)/(1-mu),
    w_k = w_0 - lr g [k - mu (1-mu^k)/(1-mu)]/(1-mu)  (sum of the geometric series)."""
    P, K = 257, 20
    w0 = rand((1, P), 3, 0.05)
    g = rand((1, 1, P), 4, 1e-3)
    gd, wd = g[0].astype(np.float64), w0.astype(np.float64)
    lr, mu = np.float64(np.float32(LR)), np.float64(np.float32(MU))   # the fp32 values actually used
    w32, v32 = w0.copy(), np.zeros((1, P), np.float32)
    w64, v64 = wd.copy(), np.zeros((1, P), np.float64)
    for k in range(1, K + 1):
        oracle_mod.step(g, w32, v32, LR, MU, k - 1)
        oracle_mod.step_f64(g, w64, v64, float(lr), float(mu), k - 1)
        v_cf = gd * (1 - mu ** k) / (1 - mu)
        w_cf = wd - lr * gd * (k - mu * (1 - mu ** k) / (1 - mu)) / (1 - mu)
        assert np.allclose(v64, v_cf, rtol=1e-12, atol=1e-18)
        assert np.allclose(w64, w_cf, rtol=1e-12, atol=1e-18)
        assert np.all(np.abs(w32 - w_cf) <= 1e-6 + 1e-5 * np.abs(w_cf))
        assert np.all(np.abs(v32 - v_cf) <= 1e-6 + 1e-5 * np.abs(v_cf))


# ------------------------------------------------------------------ eq. (4)/(6): the mean

@pytest.mark.parametrize("G", [1, 2, 4])
def test_mean_of_identical_gradients_is_exact(oracle_mod, G):
    P = 5003
    g1 = rand((2, 1, P), 5, 1e-3)
    gG = np.ascontiguousarray(np.repeat(g1, G, axis=1))
    w1, v1 = rand((2, P), 6, 0.05), rand((2, P), 7, 0.01)
    wG, vG = w1.copy(), v1.copy()
    oracle_mod.step(g1, w1, v1, LR, MU, 0)
    oracle_mod.step(gG, wG, vG, LR, MU, 0)
    assert np.array_equal(bits(w1), bits(wG)) and np.array_equal(bits(v1), bits(vG))


def test_mean_of_identical_bf16_gradients_exact_for_G8(oracle_mod):
    """bf16 values have 8 significant bits, so k*g (k<=8) is exact in fp32 and the
    left-to-right sum of 8 copies times 1/8 returns g exactly."""
    P, G = 4001, 8
    gb = gen.f32_to_bf16_bits(rand((2, 1, P), 8, 1e-3))
    g1f = gen.bf16_bits_to_f32(gb)                       # the same values as fp32 gradients
    gG = np.ascontiguousarray(np.repeat(gb, G, axis=1))
    w1, v1 = rand((2, P), 9, 0.05), np.zeros((2, P), np.float32)
    wG, vG = w1.copy(), v1.copy()
    oracle_mod.step(g1f, w1, v1, LR, MU, 1)
    oracle_mod.step(gG, wG, vG, LR, MU, 1)
    assert np.array_equal(bits(w1), bits(wG)) and np.array_equal(bits(v1), bits(vG))


def test_mean_uses_every_learner_once(oracle_mod):
    """Gradient of learner g is 2^g at element g, 0 elsewhere: the mean must be 2^g/G there
    (exact), which fails if a learner is dropped, doubled or mis-strided."""
    S, G = 2, 8
    g = np.zeros((S, G, G), np.float32)
    for s in range(S):
        for k in range(G):
            g[s, k, k] = 2.0 ** k * (s + 1)
    w, v = np.zeros((S, G), np.float32), np.zeros((S, G), np.float32)
    oracle_mod.step(g, w, v, 1.0, 0.0, 0, flags=oracle_mod.NO_MIX)
    for s in range(S):
        assert np.array_equal(v[s], (2.0 ** np.arange(G) * (s + 1) / G).astype(np.float32))
        assert np.array_equal(w[s], -v[s])


# ------------------------------------------------------------------ eq. (7): dense T_k brute force

@pytest.mark.parametrize("S,G", [(2, 1), (4, 2), (6, 3), (8, 4)])
@pytest.mark.parametrize("step_k", [0, 1])
def test_matches_dense_mixing_matrix(oracle_mod, S, G, step_k):
    """W' = (W - lr V') T_k with T_k the dense S x S matrix built in THIS file from the
    prose.  The product is formed in float64 (0.5a+0.5b is exact there) and rounded once,
    which equals fl32(0.5*fl32(a+b)) barring underflow."""
    P = 61
    g, w, v = rand((S, G, P), 10, 1e-3), rand((S, P), 11, 0.05), rand((S, P), 12, 0.01)
    invG = np.float32(1.0) / np.float32(G)
    acc = g[:, 0].copy()
    for k in range(1, G):
        acc = acc + g[:, k]
    vn = np.float32(MU) * v + acc * invG
    u = w - np.float32(LR) * vn                           # columns = learners: U is [S,P] = Theta^T
    Wd = (paper_T(S, step_k) @ u.astype(np.float64))      # (Theta T)^T = T^T Theta^T = T Theta^T
    sum32 = np.stack([u[s] + u[int(np.argmax(paper_T(S, step_k)[s] * (np.arange(S) != s)))] for s in range(S)])
    expect = (np.float32(0.5) * sum32)
    assert np.allclose(Wd, expect.astype(np.float64), rtol=1e-7, atol=0)   # dense product agrees
    d = oracle_mod.step(g, w, v, LR, MU, step_k, diag=True)
    assert np.array_equal(bits(v), bits(vn))
    assert np.array_equal(bits(w), bits(expect))
    assert np.max(np.abs(w.astype(np.float64) - Wd)) <= 2 ** -24 * np.max(np.abs(Wd))
    # diagnostics against numpy in double
    assert np.allclose(d["gsq"], ((acc * invG).astype(np.float64) ** 2).sum(1), rtol=1e-12)
    assert np.allclose(d["wsq"], (w.astype(np.float64) ** 2).sum(1), rtol=1e-12)
    p = oracle_mod.partner(S, step_k)
    assert np.allclose(d["gap"], ((u.astype(np.float64) - u[p].astype(np.float64)) ** 2).sum(1), rtol=1e-12)


def test_eq7_literal_variant_matches_dense(oracle_mod):
    """Flag EQ7_LITERAL: Theta_{k+1} = Theta_k T_k - lr V' exactly as printed."""
    S, G, P = 4, 2, 33
    g, w, v = rand((S, G, P), 13, 1e-3), rand((S, P), 14, 0.05), rand((S, P), 15, 0.01)
    w64, v64 = w.astype(np.float64), v.astype(np.float64)
    vn = np.float64(np.float32(MU)) * v64 + g.astype(np.float64).mean(1)
    expect = paper_T(S, 1) @ w64 - np.float64(np.float32(LR)) * vn
    oracle_mod.step(g, w, v, LR, MU, 1, flags=oracle_mod.EQ7_LITERAL)
    assert np.all(np.abs(w - expect) <= 1e-6 + 1e-5 * np.abs(expect))
    oracle_mod.step_f64(g, w64, v64, float(np.float32(LR)), float(np.float32(MU)), 1,
                        flags=oracle_mod.EQ7_LITERAL)
    assert np.allclose(w64, expect, rtol=1e-13, atol=1e-16)


# ------------------------------------------------------------------ caller-supplied matchings, unmixed members,
# ------------------------------------------------------------------ eq.-(7)-literal diagnostics (R8, R14)

def matching_T(partner):
    """Dense T_k for an arbitrary matching, built HERE from PAPER.md:66 generalised by DESIGN.md R8:
    a pair (a,b) puts 0.5 at (a,a),(a,b),(b,a),(b,b); an unmixed member s has T_ss = 1."""
    S = len(partner)
    T = np.zeros((S, S))
    for s, p in enumerate(partner):
        if p == s:
            T[s, s] = 1.0
        else:
            T[s, s] = T[s, p] = 0.5
    return T


def fl32_sub(a32, b32):
    """Correctly rounded fp32 a - b: the difference of two fp32 values of nearby magnitude is exact
    in double, so one rounding of the double result is the IEEE fp32 subtraction."""
    return (a32.astype(np.float64) - b32.astype(np.float64)).astype(np.float32)


def fl32_mul(a32, b32):
    """Correctly rounded fp32 product: 24 x 24 significant bits fit a double exactly."""
    return (np.asarray(a32, np.float32).astype(np.float64) * np.asarray(b32, np.float32).astype(np.float64)).astype(np.float32)


MATCHINGS = [[1, 0, 2], [0, 1, 2, 3, 4], [4, 3, 2, 1, 0], [3, 1, 5, 0, 4, 2, 6], [1, 0, 3, 2, 5, 4, 7, 6],
             [7, 2, 1, 4, 3, 6, 5, 0], [5, 4, 3, 2, 1, 0], [0]]


@pytest.mark.parametrize("partner", MATCHINGS)
@pytest.mark.parametrize("literal", [False, True])
def test_matching_entry_against_dense_T(oracle_mod, partner, literal):
    """hadpsgd_oracle_step_matching for any involution (odd S, unmixed members, non-neighbours):
    weights bit for bit against the dense product with T built in this file, momentum against the
    per-learner update, and all three diagnostics against numpy in double (R14):
      default  W' = fl32(T (W - lr V'))             gap = |u_s - u_p|^2
      literal  W' = fl32( fl32(T W) - fl32(lr V') ) gap = |w_s - w_p|^2 (OLD weights)
    gap is exactly 0 for an unmixed member either way."""
    S, G, P = len(partner), 3, 67
    g, w, v = rand((S, G, P), 200 + S, 1e-3), rand((S, P), 201 + S, 0.05), rand((S, P), 202 + S, 0.01)
    w_old = w.copy()
    T = matching_T(partner)
    assert np.array_equal(oracle_mod.mixing_matrix_matching(partner), T)
    assert np.array_equal(T, T.T) and np.array_equal(T.sum(0), np.ones(S)) and np.array_equal(T @ T, T)
    acc = g[:, 0].copy()
    for k in range(1, G):
        acc = acc + g[:, k]
    gbar = acc * (np.float32(1.0) / np.float32(G))
    vn = np.float32(MU) * v + gbar
    t = fl32_mul(np.float32(LR), vn)
    if literal:
        m = (T @ w_old.astype(np.float64)).astype(np.float32)      # 0.5a+0.5b exact in double, one rounding
        expect = fl32_sub(m, t)
        a = w_old
    else:
        u = fl32_sub(w_old, t)
        expect = (T @ u.astype(np.float64)).astype(np.float32)
        a = u
    flags = oracle_mod.EQ7_LITERAL if literal else 0
    d = oracle_mod.step(g, w, v, LR, MU, 0, flags=flags, diag=True, partner=partner)
    assert np.array_equal(bits(v), bits(vn))
    assert np.array_equal(bits(w), bits(expect))
    pt = np.asarray(partner)
    a64 = a.astype(np.float64)
    assert np.allclose(d["gsq"], (gbar.astype(np.float64) ** 2).sum(1), rtol=1e-12, atol=0)
    assert np.allclose(d["wsq"], (expect.astype(np.float64) ** 2).sum(1), rtol=1e-12, atol=0)
    assert np.allclose(d["gap"], ((a64 - a64[pt]) ** 2).sum(1), rtol=1e-12, atol=0)
    for s in range(S):
        if partner[s] == s:
            assert d["gap"][s] == 0.0                              # exactly, not merely small
        else:
            assert d["gap"][s] > 0 and d["gap"][s] == d["gap"][partner[s]]


@pytest.mark.parametrize("literal", [False, True])
def test_matching_entry_f64_shadow(oracle_mod, literal):
    partner = [3, 1, 5, 0, 4, 2, 6]
    S, G, P = 7, 2, 41
    g, w, v = rand((S, G, P), 210, 1e-3), rand((S, P), 211, 0.05), rand((S, P), 212, 0.01)
    w64, v64 = w.astype(np.float64), v.astype(np.float64)
    lr, mu = float(np.float32(LR)), float(np.float32(MU))
    vn = mu * v64 + g.astype(np.float64).mean(1)
    T = matching_T(partner)
    expect = T @ w64 - lr * vn if literal else T @ (w64 - lr * vn)
    flags = oracle_mod.EQ7_LITERAL if literal else 0
    oracle_mod.step_f64(g, w64, v64, lr, mu, 0, flags=flags, partner=partner)
    assert np.allclose(w64, expect, rtol=1e-13, atol=1e-17) and np.allclose(v64, vn, rtol=1e-14, atol=0)
    oracle_mod.step(g, w, v, LR, MU, 0, flags=flags, partner=partner)
    assert np.all(np.abs(w - expect) <= 1e-6 + 1e-5 * np.abs(expect))


def test_matching_entry_equals_ring_entry_on_ring_matchings(oracle_mod):
    S, G, P = 8, 2, 129
    for k in (0, 1):
        for flags in (0, oracle_mod.EQ7_LITERAL):
            g, w, v = rand((S, G, P), 220 + k, 1e-3), rand((S, P), 221, 0.05), rand((S, P), 222, 0.01)
            w2, v2 = w.copy(), v.copy()
            d1 = oracle_mod.step(g, w, v, LR, MU, k, flags=flags, diag=True)
            d2 = oracle_mod.step(g, w2, v2, LR, MU, 99, flags=flags, diag=True, partner=oracle_mod.partner(S, k))
            assert np.array_equal(bits(w), bits(w2)) and np.array_equal(bits(v), bits(v2))
            for name in ("gsq", "wsq", "gap"):
                assert np.array_equal(d1[name], d2[name])


def test_matching_entry_rejects_non_involutions(oracle_mod):
    g, w, v = np.zeros((3, 1, 4), np.float32), np.zeros((3, 4), np.float32), np.zeros((3, 4), np.float32)
    for bad in ([1, 2, 0], [1, 1, 2], [0, 1, 3], [-1, 1, 2]):
        with pytest.raises(ValueError):
            oracle_mod.step(g, w, v, LR, MU, 0, partner=bad)
        with pytest.raises(ValueError):
            oracle_mod.mixing_matrix_matching(bad)
    with pytest.raises(ValueError):
        oracle_mod.step(g, w, v, LR, MU, 0, partner=[0, 1])           # wrong length


@pytest.mark.parametrize("literal", [False, True])
def test_exact_rational_example_with_matching_and_diagnostics(oracle_mod, literal):
    """Dyadic inputs for which EVERY fp32 and double operation is exact, S = 5 with one unmixed
    member and a non-neighbour pair: weights, momentum AND the three diagnostics must equal the
    exact rational values (fractions.Fraction) of
        v' = mu v + (1/G) sum_g g
        default: u = w - lr v' ; w'_s = (u_s + u_p)/2            ; gap = sum (u_s - u_p)^2
        literal: w'_s = (w_s + w_p)/2 - lr v'_s   ; gap = sum (w_s - w_p)^2
        unmixed: w'_s = w_s - lr v'_s                            ; gap = 0
        gsq = sum gbar^2 ; wsq = sum w'^2."""
    F = Fraction
    S, G, P = 5, 2, 3
    partner = [3, 4, 2, 0, 1]                                # pairs (0,3), (1,4); 2 unmixed
    lr, mu = F(1, 2), F(1, 4)
    w = [[F(s * 8 + i * 3 - 7, 16) for i in range(P)] for s in range(S)]
    v = [[F(-(s + 1) * (i + 2), 32) for i in range(P)] for s in range(S)]
    g = [[[F((s * 5 + gg * 3 + i * 7) % 11 - 5, 8) for i in range(P)] for gg in range(G)] for s in range(S)]
    wn = np.array([[float(x) for x in r] for r in w], np.float32)
    vn = np.array([[float(x) for x in r] for r in v], np.float32)
    gn = np.array([[[float(x) for x in r] for r in q] for q in g], np.float32)
    d = oracle_mod.step(gn, wn, vn, float(lr), float(mu), 0, flags=oracle_mod.EQ7_LITERAL if literal else 0,
                        diag=True, partner=partner)
    gbar = [[sum(g[s][gg][i] for gg in range(G)) / G for i in range(P)] for s in range(S)]
    v2 = [[mu * v[s][i] + gbar[s][i] for i in range(P)] for s in range(S)]
    u = [[w[s][i] - lr * v2[s][i] for i in range(P)] for s in range(S)]
    w2 = [[None] * P for _ in range(S)]
    gap = [F(0)] * S
    for s in range(S):
        p = partner[s]
        for i in range(P):
            if literal:
                w2[s][i] = (w[s][i] + w[p][i]) / 2 - lr * v2[s][i]
            else:
                w2[s][i] = (u[s][i] + u[p][i]) / 2
        a = w if literal else u
        gap[s] = sum((a[s][i] - a[p][i]) ** 2 for i in range(P))
    for s in range(S):
        for i in range(P):
            assert F(float(vn[s, i])) == v2[s][i], (s, i)
            assert F(float(wn[s, i])) == w2[s][i], (s, i)
        assert F(float(d["gsq"][s])) == sum(x * x for x in gbar[s]), s
        assert F(float(d["wsq"][s])) == sum(x * x for x in w2[s]), s
        assert F(float(d["gap"][s])) == gap[s], s
    assert gap[2] == 0 and gap[0] == gap[3] != 0 and gap[1] == gap[4] != 0
    if literal:                                                  # pair members end up DIFFERENT (R3)
        assert w2[0] != w2[3]
    else:
        assert w2[0] == w2[3] and w2[1] == w2[4]


def test_eq7_literal_with_equal_pair_weights_is_plain_momentum_sgd(oracle_mod):
    """T_k is doubly stochastic, so mixing columns that are already EQUAL changes nothing
    (PAPER.md:66, :72).  With w_s == w_p in every pair, eq. (7) as printed therefore collapses to
    each learner's own eq.-(3)+momentum update: the EQ7_LITERAL step must equal the unmixed step
    bit for bit (this fixes the fp32 order: the mixed OLD weights are formed first, exactly, and
    lr v' is subtracted once -- any other association rounds differently), and gap must be 0."""
    S, G, P = 6, 2, 5001
    partner = [1, 0, 3, 2, 5, 4]
    base = rand((S // 2, P), 230, 0.05)
    w = np.ascontiguousarray(np.repeat(base, 2, axis=0))
    v, g = rand((S, P), 231, 0.01), rand((S, G, P), 232, 1e-3)
    wa, va, wb, vb = w.copy(), v.copy(), w.copy(), v.copy()
    da = oracle_mod.step(g, wa, va, LR, MU, 0, flags=oracle_mod.EQ7_LITERAL, diag=True, partner=partner)
    db = oracle_mod.step(g, wb, vb, LR, MU, 0, flags=oracle_mod.NO_MIX, diag=True)
    assert np.array_equal(bits(wa), bits(wb)) and np.array_equal(bits(va), bits(vb))
    assert not da["gap"].any() and not db["gap"].any()
    assert np.array_equal(da["wsq"], db["wsq"]) and np.array_equal(da["gsq"], db["gsq"])
    assert np.all(da["wsq"] > 0) and np.all(da["gsq"] > 0)


@pytest.mark.parametrize("case", ["no_mix", "S1", "identity_matching"])
def test_unmixed_diagnostics(oracle_mod, case):
    """T_k = I (NO_MIX, S = 1, or a matching of fixed points): gap is exactly 0, gsq and wsq are the
    plain sums of squares in double, and w' = u."""
    S = 1 if case == "S1" else 5
    G, P = 4, 333
    g, w, v = rand((S, G, P), 240, 1e-3), rand((S, P), 241, 0.05), rand((S, P), 242, 0.01)
    acc = g[:, 0].copy()
    for k in range(1, G):
        acc = acc + g[:, k]
    gbar = acc * np.float32(0.25)
    vn = np.float32(MU) * v + gbar
    u = fl32_sub(w, fl32_mul(np.float32(LR), vn))
    if case == "identity_matching":
        d = oracle_mod.step(g, w, v, LR, MU, 0, diag=True, partner=list(range(S)))
    else:
        d = oracle_mod.step(g, w, v, LR, MU, 1, flags=oracle_mod.NO_MIX if case == "no_mix" else 0, diag=True)
    assert np.array_equal(bits(w), bits(u)) and np.array_equal(bits(v), bits(vn))
    assert np.array_equal(d["gap"], np.zeros(S))
    assert np.allclose(d["gsq"], (gbar.astype(np.float64) ** 2).sum(1), rtol=1e-12, atol=0)
    assert np.allclose(d["wsq"], (u.astype(np.float64) ** 2).sum(1), rtol=1e-12, atol=0)


# ------------------------------------------------------------------ consensus

@pytest.mark.parametrize("S", [2, 4, 8, 16])
def test_zero_gradient_preserves_mean_and_contracts(oracle_mod, S):
    """'If we halt the local updates and only conduct the model averaging ... the system
    will converge to ... (1/n) sum theta^i'."""
    P = 501
    w = rand((S, P), 20 + S, 0.05)
    w64 = w.astype(np.float64)
    v, v64 = np.zeros((S, P), np.float32), np.zeros((S, P), np.float64)
    g = np.zeros((S, 1, P), np.float32)
    mean0 = w64.mean(0)
    D_prev = oracle_mod.consensus_distance(w)
    for k in range(2 * S):
        oracle_mod.step(g, w, v, LR, MU, k)
        oracle_mod.step_f64(g, w64, v64, LR, MU, k)
        assert np.allclose(w64.mean(0), mean0, rtol=0, atol=1e-16)               # exact shadow
        assert np.max(np.abs(w.astype(np.float64).mean(0) - mean0)) <= (k + 1) * 2 ** -24 * 0.3
        D = oracle_mod.consensus_distance(w)
        assert D <= D_prev * (1 + 1e-6)
        D_prev = D
        assert not v.any()
    if S == 2:
        assert D_prev == 0.0
    assert D_prev <= 1e-3 * oracle_mod.consensus_distance(rand((S, P), 20 + S, 0.05))


def test_mixing_equal_columns_is_the_identity_down_to_subnormals(oracle_mod):
    """T_k is doubly stochastic: mixing columns that are already equal changes nothing.
    In fp32 that holds for EVERY finite value only in the stated order 0.5f * (a + a) -- a + a is exact
    (also for subnormals), and halving it is exact again -- while 0.5f*a + 0.5f*a loses the last bit of
    an odd subnormal.  No flush-to-zero (R17).  And where a + a overflows (|a| > FLT_MAX / 2) the stated
    order gives Inf: IEEE propagation, not a rescue (R17)."""
    tiny = np.float32(1e-45)                                   # the smallest subnormal
    vals = np.array([tiny, -tiny, 3 * tiny, 5 * tiny, 1.1754942e-38, 1.1754944e-38, 0.0, -0.0, 1.0, -2.5e-7,
                     1.7e38, -1.7e38], np.float32)
    P = len(vals)
    for S, k in ((2, 0), (4, 0), (4, 1), (8, 1)):
        w = np.ascontiguousarray(np.tile(vals, (S, 1)))
        v, g = np.zeros((S, P), np.float32), np.zeros((S, 2, P), np.float32)
        with np.errstate(all="ignore"):
            oracle_mod.step(g, w, v, LR, MU, k)
        assert np.array_equal(bits(w), bits(np.tile(vals, (S, 1)))), (S, k)
        assert not v.any()
    w = np.full((2, 2), 3.0e38, np.float32)
    with np.errstate(all="ignore"):
        oracle_mod.step(np.zeros((2, 1, 2), np.float32), w, np.zeros((2, 2), np.float32), LR, MU, 0)
    assert np.all(np.isposinf(w))                             # u_s + u_p overflows before the halving


def test_consensus_exact_after_one_step_S2_two_steps_S4(oracle_mod):
    P = 300
    for S, steps in ((2, 1), (4, 2)):
        w = rand((S, P), 30 + S, 0.05)
        v, g = np.zeros((S, P), np.float32), np.zeros((S, 1, P), np.float32)
        for k in range(steps):
            oracle_mod.step(g, w, v, LR, MU, k)
        for s in range(1, S):
            assert np.array_equal(bits(w[s]), bits(w[0]))     # bitwise consensus


@pytest.mark.parametrize("S,rate", [(8, 0.5), (16, 0.8535533905932737)])
def test_consensus_rate_closed_form(oracle_mod, S, rate):
    """After step 0 the state is constant on pairs; each (odd, even) double step then acts
    on the S/2 pair values as the circulant x_i <- (x_{i-1}+2x_i+x_{i+1})/4 with
    eigenvalues cos^2(pi j/(S/2)).  Seeding the slowest mode j=1 must decay by exactly
    cos^2(2 pi / S) per double step."""
    m = S // 2
    assert abs(np.cos(np.pi / m) ** 2 - rate) < 1e-15
    P = 4
    mode = np.cos(2 * np.pi * np.arange(m) / m)
    w64 = np.repeat(mode, 2)[:, None] * np.ones((1, P))      # constant on even-step pairs
    v64, g = np.zeros((S, P)), np.zeros((S, 1, P), np.float32)
    amp0 = np.abs(w64).max()
    for dbl in range(1, 6):
        oracle_mod.step_f64(g, w64, v64, LR, MU, 1)            # odd
        oracle_mod.step_f64(g, w64, v64, LR, MU, 2)            # even
        assert np.allclose(w64[:, 0], np.repeat(mode, 2) * rate ** dbl, atol=1e-14)
        assert abs(np.abs(w64).max() / amp0 - rate ** dbl) < 1e-14


def test_variance_identity_links_gap_to_consensus(oracle_mod):
    """D(u) - D(w') = 1/2 sum_pairs ||u_s - u_p||^2  (gap is reported per member, so the
    sum over s counts each pair twice => 1/4 sum_s gap[s])."""
    S, G, P = 8, 2, 257
    g, w, v = rand((S, G, P), 40, 1e-3), rand((S, P), 41, 0.05), rand((S, P), 42, 0.01)
    wn, vn = w.copy(), v.copy()
    oracle_mod.step(g, wn, vn, LR, MU, 1, flags=oracle_mod.NO_MIX)    # wn = u
    D_u = oracle_mod.consensus_distance(wn)
    d = oracle_mod.step(g, w, v, LR, MU, 1, diag=True)
    D_w = oracle_mod.consensus_distance(w)
    assert abs((D_u - D_w) - 0.25 * d["gap"].sum()) <= 1e-6 * D_u


def test_consensus_distance_against_two_independent_formulas(oracle_mod):
    """D = sum_s |w_s - wbar|^2 (wbar = (1/n) sum theta^i is where mixing converges).
    Checked against numpy's mean-based form and against the mean-free pairwise identity
    D = (1/(2S)) sum_{s,t} |w_s - w_t|^2; zero exactly when all learners agree."""
    for S, P in ((2, 5), (3, 64), (8, 257), (16, 33)):
        w = rand((S, P), 70 + S, 0.05)
        w64 = w.astype(np.float64)
        D = oracle_mod.consensus_distance(w)
        assert D == pytest.approx(((w64 - w64.mean(0)) ** 2).sum(), rel=1e-12)
        pair = sum(((w64[s] - w64[t]) ** 2).sum() for s in range(S) for t in range(S)) / (2.0 * S)
        assert D == pytest.approx(pair, rel=1e-11)
    same = np.repeat(rand((1, 100), 3, 0.05), 6, axis=0)
    assert oracle_mod.consensus_distance(np.ascontiguousarray(same)) == 0.0


# ------------------------------------------------------------------ special cases

def test_ssgd_special_case(oracle_mod):
    """'ADPSGD has synchronous SGD as its special case': identical weights and
    identical gradients on every super-learner stay bit-identical to a single learner."""
    S, G, P, K = 8, 2, 777, 6
    w1 = rand((1, P), 50, 0.05)
    v1 = np.zeros((1, P), np.float32)
    wS, vS = np.repeat(w1, S, 0).copy(), np.repeat(v1, S, 0).copy()
    for k in range(K):
        g1 = rand((1, G, P), 60 + k, 1e-3)
        oracle_mod.step(g1, w1, v1, LR, MU, k)
        oracle_mod.step(np.ascontiguousarray(np.repeat(g1, S, 0)), wS, vS, LR, MU, k)
        for s in range(S):
            assert np.array_equal(bits(wS[s]), bits(w1[0])) and np.array_equal(bits(vS[s]), bits(v1[0]))


@pytest.mark.parametrize("G", [2, 3, 4, 8])
def test_hierarchy_equivalence(oracle_mod, G):
    """'lambda-learner H-ADPSGD is equivalent to a (lambda/N)-learner ADPSGD':
    (S,G) equals (S,1) fed the pre-averaged gradient.  Bit-exact when 1/G is a power of
    two (multiplying by 1.0f afterwards is the identity); G=3 within 1 ulp of gbar."""
    S, P = 4, 1001
    g = rand((S, G, P), 70, 1e-3)
    acc = g[:, 0].copy()
    for k in range(1, G):
        acc = acc + g[:, k]
    gbar = (acc * (np.float32(1.0) / np.float32(G)))[:, None, :].copy()
    wa, va = rand((S, P), 71, 0.05), rand((S, P), 72, 0.01)
    wb, vb = wa.copy(), va.copy()
    oracle_mod.step(g, wa, va, LR, MU, 1)
    oracle_mod.step(gbar, wb, vb, LR, MU, 1)
    assert np.array_equal(bits(wa), bits(wb)) and np.array_equal(bits(va), bits(vb))


def test_pair_symmetry_and_relabelling(oracle_mod):
    """Reversing the ring labels maps matchings to matchings; results must be the reversed
    arrays bit for bit (fp add commutes; no dependence on which member is 's')."""
    S, G, P = 8, 2, 513
    g, w, v = rand((S, G, P), 80, 1e-3), rand((S, P), 81, 0.05), rand((S, P), 82, 0.01)
    # s -> S-1-s maps even pairs (2i,2i+1) onto even pairs, odd pairs onto odd pairs
    gr, wr, vr = g[::-1].copy(), w[::-1].copy(), v[::-1].copy()
    for k in (0, 1):
        oracle_mod.step(g, w, v, LR, MU, k)
        oracle_mod.step(gr, wr, vr, LR, MU, k)
        assert np.array_equal(bits(w[::-1]), bits(wr)) and np.array_equal(bits(v[::-1]), bits(vr))
    po = oracle_mod.partner(S, 1)
    for s in range(S):
        assert np.array_equal(bits(w[s]), bits(w[po[s]]))                 # both members get the same bits


def test_elementwise_independence_windows(oracle_mod):
    """The method is element-wise: running on a window equals slicing the full run.  This is
    what lets full-size GPU parity be checked window by window."""
    S, G, P = 4, 2, 3000
    g, w, v = rand((S, G, P), 90, 1e-3), rand((S, P), 91, 0.05), rand((S, P), 92, 0.01)
    lo, hi = 1234, 2345
    gw = np.ascontiguousarray(g[:, :, lo:hi])
    ww, vw = np.ascontiguousarray(w[:, lo:hi]), np.ascontiguousarray(v[:, lo:hi])
    for k in range(3):
        oracle_mod.step(g, w, v, LR, MU, k)
        oracle_mod.step(gw, ww, vw, LR, MU, k)
    assert np.array_equal(bits(w[:, lo:hi]), bits(ww)) and np.array_equal(bits(v[:, lo:hi]), bits(vw))


def test_bf16_gradients_equal_widened_fp32(oracle_mod):
    S, G, P = 2, 8, 999
    gb = gen.f32_to_bf16_bits(rand((S, G, P), 95, 1e-3))
    gf = gen.bf16_bits_to_f32(gb)
    wa, va = rand((S, P), 96, 0.05), rand((S, P), 97, 0.01)
    wb, vb = wa.copy(), va.copy()
    oracle_mod.step(gb, wa, va, LR, MU, 0)
    oracle_mod.step(gf, wb, vb, LR, MU, 0)
    assert np.array_equal(bits(wa), bits(wb)) and np.array_equal(bits(va), bits(vb))


def test_f32_tracks_f64_shadow_within_north_star_tolerance(oracle_mod):
    """Tolerance derivation: after 20 steps the fp32 trajectory stays
    within 1e-6 + 1e-5|w| of the double shadow on config-like data."""
    S, G, P = 4, 4, 4096
    w = gen.weights_window(7, S, 0, P)
    v = np.zeros((S, P), np.float32)
    w64, v64 = w.astype(np.float64), v.astype(np.float64)
    for k in range(20):
        g = gen.grads_window(7, k, S, G, 0, P)
        oracle_mod.step(g, w, v, LR, MU, k)
        oracle_mod.step_f64(g, w64, v64, float(np.float32(LR)), float(np.float32(MU)), k)
    assert np.all(np.abs(w - w64) <= 1e-6 + 1e-5 * np.abs(w64))
    assert np.all(np.abs(v - v64) <= 1e-6 + 1e-5 * np.abs(v64))
    assert np.max(np.abs(w - w64)) < 2e-7          # measured head-room, used to justify the bound


def test_invalid_arguments(oracle_mod):
    g, w, v = np.zeros((3, 1, 4), np.float32), np.zeros((3, 4), np.float32), np.zeros((3, 4), np.float32)
    with pytest.raises(ValueError):
        oracle_mod.step(g, w, v, LR, MU, 0)               # odd S > 1
    oracle_mod.step(g, w, v, LR, MU, 0, flags=oracle_mod.NO_MIX)   # fine without mixing


# ------------------------------------------------------------------ bf16 working copy (row f2)

def _all_finite_bf16():
    bits = np.arange(65536, dtype=np.uint32)
    f32 = (bits << np.uint32(16)).view(np.float32)
    keep = np.isfinite(f32)
    vals = np.where(keep, f32, np.float32(0)).astype(np.float64)
    return bits[keep].astype(np.uint16), vals[keep]


def test_round_bf16_brute_force_nearest_ties_to_even(oracle_mod):
    """Brute force over ALL finite bf16 values: the result must be the nearest one, and on an exact
    tie the one with an even last mantissa bit (IEEE round-to-nearest-even)."""
    cand_bits, cand = _all_finite_bf16()
    rng = np.random.default_rng(5)
    x = np.concatenate([rand(300, 1, 0.05).ravel(), rand(100, 2, 1e-3).ravel(),
                        rng.integers(0, 2 ** 32, 400, dtype=np.uint64).astype(np.uint32).view(np.float32)])
    x = x[np.isfinite(x) & (np.abs(x) < 3.0e38)].astype(np.float32)
    # exact halfway points between neighbouring bf16 values (fp32 can hold them)
    ties = ((np.array([0x3F80, 0x3F81, 0x4000, 0x00FF, 0xBF80, 0x3DCC], dtype=np.uint32) << 16) | 0x8000).view(np.float32)
    x = np.concatenate([x, ties])
    got = oracle_mod.round_bf16(x)
    for xi, gi in zip(x.astype(np.float64), got):
        d = np.abs(cand - xi)
        best = np.flatnonzero(d == d.min())
        if (cand[best] == 0).all():                             # +0 / -0 are the same value
            assert int(gi) in (0x0000, 0x8000)
        elif len(best) == 1:
            assert int(gi) == int(cand_bits[best[0]])
        else:                                                   # tie: even last mantissa bit wins
            even = [int(b) for b in cand_bits[best] if b % 2 == 0]
            assert len(even) == 1 and int(gi) == even[0], (xi, hex(int(gi)), [hex(int(b)) for b in cand_bits[best]])
        assert np.abs(np.float64(gen.bf16_bits_to_f32(np.array([gi], np.uint16))[0]) - xi) == d.min()


def test_round_bf16_matches_library_and_fixed_points(oracle_mod):
    import torch
    x = rand(200_000, 9, 0.05).ravel()
    lib = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)   # library RNE cast
    assert np.array_equal(oracle_mod.round_bf16(x), lib)
    # bf16-representable values are fixed points; widening the result is exact
    r = gen.bf16_bits_to_f32(oracle_mod.round_bf16(x))
    assert np.array_equal(oracle_mod.round_bf16(r), oracle_mod.round_bf16(x))
    assert np.all(np.abs(r.astype(np.float64) - x) <= np.abs(x.astype(np.float64)) * 2.0 ** -8)   # half an ulp of 8 bits
    sp = np.array([np.inf, -np.inf, 3.4028235e38, -3.4028235e38, 0.0, -0.0], np.float32)
    assert [int(v) for v in oracle_mod.round_bf16(sp)] == [0x7F80, 0xFF80, 0x7F80, 0xFF80, 0x0000, 0x8000]
    nan = oracle_mod.round_bf16(np.array([np.nan], np.float32))[0]
    assert (nan & 0x7F80) == 0x7F80 and (nan & 0x007F) != 0


# ------------------------------------------------------------------ bf16 edge values (R6, R17)

BF16_EDGE = [0x0000, 0x8000,             # +0, -0
             0x0001, 0x007F, 0x8001,     # subnormal bf16: smallest, largest, negative smallest
             0x0080, 0x8080,             # smallest normals
             0x3F80, 0xBF80,             # +-1
             0x7F7F, 0xFF7F,             # largest finite
             0x7F80, 0xFF80,             # +-Inf
             0x7FC0, 0xFFC1, 0x7F81]     # NaNs: quiet, negative with payload, quiet bit clear


def test_bf16_gradient_widening_is_exact_on_edge_values(oracle_mod):
    """R6 ("bf16 -> fp32 widening is exact") with R17 (no flush-to-zero) on the values a
    Gaussian draw never produces.  S = 1, G = 1, mu = 0, lr = 1, w = v = 0: the mean is the gradient
    itself (eq. (6) with one learner), so v' = 0*0 + g must be the widened gradient
    (h << 16 as an fp32 pattern, built here) bit for bit and w' = 0 - 1*v' its negation -- down to the
    smallest subnormal.  -0 is the one value the arithmetic itself changes: (+0) + (-0) = +0."""
    h = np.array(BF16_EDGE, dtype=np.uint16)
    want = (h.astype(np.uint32) << np.uint32(16)).view(np.float32)        # the definition of bf16
    P = len(h)
    for G in (1, 2):                        # G = 2: (g + 0) * 0.5 halves exactly unless it underflows
        g = np.zeros((1, G, P), np.uint16)
        g[0, 0] = h
        w, v = np.zeros((1, P), np.float32), np.zeros((1, P), np.float32)
        oracle_mod.step(g, w, v, 1.0, 0.0, 0)
        with np.errstate(invalid="ignore"):
            exp_v = want if G == 1 else (want.astype(np.float64) * 0.5).astype(np.float32)   # exact or RNE once: the definition
        nan = np.isnan(want)
        assert np.array_equal(np.isnan(v[0]), nan) and np.array_equal(np.isnan(w[0]), nan)
        ok = ~nan & (h != 0x8000)
        assert np.array_equal(bits(v[0][ok]), bits(exp_v[ok])), [hex(int(x)) for x in bits(v[0])]
        assert np.array_equal(bits(w[0][ok]), bits(np.float32(0) - exp_v[ok]))        # 0 - 1*v': exact; (+0) - (+0) = +0
        assert bits(v[0][h == 0x8000])[0] == 0 and bits(w[0][h == 0x8000])[0] == 0        # -0 -> +0 + -0 = +0
        if G == 1:                          # the subnormals in particular: not flushed
            assert [int(x) for x in bits(v[0][2:5])] == [0x00010000, 0x007F0000, 0x80010000]
            assert v[0][2] > 0 and v[0][4] < 0
    # the double-precision shadow widens the same way
    g = np.zeros((1, 1, P), np.uint16)
    g[0, 0] = h
    w64, v64 = np.zeros((1, P)), np.zeros((1, P))
    oracle_mod.step_f64(g, w64, v64, 1.0, 0.0, 0)
    fin = np.isfinite(want)
    assert np.array_equal(v64[0][fin], want[fin].astype(np.float64))


def test_round_bf16_of_a_nan_is_a_nan_never_inf(oracle_mod):
    """R17 reading for the bf16 working copy (row f2): a NaN weight rounds to A NaN -- which one (sign,
    payload) is not specified, because the CUDA path's cvt.rn.bf16x2.f32 returns the canonical 0x7FFF
    while this oracle keeps sign and upper payload -- so the tests compare NaN-ness.  What IS fixed:
    never +-Inf (a NaN whose upper seven mantissa bits are zero must not truncate to 0x7F80), and
    +-Inf / finite values are never turned into NaN."""
    nan_bits = np.array([0x7F800001, 0xFF800001, 0x7F80FFFF, 0x7FC00000, 0xFFC00000, 0x7F8ABCDE, 0xFFFFFFFF,
                         0x7FBFFFFF, 0x7F810000], dtype=np.uint32)
    got = oracle_mod.round_bf16(nan_bits.view(np.float32))
    for b, r in zip(nan_bits, got):
        assert (int(r) & 0x7F80) == 0x7F80 and (int(r) & 0x007F) != 0, (hex(int(b)), hex(int(r)))
    widened = (got.astype(np.uint32) << np.uint32(16)).view(np.float32)
    assert np.isnan(widened).all()
    # and nothing that is not a NaN becomes one: Inf, the overflow to Inf, the largest values that stay finite
    sp = np.array([0x7F800000, 0xFF800000, 0x7F7FFFFF, 0xFF7FFFFF, 0x7F7F8000, 0x7F7F7FFF, 0x7F7F0000], dtype=np.uint32)
    assert [int(x) for x in oracle_mod.round_bf16(sp.view(np.float32))] == [0x7F80, 0xFF80, 0x7F80, 0xFF80, 0x7F80, 0x7F7F, 0x7F7F]
    # subnormal fp32 weights round among subnormal bf16 values (no flush): 0x00008000 is a tie -> even (0),
    # 0x00018000 a tie -> even (2), 0x00008001 just above the tie -> 1
    sub = np.array([0x00008000, 0x00018000, 0x00008001, 0x80008001, 0x007FFFFF], dtype=np.uint32)
    assert [int(x) for x in oracle_mod.round_bf16(sub.view(np.float32))] == [0x0000, 0x0002, 0x0001, 0x8001, 0x0080]
