"""CPU oracle for the H-ADPSGD super-learner step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes/numpy wrapper over ``libhadpsgd_oracle.so`` (plain single-threaded C++,
``oracle/hadpsgd_oracle.cpp``, written from PAPER.md).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1907_05701_b200`` and the product imports nothing from here.
"""
import ctypes
import os

import numpy as np

GRAD_F32 = 0
GRAD_BF16 = 1
NO_MIX = 1 << 0
EQ7_LITERAL = 1 << 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        from . import build as _build  # lazy: keeps `python -m oracle.build` clean
        path = _build.build()
        L = ctypes.CDLL(path)
        i32, i64, u64, u32 = ctypes.c_int, ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint32
        vp, f32, f64 = ctypes.c_void_p, ctypes.c_float, ctypes.c_double
        L.hadpsgd_oracle_partner.argtypes = [i32, u64, vp]
        L.hadpsgd_oracle_mixing_matrix.argtypes = [i32, u64, vp]
        L.hadpsgd_oracle_step.argtypes = [i32, i32, i64, vp, i32, vp, vp, f32, f32, u64, u32, vp]
        L.hadpsgd_oracle_step_f64.argtypes = [i32, i32, i64, vp, i32, vp, vp, f64, f64, u64, u32]
        L.hadpsgd_oracle_step_matching.argtypes = [i32, i32, i64, vp, i32, vp, vp, f32, f32, vp, u32, vp]
        L.hadpsgd_oracle_step_matching_f64.argtypes = [i32, i32, i64, vp, i32, vp, vp, f64, f64, vp, u32]
        L.hadpsgd_oracle_mixing_matrix_matching.argtypes = [i32, vp, vp]
        L.hadpsgd_oracle_consensus_distance.argtypes = [i32, i64, vp, vp]
        L.hadpsgd_oracle_round_bf16.argtypes = [i64, vp, vp]
        L.hadpsgd_oracle_round_bf16.restype = i32
        for fn in (L.hadpsgd_oracle_partner, L.hadpsgd_oracle_mixing_matrix, L.hadpsgd_oracle_step,
                   L.hadpsgd_oracle_step_f64, L.hadpsgd_oracle_consensus_distance, L.hadpsgd_oracle_step_matching,
                   L.hadpsgd_oracle_step_matching_f64, L.hadpsgd_oracle_mixing_matrix_matching):
            fn.restype = i32
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def partner(S, step_k):
    out = np.empty(S, dtype=np.int32)
    rc = lib().hadpsgd_oracle_partner(S, step_k, _ptr(out))
    if rc != 0:
        raise ValueError(f"hadpsgd_oracle_partner(S={S}) rc={rc}")
    return out


def mixing_matrix(S, step_k):
    T = np.empty((S, S), dtype=np.float64)
    rc = lib().hadpsgd_oracle_mixing_matrix(S, step_k, _ptr(T))
    if rc != 0:
        raise ValueError(f"hadpsgd_oracle_mixing_matrix(S={S}) rc={rc}")
    return T


def _check(grads, w, v, wdtype):
    assert grads.ndim == 3 and grads.flags.c_contiguous
    S, G, P = grads.shape
    if grads.dtype == np.float32:
        gd = GRAD_F32
    elif grads.dtype == np.uint16:  # bf16 bit patterns
        gd = GRAD_BF16
    else:
        raise TypeError("grads must be float32 or uint16 (bf16 bits)")
    for a in (w, v):
        assert a.dtype == wdtype and a.shape == (S, P) and a.flags.c_contiguous and a.flags.writeable
    return S, G, P, gd


def _matching(partner, S):
    p = np.ascontiguousarray(partner, dtype=np.int32)
    if p.shape != (S,):
        raise ValueError("partner must have S entries")
    return p


def mixing_matrix_matching(partner):
    p = _matching(partner, len(partner))
    T = np.empty((len(p), len(p)), dtype=np.float64)
    rc = lib().hadpsgd_oracle_mixing_matrix_matching(len(p), _ptr(p), _ptr(T))
    if rc != 0:
        raise ValueError("hadpsgd_oracle_mixing_matrix_matching: partner is not a matching")
    return T


def step(grads, w, v, lr, mu, step_k, flags=0, diag=False, partner=None):
    """In-place fp32 step on w, v (numpy float32 [S,P]); grads [S,G,P] float32 or uint16(bf16).
    partner=None: the ring matching of step_k's parity; else a caller-supplied matching [S]
    (an involution; partner[s] == s leaves s unmixed).

    Returns None, or a dict of double arrays gsq[S], wsq[S], gap[S] when diag=True."""
    S, G, P, gd = _check(grads, w, v, np.float32)
    d = np.zeros(3 * S, dtype=np.float64) if diag else None
    if partner is None:
        rc = lib().hadpsgd_oracle_step(S, G, P, _ptr(grads), gd, _ptr(w), _ptr(v),
                                       float(lr), float(mu), int(step_k), int(flags),
                                       _ptr(d) if diag else None)
    else:
        pt = _matching(partner, S)
        rc = lib().hadpsgd_oracle_step_matching(S, G, P, _ptr(grads), gd, _ptr(w), _ptr(v),
                                                float(lr), float(mu), _ptr(pt), int(flags),
                                                _ptr(d) if diag else None)
    if rc != 0:
        raise ValueError(f"hadpsgd_oracle_step rc={rc}")
    if diag:
        return {"gsq": d[:S].copy(), "wsq": d[S:2 * S].copy(), "gap": d[2 * S:].copy()}
    return None


def step_f64(grads, w, v, lr, mu, step_k, flags=0, partner=None):
    """In-place double-precision shadow step on w, v (numpy float64 [S,P])."""
    S, G, P, gd = _check(grads, w, v, np.float64)
    if partner is None:
        rc = lib().hadpsgd_oracle_step_f64(S, G, P, _ptr(grads), gd, _ptr(w), _ptr(v),
                                           float(lr), float(mu), int(step_k), int(flags))
    else:
        pt = _matching(partner, S)
        rc = lib().hadpsgd_oracle_step_matching_f64(S, G, P, _ptr(grads), gd, _ptr(w), _ptr(v),
                                                    float(lr), float(mu), _ptr(pt), int(flags))
    if rc != 0:
        raise ValueError(f"hadpsgd_oracle_step_f64 rc={rc}")


def round_bf16(w):
    """bf16 bit patterns (uint16, same shape) of the fp32 array w, round-to-nearest-even."""
    w = np.ascontiguousarray(w, dtype=np.float32)
    out = np.empty(w.shape, dtype=np.uint16)
    rc = lib().hadpsgd_oracle_round_bf16(w.size, _ptr(w), _ptr(out))
    if rc != 0:
        raise ValueError("hadpsgd_oracle_round_bf16 failed")
    return out


def consensus_distance(w):
    assert w.dtype == np.float32 and w.ndim == 2 and w.flags.c_contiguous
    out = np.zeros(1, dtype=np.float64)
    rc = lib().hadpsgd_oracle_consensus_distance(w.shape[0], w.shape[1], _ptr(w), _ptr(out))
    if rc != 0:
        raise ValueError("hadpsgd_oracle_consensus_distance failed")
    return float(out[0])
