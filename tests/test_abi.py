"""Boundary checks that need no GPU: the C-ABI library loads, exports every symbol that
include/hadpsgd.h declares, and its host-only entry points (allocator a0, scheduler a1)
behave.  No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def H():
    import __graft_entry__  # noqa: F401  (build() compiles the library when it is stale)
    from paper_1907_05701_b200 import build as b
    b.build()
    import paper_1907_05701_b200 as m
    return m


def declared_symbols():
    names = set()
    for fn in os.listdir(os.path.join(ROOT, "include")):
        if fn.endswith(".h"):
            src = open(os.path.join(ROOT, "include", fn)).read()
            src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
            names |= set(re.findall(r"\b(hadpsgd_[a-z_0-9]+)\s*\(", src))
    return names


def test_library_exports_every_declared_symbol(H):
    L = H.lib()
    names = declared_symbols()
    assert {"hadpsgd_create", "hadpsgd_step", "hadpsgd_weights", "hadpsgd_step_host", "hadpsgd_pairing"} <= names
    for n in sorted(names):
        assert hasattr(L, n), f"libhadpsgd.so does not export {n}"


def test_pairing_matches_oracle_and_paper(H, oracle_mod):
    """Scheduler (product) vs the oracle's independent implementation, and vs the structure
    PAPER.md:66 demands (perfect matching of ring neighbours)."""
    for S in (1, 2, 4, 6, 8, 16, 64, 512):
        for k in (0, 1, 2, 3, 2 ** 40 + 1):
            p = np.array(H.hadpsgd_pairing(S, k))
            assert np.array_equal(p, oracle_mod.partner(S, k))
            if S > 1:
                assert np.array_equal(p[p], np.arange(S))
                assert np.all(((p - np.arange(S)) % S == 1) | ((p - np.arange(S)) % S == S - 1))
    for S in (0, 3, 5, -1):
        with pytest.raises(H.HadpsgdError):
            H.hadpsgd_pairing(S, 0)


def test_allocator_layout(H):
    from fixtures import shapes
    # flat config 2: no padding, regions 256 B aligned, total = 55.7 GB + scratch
    P = shapes.total(shapes.SWB2000_SEGMENTS)
    lay = H.hadpsgd_layout(16, 4, [P])
    assert lay["P_padded"] == P and lay["seg_offset"] == [0]
    assert lay["w_off"] == 0 and lay["v_off"] == 16 * P * 4 and lay["g_off"] == 32 * P * 4
    need = H.hadpsgd_required_bytes(16, 4, [P])
    assert 16 * P * (4 * 4 + 8) <= need <= 16 * P * (4 * 4 + 8) + (16 << 20)      # + diagnostics scratch
    # ragged bf16 config 3: 40 segments, every natural length is a multiple of 64 -> no padding
    seg = [n for _, n in shapes.SWB2000_SEGMENTS]
    lay = H.hadpsgd_layout(8, 8, seg, H.BF16)
    assert lay["P_padded"] == P and lay["seg_offset"] == list(np.concatenate([[0], np.cumsum(seg)[:-1]]))
    assert lay["g_off"] == 16 * P * 4                      # 8 w + 8 v fp32 buffers, then bf16 grads
    # adversarial odd table: starts aligned to 64 elements, padded total
    odd = [1, 3, 7, 1025, 64, 63, 65]
    lay = H.hadpsgd_layout(2, 2, odd)
    assert all(o % 64 == 0 for o in lay["seg_offset"])
    assert lay["seg_offset"] == [0, 64, 128, 192, 192 + 1088, 192 + 1088 + 64, 192 + 1088 + 128]
    assert lay["P_padded"] == 192 + 1088 + 128 + 128
    for off in ("w_off", "v_off", "g_off"):
        assert lay[off] % 256 == 0
    # bf16 working copy (row f2): a fourth region of S x P_padded x 2 B after the gradients
    plain, emit = H.hadpsgd_layout(4, 2, odd), H.hadpsgd_layout(4, 2, odd, H.F32, H.BF16)
    assert {k: emit[k] for k in ("seg_offset", "P_padded", "w_off", "v_off", "g_off")} == \
           {k: plain[k] for k in ("seg_offset", "P_padded", "w_off", "v_off", "g_off")}
    assert emit["wb_off"] % 256 == 0 and emit["wb_off"] >= emit["g_off"] + 4 * 2 * emit["P_padded"] * 4
    extra = H.hadpsgd_required_bytes(4, 2, odd, H.F32, H.BF16) - H.hadpsgd_required_bytes(4, 2, odd)
    assert 4 * emit["P_padded"] * 2 <= extra < 4 * emit["P_padded"] * 2 + 256
    with pytest.raises(H.HadpsgdError):
        H.hadpsgd_required_bytes(4, 2, odd, H.F32, 7)
    for bad in ((0, 1, [4]), (2, 0, [4]), (2, 2, []), (2, 2, [4, 0]), (513 * 2, 1, [4])):
        with pytest.raises(H.HadpsgdError):
            H.hadpsgd_required_bytes(*bad)


def test_error_strings(H):
    L = H.lib()
    assert L.hadpsgd_error_string(0) == b"ok"
    assert b"sm_100a" in L.hadpsgd_error_string(-4)


def test_no_cpu_fallback_without_gpu(H):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        H.Hadpsgd(2, 2, [1000])
