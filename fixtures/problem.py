"""Seeded problems: the same synthetic inputs for the CUDA path (filled in HBM) and for the
oracle (numpy windows).  No method arithmetic here -- only which generator value goes where.

Values are a function of the NATURAL (model-order, unpadded) parameter index, so a ragged
segment table and the flat concatenation hold the same numbers.
"""
import numpy as np

from . import generator as gen


def natural_offsets(seg_len):
    return np.concatenate([[0], np.cumsum(np.asarray(seg_len, dtype=np.int64))])


# ---- device side: `handle` is any object with S, G, seg_len, hadpsgd_segment(k),
# hadpsgd_weights(s), hadpsgd_momentum(s), hadpsgd_grads(s, g) returning torch views --------

def fill_weights(handle, seed, sd=0.05):
    from . import device
    nat = natural_offsets(handle.seg_len)
    for s in range(handle.S):
        w = handle.hadpsgd_weights(s)
        key = gen.stream_key(seed, gen.STREAM_WEIGHT, 0, s, 0)
        for k, n in enumerate(handle.seg_len):
            off, _ = handle.hadpsgd_segment(k)
            device.fill(w[off:off + n], key, "normal", sd, elem_offset=int(nat[k]))
        handle.hadpsgd_momentum(s).zero_()


def fill_grads(handle, seed, step, dist="normal", scale=1e-3):
    from . import device
    nat = natural_offsets(handle.seg_len)
    for s in range(handle.S):
        for g in range(handle.G):
            buf = handle.hadpsgd_grads(s, g)
            key = gen.stream_key(seed, gen.STREAM_GRAD, step, s, g)
            for k, n in enumerate(handle.seg_len):
                off, _ = handle.hadpsgd_segment(k)
                device.fill(buf[off:off + n], key, dist, scale, elem_offset=int(nat[k]))


# ---- host side: windows [lo, hi) of the natural index space -----------------------------

def host_weights(seed, S, lo, hi, sd=0.05):
    return gen.weights_window(seed, S, lo, hi - lo, sd)


def host_grads(seed, step, S, G, lo, hi, dist="normal", scale=1e-3, bf16=False):
    return gen.grads_window(seed, step, S, G, lo, hi - lo, dist, scale, bf16)


def padded_index(seg_len, seg_offset, lo, hi):
    """Padded-buffer indices of natural elements [lo, hi)."""
    nat = natural_offsets(seg_len)
    out = []
    for k, n in enumerate(seg_len):
        a, b = max(lo, int(nat[k])), min(hi, int(nat[k]) + n)
        if a < b:
            out.append(np.arange(a - int(nat[k]) + seg_offset[k], b - int(nat[k]) + seg_offset[k], dtype=np.int64))
    return np.concatenate(out) if out else np.empty(0, np.int64)
