"""Seeded synthetic inputs (host side) -- serves BOTH the oracle and the CUDA path.

This module holds none of the method's arithmetic: it only manufactures numbers.  Every
value is a pure function of (seed, stream, step, s, g, i) through a 64-bit counter hash,
then shaped with INTEGER operations and ONE fp32 multiply, so that this numpy version and
the device version in ``fixtures/gen_device.cu`` agree bit for bit without libm
(tests/test_parity_gpu.py::test_device_generator_matches_host compares them).

Recipe:
  key   = mix64(seed ^ mix64(GOLDEN * (1 + tag)))   tag = ((stream*2^24 + step)*2^12 + s)*2^12 + g
  x(i)  = mix64(key + GOLDEN * (i + 1))             mix64 = the splitmix64 finaliser
  uniform(a): top 24 bits k in [0,2^24) -> float(k - 2^23) * fp32(a / 2^23)        in [-a, a)
  normal(sd): sum of the four 16-bit lanes (Irwin-Hall n=4), minus 131070, as float,
              times fp32(sd / sqrt((65536^2-1)/3))  -- a bell-shaped stand-in for N(0, sd)
  bf16:       round-to-nearest-even of that fp32, done on the bit pattern
"""
import numpy as np

GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

STREAM_WEIGHT = 1
STREAM_GRAD = 2
STREAM_MOMENTUM = 3

IH4_SIGMA = float(np.sqrt((65536.0 ** 2 - 1.0) / 3.0))  # std of the sum of four uniform 16-bit lanes


def _mix64(x):
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = (x ^ (x >> np.uint64(30))) * _M1
        x = (x ^ (x >> np.uint64(27))) * _M2
        x = x ^ (x >> np.uint64(31))
    return x


def stream_key(seed, stream, step, s, g):
    """64-bit key for one buffer; python ints in, python int out (passed by value to the device)."""
    tag = ((int(stream) * (1 << 24) + int(step)) * (1 << 12) + int(s)) * (1 << 12) + int(g)
    with np.errstate(over="ignore"):
        inner = _mix64(np.uint64((int(GOLDEN) * (1 + tag)) & 0xFFFFFFFFFFFFFFFF))
        key = _mix64(np.uint64(int(seed) & 0xFFFFFFFFFFFFFFFF) ^ inner)
    return int(key)


def raw_bits(key, elem_offset, n):
    """x(i) for i in [elem_offset, elem_offset+n) as uint64."""
    i = np.arange(elem_offset + 1, elem_offset + n + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        return _mix64(np.uint64(key) + GOLDEN * i)


def uniform_scale(a):
    return np.float32(a / 8388608.0)


def normal_scale(sd):
    return np.float32(sd / IH4_SIGMA)


def uniform_f32(key, elem_offset, n, a):
    x = raw_bits(key, elem_offset, n)
    k = (x >> np.uint64(40)).astype(np.int64) - (1 << 23)
    return k.astype(np.float32) * uniform_scale(a)


def normal_f32(key, elem_offset, n, sd):
    x = raw_bits(key, elem_offset, n)
    m = np.uint64(0xFFFF)
    t = (x & m) + ((x >> np.uint64(16)) & m) + ((x >> np.uint64(32)) & m) + (x >> np.uint64(48))
    k = t.astype(np.int64) - 131070
    return k.astype(np.float32) * normal_scale(sd)


def f32_to_bf16_bits(f):
    """Round-to-nearest-even fp32 -> bf16 on the bit pattern (finite inputs)."""
    b = np.ascontiguousarray(f, dtype=np.float32).view(np.uint32)
    r = b + np.uint32(0x7FFF) + ((b >> np.uint32(16)) & np.uint32(1))
    return (r >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(h):
    return (np.ascontiguousarray(h, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal_bf16(key, elem_offset, n, sd):
    return f32_to_bf16_bits(normal_f32(key, elem_offset, n, sd))


# ---------------------------------------------------------------------------------------
# Whole-problem helpers: windows [elem_offset, elem_offset+n) of every buffer.
# ---------------------------------------------------------------------------------------

def weights_window(seed, S, elem_offset, n, sd=0.05):
    """w[s][elem_offset : elem_offset+n], fp32, ~N(0, sd)."""
    return np.stack([normal_f32(stream_key(seed, STREAM_WEIGHT, 0, s, 0), elem_offset, n, sd)
                     for s in range(S)])


def grads_window(seed, step, S, G, elem_offset, n, dist="normal", scale=1e-3, bf16=False):
    """grads[s][g][elem_offset : elem_offset+n] for one step; float32, or uint16 bf16 bits."""
    out = np.empty((S, G, n), dtype=np.uint16 if bf16 else np.float32)
    for s in range(S):
        for g in range(G):
            key = stream_key(seed, STREAM_GRAD, step, s, g)
            f = normal_f32(key, elem_offset, n, scale) if dist == "normal" \
                else uniform_f32(key, elem_offset, n, scale)
            out[s, g] = f32_to_bf16_bits(f) if bf16 else f
    return out
