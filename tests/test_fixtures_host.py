"""Host-side input generator and workload shapes (no method arithmetic here)."""
import numpy as np
import torch

from fixtures import generator as gen
from fixtures import shapes


def test_shapes_match_baseline_configs():
    assert shapes.total(shapes.SWB300_SEGMENTS) == 94_797_312 and len(shapes.SWB300_SEGMENTS) == 28
    assert shapes.total(shapes.SWB2000_SEGMENTS) == 145_145_344 and len(shapes.SWB2000_SEGMENTS) == 40
    # PAPER.md:106 "over 43 million parameters ... about 165MB"
    n = shapes.total(shapes.PAPER_LITERAL_SEGMENTS)
    assert n == 43_130_368 and abs(n * 4 / 2 ** 20 - 164.5) < 0.1
    assert len(shapes.sweep_points()) == 119
    assert (1 << 28, 16, 8) not in shapes.sweep_points()


def test_generator_is_a_pure_function_of_its_counter():
    k = gen.stream_key(123, gen.STREAM_GRAD, 5, 3, 1)
    a = gen.normal_f32(k, 0, 10_000, 1e-3)
    b = gen.normal_f32(k, 2_500, 5_000, 1e-3)
    assert np.array_equal(a[2_500:7_500], b)               # windows agree with the full buffer
    assert not np.array_equal(a, gen.normal_f32(gen.stream_key(123, gen.STREAM_GRAD, 5, 3, 2), 0, 10_000, 1e-3))
    assert not np.array_equal(a, gen.normal_f32(gen.stream_key(124, gen.STREAM_GRAD, 5, 3, 1), 0, 10_000, 1e-3))


def test_generator_moments():
    k = gen.stream_key(1, gen.STREAM_WEIGHT, 0, 0, 0)
    x = gen.normal_f32(k, 0, 1_000_000, 0.05).astype(np.float64)
    assert abs(x.mean()) < 3 * 0.05 / 1000 and abs(x.std() / 0.05 - 1) < 5e-3
    assert abs(((x / 0.05) ** 4).mean() - 2.7) < 0.05      # Irwin-Hall n=4 kurtosis 3 - 6/(5*4) = 2.7
    u = gen.uniform_f32(k, 0, 1_000_000, 1e-3).astype(np.float64)
    assert u.min() >= -1e-3 and u.max() < 1e-3 and abs(u.std() / (1e-3 / 3 ** 0.5) - 1) < 5e-3


def test_bf16_rounding_is_rne():
    x = gen.normal_f32(gen.stream_key(9, gen.STREAM_GRAD, 0, 0, 0), 0, 100_000, 1e-3)
    ours = gen.f32_to_bf16_bits(x)
    ref = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(ours, ref)
    assert np.array_equal(gen.bf16_bits_to_f32(ours), torch.from_numpy(x).to(torch.bfloat16).float().numpy())
