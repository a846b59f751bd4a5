"""Host-only helpers of the product library (no GPU): the LR recipe of PAPER.md:70 against the
values the paper prints (tests/golden/lr_schedule_paper_example.txt) and the parameter-range
split used for multi-GPU sharding."""
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "lr_schedule_paper_example.txt")


@pytest.fixture(scope="module")
def H():
    from paper_1907_05701_b200 import build as b
    b.build()
    import paper_1907_05701_b200 as m
    return m


def test_lr_schedule_matches_paper_example(H):
    """baseline batch 256 at lr 0.1, total batch 2560 -> +0.1 per epoch, 1.0 at the
    10th epoch, then x 1/sqrt(2) per epoch."""
    rows = [line.split() for line in open(GOLDEN) if line.strip() and not line.startswith("#")]
    assert len(rows) == 16
    for epoch, lr in rows:
        got = H.hadpsgd_lr_schedule(0.1, 256, 2560, 10, int(epoch))
        assert got == pytest.approx(float(lr), rel=1e-12, abs=1e-15), (epoch, got, lr)


def test_lr_schedule_properties(H):
    # linear scaling: the peak is base_lr * ratio, whatever the ratio
    for ratio in (1, 4, 16, 32, 48):
        assert H.hadpsgd_lr_schedule(0.1, 256, 256 * ratio, 10, 10) == pytest.approx(0.1 * ratio, rel=1e-15)
        assert H.hadpsgd_lr_schedule(0.1, 256, 256 * ratio, 10, 1) == pytest.approx(0.1, rel=1e-15)
        # two annealing epochs halve the rate
        a = H.hadpsgd_lr_schedule(0.1, 256, 256 * ratio, 10, 12)
        assert a == pytest.approx(0.05 * ratio, rel=1e-14)
    # monotone up then down
    lrs = [H.hadpsgd_lr_schedule(0.1, 256, 8192, 10, e) for e in range(1, 17)]
    assert all(x < y for x, y in zip(lrs[:9], lrs[1:10])) and all(x > y for x, y in zip(lrs[9:], lrs[10:]))
    assert H.hadpsgd_lr_schedule(0.1, 256, 2560, 1, 1) == pytest.approx(1.0)
    for bad in ((0.0, 256, 2560, 10, 1), (0.1, 0, 2560, 10, 1), (0.1, 256, -1, 10, 1), (0.1, 256, 2560, 0, 1),
                (0.1, 256, 2560, 10, 0)):
        with pytest.raises(H.HadpsgdError):
            H.hadpsgd_lr_schedule(*bad)


@pytest.mark.parametrize("blocks", [0, 1, 2, 7, 8, 9, 1000, 2267896])
@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_shard_ranges_partition_the_buffer(H, blocks, world):
    P = blocks * 64
    ranges = [H.hadpsgd_shard_range(P, world, r) for r in range(world)]
    assert ranges[0][0] == 0 and ranges[-1][1] == P
    for (lo, hi), (lo2, _) in zip(ranges, ranges[1:]):
        assert hi == lo2                                   # contiguous, ordered, disjoint
    sizes = np.array([hi - lo for lo, hi in ranges])
    assert np.all(sizes % 64 == 0) and sizes.max() - sizes.min() <= 64   # balanced to one block
    assert np.all(np.diff(sizes) <= 0)                     # the first ranks take the remainder


def test_shard_range_errors(H):
    for bad in ((63, 2, 0), (64, 0, 0), (64, 2, 2), (64, 2, -1), (-64, 2, 0)):
        with pytest.raises(H.HadpsgdError):
            H.hadpsgd_shard_range(*bad)
