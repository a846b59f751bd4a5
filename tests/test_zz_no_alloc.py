"""hadpsgd_consensus_noalloc: the consensus distance for callers that cannot hand this
library any device memory.

Who they are: a process whose framework allocator already holds (nearly) the whole GPU, so that a raw
cudaMalloc inside a library fails; a monitor between two steps of a latency-bound training loop, where
cudaMalloc / cudaFree would stall every stream of the device; a hook that merely borrows S weight
tensors and has no arena of its own.  hadpsgd_consensus() needs a handle (hence an arena holding the
reduction's block partials); the no-allocation entry point keeps those partials in a fixed
HADPSGD_NOALLOC_SCRATCH_BYTES array inside libhadpsgd.so instead, takes only the S weight pointers
and a device double for the result, and is limited to S <= HADPSGD_NOALLOC_MAX_S buffers.

What is checked: its result against the existing handle path (and the CPU oracle) on two calls in a
row that share the scratch array -- a large problem first, then a smaller one with a ragged length,
then the large one again -- at the tolerance the consensus tests of test_parity_gpu.py use (rel 1e-10),
that the calls leave the device's free memory untouched, and that sizes beyond the limits are refused
with a message.  This file sorts last on purpose (`pytest --collect-only`): with -x a failure here
cannot hide a test behind it.  It passes alone in a fresh process (its first call then does the
per-device set-up) and after the rest of the suite.
"""
import os

import numpy as np
import pytest

REL = 1e-10          # the bar of test_consensus_distance_and_variance_identity
MAX_S, MAX_BLOCKS, SCRATCH_BYTES, MAX_ELEMS = 64, 2048, (2048 + 32) * 8, 1 << 36   # include/hadpsgd.h


@pytest.fixture(scope="module")
def H():
    import paper_1907_05701_b200 as m
    m.lib()                      # fail loudly if the extension is missing
    return m


def test_limits_are_refused_with_a_message_before_any_gpu_work(H):
    """No GPU needed: argument checks come before the first CUDA call, so a caller that asks for more
    than the fixed tables hold learns it from the status and the text, not from a fault."""
    with pytest.raises(H.HadpsgdError, match="HADPSGD_NOALLOC_MAX_S"):
        H.hadpsgd_consensus_noalloc([256 * (i + 1) for i in range(MAX_S + 1)], 1024, 256)
    with pytest.raises(H.HadpsgdError, match="HADPSGD_NOALLOC_MAX_ELEMS"):
        H.hadpsgd_consensus_noalloc([256, 512], MAX_ELEMS + 1, 256)
    with pytest.raises(H.HadpsgdError, match="at least one"):
        H.hadpsgd_consensus_noalloc([], 1024, 256)
    with pytest.raises(H.HadpsgdError, match="16-byte aligned"):
        H.hadpsgd_consensus_noalloc([256, 516], 1024, 256)
    with pytest.raises(H.HadpsgdError, match="NULL"):
        H.hadpsgd_consensus_noalloc([256, 0], 1024, 256)
    with pytest.raises(H.HadpsgdError, match="NULL"):
        H.hadpsgd_consensus_noalloc([256, 512], 1024, 0)
    src = open(os.path.join(os.path.dirname(H.__file__), "..", "include", "hadpsgd.h")).read()
    for name, val in (("MAX_S", "64"), ("MAX_BLOCKS", "2048")):
        assert f"#define HADPSGD_NOALLOC_{name} {val}" in src      # the constants this file repeats


@pytest.mark.gpu
def test_no_alloc_consensus_equals_the_handle_path_on_consecutive_calls(H, oracle_mod):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from fixtures import problem
    stream = torch.cuda.current_stream()
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")   # the caller's output memory

    def both(S, seg, seed):
        """D through the handle (existing path), through the no-allocation entry point, and the oracle's."""
        h = H.Hadpsgd(S, 2, seg, H.F32, H.DETERMINISTIC)
        problem.fill_weights(h, seed)
        P = sum(seg)
        d_handle = h.hadpsgd_consensus()
        ptrs = [h.hadpsgd_weights(s).data_ptr() for s in range(S)]
        return h, ptrs, d_handle, oracle_mod.consensus_distance(problem.host_weights(seed, S, 0, P))

    # call 1: enough elements for the full grid (#SMs x 8 blocks): every partial slot in use
    S1, P1 = 8, 1_300_032
    h1, ptrs1, d1_handle, d1_oracle = both(S1, [P1], 501)
    H.hadpsgd_consensus_noalloc(ptrs1, h1.P_padded, out[0:1].data_ptr(), stream.cuda_stream)
    # call 2, straight behind it on the same stream: a SMALLER problem (fewer blocks, so the scratch
    # still holds call 1's partials behind this grid and the counter must have gone back to zero) ...
    S2, seg2 = 5, [1, 3, 7, 1025, 64, 63, 65, 4099, 2, 100_001]
    h2, ptrs2, d2_handle, d2_oracle = both(S2, seg2, 502)
    free_before = torch.cuda.mem_get_info()[0]
    H.hadpsgd_consensus_noalloc(ptrs2, h2.P_padded, out[1:2].data_ptr(), stream.cuda_stream)
    # ... and call 3: a ragged length (not a multiple of 4) over contiguous flat weights
    n3 = 70_003
    flat = problem.host_weights(503, 3, 0, n3)
    flat_dev = [torch.from_numpy(flat[s]).cuda() for s in range(3)]
    free_before3 = torch.cuda.mem_get_info()[0]
    H.hadpsgd_consensus_noalloc([t.data_ptr() for t in flat_dev], n3, out[2:3].data_ptr(), stream.cuda_stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before3      # nothing was allocated by call 3 ...
    assert torch.cuda.mem_get_info()[0] >= free_before       # ... nor by call 2 (call 1 may load the kernel image)
    got = out.cpu().numpy()
    assert got[0] == pytest.approx(d1_handle, rel=REL) and got[0] == pytest.approx(d1_oracle, rel=REL)
    assert got[1] == pytest.approx(d2_handle, rel=REL) and got[1] == pytest.approx(d2_oracle, rel=REL)
    assert got[2] == pytest.approx(oracle_mod.consensus_distance(flat), rel=REL)
    assert d1_handle > 0 and d2_handle > 0 and got[2] > 0
    # same buffers, same grid as hadpsgd_consensus, same summation order: the bits agree on a B200
    props = torch.cuda.get_device_properties(0)
    if props.multi_processor_count * 8 <= MAX_BLOCKS:
        assert got[0] == d1_handle and got[1] == d2_handle
    # repeat call 1 after the others: stale partials and the shared counter change nothing
    again = torch.zeros(1, dtype=torch.float64, device="cuda")
    H.hadpsgd_consensus_noalloc(ptrs1, h1.P_padded, again.data_ptr(), stream.cuda_stream)
    H.hadpsgd_consensus_noalloc(ptrs1, h1.P_padded, out[1:2].data_ptr(), stream.cuda_stream)
    torch.cuda.synchronize()
    assert again.item() == got[0] and out[1].item() == got[0]
    # empty input: defined (D = 0), and a plain host pointer is refused instead of faulting in the kernel
    H.hadpsgd_consensus_noalloc(ptrs1, 0, again.data_ptr(), stream.cuda_stream)
    torch.cuda.synchronize()
    assert again.item() == 0.0
    host = np.zeros(16, np.float32)
    with pytest.raises(H.HadpsgdError, match="plain host pointer"):
        H.hadpsgd_consensus_noalloc([ptrs1[0], host.ctypes.data // 16 * 16], 4, again.data_ptr(), stream.cuda_stream)
    h1.close()
    h2.close()
