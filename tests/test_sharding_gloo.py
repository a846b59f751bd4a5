"""Multi-rank path on CPU: world_size 2 over gloo.

Each rank takes its parameter range from the PRODUCT library (hadpsgd_shard_range, host-only),
runs the step arithmetic on that range (the oracle stands in for the GPU kernel here: there is
no GPU and the product has no CPU fallback), and the diagnostics are summed with the product's
allreduce helper -- the same helpers bench.py --gpus N uses.  Rank 0 checks that the sharded run
reproduces the unsharded one: w, v bit for bit, diagnostics to rounding."""
import os
import socket

import numpy as np
import pytest

S, G, P, STEPS, SEED = 4, 2, 64 * 1001, 3, 17
LR, MU = 0.1, 0.9


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    import oracle
    from fixtures import problem
    from paper_1907_05701_b200 import sharding
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lo, hi = sharding.rank_shard(P, dist)
        w, v = problem.host_weights(SEED, S, lo, hi), np.zeros((S, hi - lo), np.float32)
        diags = []
        for k in range(STEPS):
            d = oracle.step(problem.host_grads(SEED, k, S, G, lo, hi), w, v, LR, MU, k, diag=True)
            diags.append(sharding.allreduce_diagnostics(d, dist))
        t = sharding.max_over_ranks(1.0 + rank, dist)
        assert t == float(world)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), lo=lo, hi=hi, w=w, v=v,
                 gsq=np.stack([d["gsq"] for d in diags]), wsq=np.stack([d["wsq"] for d in diags]),
                 gap=np.stack([d["gap"] for d in diags]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_sharded_run_equals_unsharded(tmp_path, oracle_mod):
    import torch.multiprocessing as mp
    from fixtures import problem
    from paper_1907_05701_b200 import build as b
    b.build()
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w, v = problem.host_weights(SEED, S, 0, P), np.zeros((S, P), np.float32)
    full = [oracle_mod.step(problem.host_grads(SEED, k, S, G, 0, P), w, v, LR, MU, k, diag=True) for k in range(STEPS)]
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert int(parts[0]["lo"]) == 0 and int(parts[0]["hi"]) == int(parts[1]["lo"]) and int(parts[1]["hi"]) == P
    gw = np.concatenate([p["w"] for p in parts], axis=1)
    gv = np.concatenate([p["v"] for p in parts], axis=1)
    assert np.array_equal(gw.view(np.uint32), w.view(np.uint32))
    assert np.array_equal(gv.view(np.uint32), v.view(np.uint32))
    for p in parts:                                   # every rank holds the GLOBAL diagnostics
        for k in range(STEPS):
            for name in ("gsq", "wsq", "gap"):
                assert np.allclose(p[name][k], full[k][name], rtol=1e-12, atol=0)
