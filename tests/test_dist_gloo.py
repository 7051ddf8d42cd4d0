"""world_size-2 gloo test (CPU) of the N>1 host logic: token sharding + the LoRA-gradient
all-reduce reproduce the unsharded oracle result."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    from oracle import layer as olayer
    from paper_2607_05711_b200 import parallel, synth
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    M, K, N, r_s, r = 50, 64, 48, 2, 4
    d = synth.layer_inputs(7, M, K, N, r)
    rng = synth.make_rng(8)
    H = synth.normal(rng, (M, r_s + r), 1.0)
    P = synth.normal(rng, (M, r_s + r), 1.0)
    lo, hi = parallel.shard_rows(M, rank, world)
    w = olayer.wgrad(d["X"][lo:hi], d["dY"][lo:hi], H[lo:hi], P[lo:hi], r_s)
    dA, dBt = torch.from_numpy(w["dA"].copy()), torch.from_numpy(np.ascontiguousarray(w["dB"].T))
    parallel.allreduce_lora_grads(dA, dBt)
    full = olayer.wgrad(d["X"], d["dY"], H, P, r_s)
    amax = parallel.allreduce_amax(torch.tensor([float(np.abs(d["X"][lo:hi]).max())]))
    ok = (np.allclose(dA.numpy(), full["dA"], rtol=1e-5, atol=1e-6)
          and np.allclose(dBt.numpy().T, full["dB"], rtol=1e-5, atol=1e-6)
          and float(amax) == float(np.abs(d["X"]).max()))
    ret[rank] = bool(ok)
    dist.destroy_process_group()


def test_shard_rows_partition():
    from paper_2607_05711_b200 import parallel
    for M in (1, 7, 256, 4608):
        for world in (1, 2, 3, 8):
            spans = [parallel.shard_rows(M, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == M
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def test_sharded_wgrad_allreduce_world2():
    world = 2
    port = 29000 + os.getpid() % 2000
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    assert all(ret.get(r) for r in range(world))
