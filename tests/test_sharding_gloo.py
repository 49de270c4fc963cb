"""world_size-2 gloo test of the N>1 path's host logic: each rank handles a batch shard and the
shared-theta gradients are summed with one all-reduce; the result must equal the single-process batch sum.
The per-rank compute stands in with the oracle here (CPU box, no GPU); the exchange code is the product's."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads as W
    from oracle import cosmo_oracle as O
    from paper_2606_13825_b200.sharding import shard_indices, allreduce_shared_grads
    wl = W.make_config(1, batch=4, K=6)
    mine = shard_indices(wl.batch, rank, world)
    res = O.run_workload(wl, problems=mine)
    g = dict(g_rho=torch.tensor(res["g_rho"]), g_alpha=torch.tensor(res["g_alpha"]), g_sigma=torch.tensor([res["g_sigma"]], dtype=torch.float64))
    allreduce_shared_grads(g)
    if rank == 0:
        ret["g_rho"] = g["g_rho"].numpy(); ret["g_alpha"] = g["g_alpha"].numpy(); ret["g_sigma"] = float(g["g_sigma"][0])
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_gradients_equal_single_process_sum():
    sys.path.insert(0, ROOT)
    import workloads as W
    from oracle import cosmo_oracle as O
    mgr = mp.Manager()
    ret = mgr.dict()
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    wl = W.make_config(1, batch=4, K=6)
    ref = O.run_workload(wl)
    np.testing.assert_allclose(ret["g_rho"], ref["g_rho"], rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(ret["g_alpha"], ref["g_alpha"], rtol=1e-12, atol=1e-12)
    assert abs(ret["g_sigma"] - ref["g_sigma"]) <= 1e-12 * max(1.0, abs(ref["g_sigma"]))
