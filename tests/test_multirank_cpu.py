"""world_size-2 gloo test (CPU) of the N>1 host logic: pixel sharding, max-over-ranks timing,
whole-job rate, and that sharded lines of sight reproduce the unsharded result (no exchange step)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    import rmsynth_inputs as ri
    from paper_1810_06250_b200 import sharding as sh
    cfg = ri.scaled(ri.CONFIGS[1], 20)                       # 400 pixels: shards of 256 and 144
    nu, w, phi = ri.grids(cfg)
    lo, hi = sh.shard_pixels(cfg.n_pix, rank, world)
    q, u = ri.generate_pixels(cfg, torch.arange(lo, hi))
    plan = oracle.make_plan(nu, w, phi)
    FQ, FU = oracle.synth_table(plan, q.numpy(), u.numpy(), n_threads=1)
    t_max = sh.max_over_ranks(1.0 + rank)                     # slowest rank decides
    gathered = [None] * world
    dist.all_gather_object(gathered, (lo, hi, FQ, FU))        # test-only gather; the product path has none
    if rank == 0:
        out["t_max"] = t_max
        out["rate"] = sh.whole_job_rate(100.0, t_max, world)
        out["parts"] = gathered
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_without_exchange():
    import oracle
    import rmsynth_inputs as ri
    oracle.build()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert out["t_max"] == 2.0 and out["rate"] == 100.0
    parts = sorted(out["parts"], key=lambda x: x[0])
    assert parts[0][0] == 0 and parts[0][1] == parts[1][0] == 256 and parts[1][1] == 400
    cfg = ri.scaled(ri.CONFIGS[1], 20)
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(cfg.n_pix))
    FQ, FU = oracle.synth_table(oracle.make_plan(nu, w, phi), q.numpy(), u.numpy())
    assert np.array_equal(np.concatenate([p[2] for p in parts]), FQ)
    assert np.array_equal(np.concatenate([p[3] for p in parts]), FU)


def test_shard_pixels_partitions_exactly():
    from paper_1810_06250_b200 import sharding as sh
    for n_pix in (0, 1, 127, 128, 129, 4096, 262144, 4194304, 1000003):
        for world in (1, 2, 3, 4, 8):
            edges = [sh.shard_pixels(n_pix, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n_pix
            for a, b in zip(edges, edges[1:]):
                assert a[1] == b[0] and a[0] <= a[1]
            assert all(lo % 128 == 0 for lo, _ in edges)
    assert sh.rank_seed(5, 3) == 3005
