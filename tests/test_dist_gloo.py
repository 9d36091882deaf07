"""World-size-2 gloo test (CPU) of the data-parallel plumbing (Eq. 37-38):
the sum over ranks of Phi_j^dagger y_j equals Phi^dagger y over the union of the visibilities, and Phi over
the union is the concatenation of the per-rank Phi_j x.  The per-rank operator here is the CPU oracle
(the CUDA library cannot run without a GPU); what is under test is dist.py."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1903_04502_b200 import dist as pdist
from inputs import synth


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert pdist.world() == (rank, rank, world)
        cfg, x, uv, w = synth.make_problem(1, M=3001)
        w = synth.rng_for(7, synth.STREAM_W).uniform(0.5, 1.5, size=len(uv))
        yv = synth.random_complex((len(uv),), seed=5)
        lo, hi = pdist.shard_bounds(len(uv), rank, world)
        oracle.set_num_threads(1)
        img = torch.from_numpy(oracle.grid(yv[lo:hi], uv[lo:hi], w[lo:hi], cfg.n, cfg.J))
        pdist.allreduce_image(img)
        y_part = oracle.degrid(x, uv[lo:hi], w[lo:hi], cfg.J)
        t = pdist.max_over_ranks(float(rank + 1))
        pdist.barrier()
        if rank == 0:
            full = oracle.grid(yv, uv, w, cfg.n, cfg.J)
            out["img_err"] = float(np.linalg.norm(img.numpy() - full) / np.linalg.norm(full))
            y_full = oracle.degrid(x, uv, w, cfg.J)
            out["y_err"] = float(np.linalg.norm(y_part - y_full[lo:hi]) / np.linalg.norm(y_full[lo:hi]))
            out["tmax"] = t
    finally:
        dist.destroy_process_group()


def test_shard_bounds_cover():
    for M in (0, 1, 7, 10, 3001):
        for ws in (1, 2, 3, 8):
            b = [pdist.shard_bounds(M, r, ws) for r in range(ws)]
            assert b[0][0] == 0 and b[-1][1] == M
            assert all(b[i][1] == b[i + 1][0] for i in range(ws - 1))
            assert max(h - l for l, h in b) - min(h - l for l, h in b) <= 1


def test_rank_config_seeds_differ():
    c0, c1 = pdist.rank_config(synth.CONFIGS[4], 0), pdist.rank_config(synth.CONFIGS[4], 1)
    assert c0.seed != c1.seed and c0.n == c1.n and c0.M == c1.M


def test_allreduce_image_two_ranks_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        assert out["img_err"] <= 1e-13, dict(out)      # Eq. (38): linearity of Phi^dagger in the visibility set
        assert out["y_err"] <= 1e-14, dict(out)        # Eq. (37): no exchange in Phi
        assert out["tmax"] == 2.0
