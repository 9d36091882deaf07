"""f3 - the distributed-image operator of PAPER.md:317-340 (Eq. 37-38; Algorithm 2) on the CUDA path.  -m gpu

(1) always runs on a one-GPU box: the visibility set cut into sections (shard_bounds), one handle per section on ONE
    device, no NCCL - sum_j Phi_j^dagger y_j and the concatenated Phi_j x against the oracle over the union, through
    purify_grid_dist / purify_normal_dist with a counting all-reduce callback (bands, ordering, aliasing);
(2) two NCCL ranks on two devices doing the same through torch.distributed - skipped where fewer than two GPUs are
    visible (NCCL refuses two ranks on one device)."""
import os
import socket

import numpy as np
import pytest
import torch

import oracle
from inputs import synth
from parity_util import compare

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _problem(dtype, M=60_000, J=6):
    cfg, x, uv, w = synth.make_problem(2, M=M, J=J)
    cd, rd = synth.complex_dtype(dtype), synth.real_dtype(dtype)
    return cfg, x.astype(cd), uv.astype(rd), w.astype(rd)


@pytest.mark.parametrize("dtype,parts", [("c64", 2), ("c64", 3), ("c128", 2)])
def test_sections_on_one_device_against_the_union(dtype, parts):
    from paper_1903_04502_b200 import C64, C128, PurifyOp
    from paper_1903_04502_b200 import dist as pdist
    cfg, x, uv, w = _problem(dtype)
    M, J, n = len(uv), 6, cfg.n
    tol = 1e-5 if dtype == "c64" else 1e-12
    prec = 32 if dtype == "c64" else 64
    dt = C64 if dtype == "c64" else C128
    yv = synth.random_complex((M,), seed=91, dtype=dtype)
    ops, bounds = [], []
    for r in range(parts):
        lo, hi = pdist.shard_bounds(M, r, parts)
        bounds.append((lo, hi))
        ops.append(PurifyOp(n, J, dev(uv[lo:hi]), dev(w[lo:hi]), dtype=dt))
    # Eq. (37): Phi over the union is the concatenation of the per-section Phi_j x - no exchange
    y_ref = oracle.degrid(x, uv, w, J, idx_prec=prec)
    y_cat = np.concatenate([op.degrid(dev(x)).cpu().numpy() for op in ops])
    compare("sections: concatenated Phi_j x", y_cat, y_ref, tol, dtype=dtype, parts=parts)
    # Eq. (38): sum_j Phi_j^dagger y_j.  The "all-reduce" of this one-process test adds the band into an accumulator:
    # what a sum over ranks does to rank 0's copy.
    img_ref = oracle.grid(yv, uv, w, n, J, idx_prec=prec)
    acc = torch.zeros((n, n), dtype=torch.complex64 if dtype == "c64" else torch.complex128, device="cuda")
    acc_flat = torch.view_as_real(acc).reshape(-1)
    calls = []
    for op, (lo, hi) in zip(ops, bounds):
        y_nat = op.permute_to_native(dev(yv[lo:hi]))
        out = torch.full_like(acc, float("nan"))
        base = torch.view_as_real(out).reshape(-1).data_ptr()

        def allreduce(band, base=base):
            off = (band.data_ptr() - base) // band.element_size()
            calls.append((off, band.numel()))
            acc_flat[off:off + band.numel()] += band          # runs on the handle's side stream, after the band's crop
        op.grid_dist(y_nat, out, allreduce=allreduce, bands=5)
        torch.cuda.synchronize()
        # the bands tile the image exactly (gridding is not bit-reproducible from call to call: compare to the tolerance)
        compare("sections: banded crop vs plain", out.cpu().numpy(), op.grid(y_nat, native=True).cpu().numpy(), tol, dtype=dtype)
    compare("sections: sum_j Phi_j^dagger y_j", acc.cpu().numpy(), img_ref, tol, dtype=dtype, parts=parts)
    per_op = len(calls) // parts
    assert per_op == 5 and sum(c for _, c in calls[:5]) == 2 * n * n and [o for o, _ in calls[:5]] == sorted(o for o, _ in calls[:5])
    # Phi^dagger Phi, distributed: sum_j Phi_j^dagger Phi_j x; in place (x_out = x_in) on a copy
    nrm_ref = oracle.grid(y_ref, uv, w, n, J, idx_prec=prec)
    acc.zero_()
    for op in ops:
        xin = dev(x)
        op.normal_dist(xin, xin, allreduce=None, bands=3)
        acc += xin
    compare("sections: sum_j Phi_j^dagger Phi_j x", acc.cpu().numpy(), nrm_ref, tol, dtype=dtype, parts=parts)
    for op in ops:
        op.close()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _nccl_worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_1903_04502_b200 import C64, PurifyOp
    from paper_1903_04502_b200 import dist as pdist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        cfg, x, uv, w = _problem("c64")
        lo, hi = pdist.shard_bounds(len(uv), rank, world)
        op = PurifyOp(cfg.n, 6, dev(uv[lo:hi]), dev(w[lo:hi]), dtype=C64)
        res = op.normal_dist(dev(x), None, allreduce=lambda band: dist.all_reduce(band, op=dist.ReduceOp.SUM), bands=4)
        torch.cuda.synchronize()
        if rank == 0:
            y_ref = oracle.degrid(x, uv, w, 6, idx_prec=32)
            nrm_ref = oracle.grid(y_ref, uv, w, cfg.n, 6, idx_prec=32)
            a = res.cpu().numpy()
            out["err"] = float(np.linalg.norm(a - nrm_ref) / np.linalg.norm(nrm_ref))
        op.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices: NCCL refuses two ranks on one device")
def test_two_nccl_ranks_allreduce_inside_normal_dist():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_nccl_worker, args=(world, port, out), nprocs=world, join=True)
        assert out["err"] <= 1e-5, dict(out)
