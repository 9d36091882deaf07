"""Parity at BASELINE.json's FULL sizes (configs 3, 4, 5), through the C ABI in the launch configuration
bench.py times (native order, default options).  -m gpu

The oracle is fast enough (OpenMP) to compute the whole Phi x and Phi^dagger y at these sizes, so the
comparison is over the complete outputs, plus properties that hold at any size (adjoint identity,
order invariance).  Tolerance: rel-L2 <= 1e-5 (complex64), <= 1e-12 (complex128) - BASELINE.json north_star.
Set PURIFY_SKIP_HUGE=1 to skip config 5 (5e8 visibilities: ~50 GB of host memory, minutes of CPU oracle)."""
import os

import numpy as np
import pytest
import torch

import oracle
from inputs import synth
from parity_util import compare

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

TOL = {"c128": 1e-12, "c64": 1e-5}


def rel_l2(a, b):
    from parity_util import errors
    return errors(a, b)[0]


def full_size_checks(cfg, x, uv, w, dtype, order=None):
    """Phi and Phi^dagger over the whole visibility set against the oracle; returns (y_gpu caller order, image)."""
    from paper_1903_04502_b200 import ANALYTIC, C64, C128, TABLE, PurifyOp
    cd, rd = synth.complex_dtype(dtype), synth.real_dtype(dtype)
    x, uv, w = x.astype(cd), np.ascontiguousarray(uv.astype(rd)), w.astype(rd)
    if order is not None:
        uv, w = np.ascontiguousarray(uv[order]), np.ascontiguousarray(w[order])
    M, tol = len(uv), TOL[dtype]
    table = cfg.kernel_mode == "table"
    okw = dict(mode=cfg.kernel_mode, R=cfg.table_R, idx_prec=32 if dtype == "c64" else 64)
    op = PurifyOp(cfg.n, cfg.J, torch.from_numpy(uv).cuda(), torch.from_numpy(w).cuda(),
                  dtype=C64 if dtype == "c64" else C128, kernel_mode=TABLE if table else ANALYTIC,
                  table_samples_per_unit=cfg.table_R if table else 0)
    info = op.info()
    assert info["M"] == M and info["M_native"] >= M
    xd = torch.from_numpy(x).cuda()
    # ---- Phi, native order (what bench.py times), compared through the permutation
    y_nat = op.degrid(xd, native=True)
    y = op.permute_from_native(y_nat).cpu().numpy()
    y_ref = oracle.degrid(x, uv, w, cfg.J, **okw)
    ctx = dict(config=cfg.index, n=cfg.n, J=cfg.J, M=M, dtype=dtype, mode=cfg.kernel_mode, order="shuffled" if order is not None else "as generated")
    compare("full size Phi", y, y_ref, tol, **ctx)
    y_call = op.degrid(xd).cpu().numpy()
    assert np.array_equal(y_call, y)
    # ---- Phi^dagger on the oracle's Phi x (rounded to storage), native order
    yv = y_ref.astype(cd)
    del y_ref
    img_ref = oracle.grid(yv, uv, w, cfg.n, cfg.J, **okw)
    yv_nat = op.permute_to_native(torch.from_numpy(yv).cuda())
    img = op.grid(yv_nat, native=True).cpu().numpy()
    compare("full size Phi^dagger", img, img_ref, tol, **ctx)
    # ---- Phi^dagger Phi (the bench step)
    nrm = op.normal(xd).cpu().numpy()
    compare("full size Phi^dagger Phi", nrm, img_ref, tol, **ctx)
    compare("full size Phi^dagger Phi (graph replay)", op.normal(xd).cpu().numpy(), img_ref, tol, **ctx)
    # ---- adjoint identity with GPU results: <Phi x, y> = <x, Phi^dagger y>
    lhs = complex(np.vdot(y.astype(np.complex128), yv.astype(np.complex128)))
    rhs = complex(np.vdot(x.astype(np.complex128), img.astype(np.complex128)))
    assert abs(lhs - rhs) / (np.linalg.norm(y.astype(np.complex128)) * np.linalg.norm(yv.astype(np.complex128))) <= tol
    op.close()
    del xd, y_nat, yv_nat
    torch.cuda.empty_cache()
    return y, img, info


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_config3_rotation_synthesis_both_orders(dtype):
    """BASELINE.json configs[2]: 1024^2 image, J=4, M=1e7 from a 27-antenna track; time-ordered and shuffled
    input must give the same y up to the permutation (and the same image)."""
    cfg, x, uv, w = synth.make_problem(3)
    y_t, img_t, info = full_size_checks(cfg, x, uv, w, dtype)
    order = synth.shuffle_order(cfg.M, cfg.seed)
    y_s, img_s, _ = full_size_checks(cfg, x, uv, w, dtype, order=order)
    assert np.array_equal(y_s, y_t[order])                       # each visibility is computed on its own: same bits
    assert rel_l2(img_s, img_t) <= TOL[dtype]
    if dtype == "c64":
        assert info["layout"] == 1 and info["M_native"] < 1.5 * cfg.M


def test_config4_full_size():
    """BASELINE.json configs[3], the metric's config: 2048^2 image, J=6, M=1e8 Gaussian-density visibilities."""
    cfg, x, uv, w = synth.make_problem(4)
    _, _, info = full_size_checks(cfg, x, uv, w, "c64")
    assert info["M_native"] <= 1.10 * cfg.M                      # padding of the batched layout stays small


@pytest.mark.skipif(os.environ.get("PURIFY_SKIP_HUGE") == "1", reason="PURIFY_SKIP_HUGE=1")
def test_config5_full_size_table_mode():
    """BASELINE.json configs[4]: 4096^2 image, J=4, M=5e8 from a 197-antenna SKA-like layout, pre-sampled
    kernel table with 4096 samples per unit."""
    cfg, x, uv, w = synth.make_problem(5)
    full_size_checks(cfg, x, uv, w, "c64")


def test_config4_admm_fidelity_step_full_size():
    """f1 at the metric's config (fused complex64 kernels, the launch configuration bench.py times): g, the updated dual
    variable and the residual norm against the oracle over all 1e8 visibilities."""
    from paper_1903_04502_b200 import C64, PurifyOp
    cfg, x, uv, w = synth.make_problem(4)
    M = cfg.M
    op = PurifyOp(cfg.n, cfg.J, torch.from_numpy(uv).cuda(), torch.from_numpy(w).cuda(), dtype=C64)
    y = synth.random_complex((M,), seed=61, dtype="c64")
    s = (synth.random_complex((M,), seed=62, dtype="c64") * np.float32(0.2)).astype(np.complex64)
    v = oracle.degrid(x, uv, w, cfg.J, idx_prec=32)
    eps = 0.5 * float(np.sqrt(sum(float(np.vdot(d, d).real) for d in
                                  ((v[i:i + (1 << 24)] + s[i:i + (1 << 24)] - y[i:i + (1 << 24)]) for i in range(0, M, 1 << 24)))))
    del v
    g_ref, s_ref, _, nrm_ref = oracle.admm_fidelity_step(x, y, s, uv, w, cfg.n, cfg.J, eps, 0.9, idx_prec=32)
    y_nat = op.permute_to_native(torch.from_numpy(y).cuda())
    s_nat = op.permute_to_native(torch.from_numpy(s).cuda())
    g, nrm = op.admm_fidelity_step(torch.from_numpy(x).cuda(), y_nat, s_nat, eps, 0.9)
    assert abs(nrm - nrm_ref) <= 1e-5 * nrm_ref
    ctx = dict(config=4, n=cfg.n, J=cfg.J, M=M, dtype="c64")
    compare("full size ADMM g", g.cpu().numpy(), g_ref, 1e-5, **ctx)
    s_out = op.permute_from_native(s_nat).cpu().numpy()
    compare("full size ADMM s_new", s_out, s_ref, 1e-5, **ctx)
    op.close()
