"""Parity of the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element on the same seeded inputs.  -m gpu

Tolerances (BASELINE.json north_star): rel-L2 <= 1e-12 for complex128, <= 1e-5 for complex64,
over the whole output vector / image."""
import numpy as np
import pytest
import torch

import oracle
from inputs import synth
from parity_util import compare

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-12, "c64": 1e-5}
# Composite operators (Phi^dagger Phi, the ADMM data-fidelity step, its residual norm) get NO multiple of the tolerance:
# measured, they stay below 0.09 tol (profiles/parity_r2.md).
ADMM_FACTOR = 1.0
ADMM_NORM_FACTOR = 1.0


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def make_op(n, J, uv, w, dtype, **kw):
    from paper_1903_04502_b200 import C64, C128, PurifyOp
    dt = C64 if dtype == "c64" else C128
    uvt = torch.from_numpy(np.ascontiguousarray(uv)).cuda()
    wt = None if w is None else torch.from_numpy(np.ascontiguousarray(w)).cuda()
    return PurifyOp(n, J, uvt, wt, dtype=dt, **kw)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def idx_prec(dtype):
    return 32 if dtype == "c64" else 64


def cast_problem(x, uv, w, dtype):
    """Round the problem to the storage precision of `dtype` (the oracle then promotes exactly)."""
    cd, rd = synth.complex_dtype(dtype), synth.real_dtype(dtype)
    return x.astype(cd), uv.astype(rd), None if w is None else w.astype(rd)


def run_all_checks(x, uv, w, J, dtype, mode="analytic", R=4096, **kw):
    """degrid (caller + native order), grid (both orders), normal, stages - all against the oracle, rel-L2 over the
    whole output AND the largest element-wise deviation (parity_util.compare)."""
    from paper_1903_04502_b200 import ANALYTIC, TABLE
    n = x.shape[0]
    tol = TOL[dtype]
    x, uv, w = cast_problem(x, uv, w, dtype)
    M = len(uv)
    op = make_op(n, J, uv, w, dtype, kernel_mode=TABLE if mode == "table" else ANALYTIC,
                 table_samples_per_unit=R if mode == "table" else 0, **kw)
    okw = dict(mode=mode, R=R, idx_prec=idx_prec(dtype))
    ctx = dict(n=n, J=J, M=M, dtype=dtype, mode=mode)
    # ---- Phi
    y_ref = oracle.degrid(x, uv, w, J, **okw)
    y = host(op.degrid(dev(x)))
    compare("Phi caller order", y, y_ref, tol, **ctx)
    perm = host(op.permutation())                          # M_native entries, -1 = padding (complex64 layout)
    valid = perm >= 0
    assert len(perm) == op.M_native >= M
    assert sorted(perm[valid].tolist()) == list(range(M))
    y_nat = host(op.degrid(dev(x), native=True))
    compare("Phi native order", y_nat[valid], y_ref[perm[valid]], tol, **ctx)
    assert np.array_equal(y_nat[valid], y[perm[valid]])     # same numbers, different order
    assert not np.any(y_nat[~valid])                        # padding entries are written as 0
    # stage: Fourier grid in the mathematical layout
    B_ref = oracle.fft2(oracle.pad(x, J), -1)
    compare("F Z S x", host(op.stage_fourier_grid(dev(x))), B_ref, tol, **ctx)
    # ---- Phi^dagger on random data (caller order and native order)
    yv = synth.random_complex((M,), seed=77, dtype=dtype)
    img_ref = oracle.grid(yv, uv, w, n, J, **okw)
    img = host(op.grid(dev(yv)))
    compare("Phi^dagger caller order", img, img_ref, tol, **ctx)
    yv_nat = np.full(len(perm), np.nan + 1j * np.nan, dtype=yv.dtype)     # padding holds NaN: must be ignored
    yv_nat[valid] = yv[perm[valid]]
    img_nat = host(op.grid(dev(yv_nat), native=True))
    compare("Phi^dagger native order", img_nat, img_ref, tol, **ctx)
    Bp_ref = oracle.grid_to_grid(yv, uv, w, 2 * n, J, **okw)
    compare("G^dagger W^dagger y", host(op.stage_gridded(dev(yv))), Bp_ref, tol, **ctx)
    # permutation helpers
    to_nat = host(op.permute_to_native(dev(yv)))
    assert np.array_equal(to_nat[valid], yv[perm[valid]]) and not np.any(to_nat[~valid])
    assert np.array_equal(host(op.permute_from_native(dev(yv_nat))), yv)
    # ---- Phi^dagger Phi
    nrm_ref = oracle.grid(y_ref, uv, w, n, J, **okw)
    xin = dev(x)
    nrm = host(op.normal(xin))
    compare("Phi^dagger Phi", nrm, nrm_ref, tol, **ctx)
    for _ in range(3):                                     # replayed from the CUDA graph: the same result
        compare("Phi^dagger Phi (graph replay)", host(op.normal(xin)), nrm_ref, tol, **ctx)
    # in place
    op.normal(xin, out=xin)
    compare("Phi^dagger Phi in place", host(xin), nrm_ref, tol, **ctx)
    # ---- adjoint identity evaluated with GPU results
    xr = synth.random_complex((n, n), seed=78, dtype=dtype)
    Px = host(op.degrid(dev(xr))).astype(np.complex128)
    Pty = img.astype(np.complex128)
    lhs, rhs = np.vdot(Px, yv.astype(np.complex128)), np.vdot(xr.astype(np.complex128), Pty)
    assert abs(lhs - rhs) / (np.linalg.norm(Px) * np.linalg.norm(yv)) <= tol
    # ---- host-buffer entry points give the same numbers
    yh = op.degrid_host(torch.from_numpy(x).pin_memory()).numpy()
    assert np.array_equal(yh, y)
    nh = op.normal_host(torch.from_numpy(x).pin_memory()).numpy()
    compare("Phi^dagger Phi host buffers", nh, nrm_ref, tol, **ctx)
    gh = op.grid_host(torch.from_numpy(yv).pin_memory()).numpy()
    compare("Phi^dagger host buffers", gh, img_ref, tol, **ctx)
    info = op.info()
    op.close()
    return info


# ------------------------------------------------------------------ config 1 (tiny)
@pytest.mark.parametrize("J", [4, 6, 8])
@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_config1_tiny(J, dtype):
    cfg, x, uv, w = synth.make_problem(1, J=J)
    info = run_all_checks(x, uv, w, J, dtype)
    assert info["M"] == cfg.M and info["K"] == 256
    assert info["poly_max_abs_err"] < (2e-7 if dtype == "c64" else 2e-15)


def test_config1_small_chunks():
    """Tile-sorted complex128 kernels (the default for J = 8, forced here for J = 4 and 6): many work items per tile
    (chunk 32 / 96) exercise the chunk flush / ragged tails."""
    cfg, x, uv, w = synth.make_problem(1)
    w = synth.rng_for(1, 1).uniform(0.5, 1.5, size=len(uv))
    for J, chunk in ((4, 32), (4, 96), (6, 64)):
        info = run_all_checks(x, uv, w, J, "c128", chunk=chunk, tile_sorted=True)
        assert info["layout"] == 0 and info["n_items"] > info["n_tiles_nonempty"]
    assert run_all_checks(x, uv, w, 4, "c128")["layout"] == 1        # default: the batched layout


# ------------------------------------------------------------------ config 2
@pytest.mark.parametrize("J", [4, 8])
def test_config2(J):
    cfg, x, uv, w = synth.make_problem(2, J=J)
    info = run_all_checks(x, uv, w, J, "c128")
    assert info["M"] == 250_000


def test_config2_noisy_data_adjoint():
    """BASELINE.json configs[1]: y = Phi x + noise at 30 dB; Phi^dagger y against the oracle."""
    cfg, x, uv, w = synth.make_problem(2)
    y0 = oracle.degrid(x, uv, w, 4)
    y = synth.add_noise(y0, 30.0, cfg.seed)
    assert np.linalg.norm(y - y0) / np.linalg.norm(y0) == pytest.approx(10 ** (-30 / 20), rel=0.02)
    op = make_op(cfg.n, 4, uv, w, "c128")
    compare("Phi^dagger on noisy data", host(op.grid(dev(y))), oracle.grid(y, uv, w, cfg.n, 4), TOL["c128"], n=cfg.n, J=4, M=len(uv), dtype="c128")
    op.close()


# ------------------------------------------------------------------ table mode
@pytest.mark.parametrize("dtype,J,R", [("c64", 4, 4096), ("c128", 4, 4096), ("c64", 6, 1000), ("c128", 8, 200000)])
def test_table_mode(dtype, J, R):
    cfg, x, uv, w = synth.make_problem(2, M=40_000, J=J)
    run_all_checks(x, uv, w, J, dtype, mode="table", R=R)


# ------------------------------------------------------------------ edge cases
def test_wrap_and_out_of_period_uv():
    """R8: taps that fall off the grid edge wrap; uv outside (-K/2, K/2) is taken mod K."""
    n, K = 64, 128
    x = synth.random_complex((n, n), seed=5)
    rng = synth.rng_for(5, 1)
    uv = rng.uniform(-K / 2, K / 2, size=(5000, 2))
    uv[:6] = [(-K / 2, -K / 2), (K / 2 - 1e-9, K / 2 - 1e-9), (K / 2 - 1e-9, 0.25), (-K / 2 + 0.5, K / 2 - 0.5),
              (K / 2 + 3.25, -K / 2 - 7.5), (5 * K + 1.5, -3 * K - 2.25)]
    w = rng.uniform(0.5, 1.5, size=5000)
    for dtype in ("c128", "c64"):
        for J in (4, 8):
            run_all_checks(x, uv, w, J, dtype)


def test_integer_and_half_integer_uv_tie_break():
    """R7: taps are the integers in (u - J/2, u + J/2]; crafted integer / half-integer coordinates."""
    n = 32
    x = synth.random_complex((n, n), seed=6)
    g = np.arange(-20, 20)
    uu, vv = np.meshgrid(g * 0.5, g * 0.5)
    uv = np.stack([uu.ravel(), vv.ravel()], axis=1)
    for dtype in ("c128", "c64"):
        run_all_checks(x, uv, None, 4, dtype)
        run_all_checks(x, uv, None, 6, dtype, mode="table", R=4096)


@pytest.mark.parametrize("n", [48, 50, 22, 8, 6])
def test_non_power_of_two_grid(n):
    """K = 96 (multiple of the tile), K = 100 and K = 44 (ragged edge tiles, non-power-of-two wrap), K = 16 and K = 12
    (grid smaller than one band box: every box wraps, some of them more than once)."""
    K = 2 * n
    x = synth.random_complex((n, n), seed=n)
    rng = synth.rng_for(n, 2)
    uv = rng.uniform(-K / 2, K / 2, size=(3000, 2))
    w = rng.uniform(0.5, 1.5, size=3000)
    run_all_checks(x, uv, w, 4, "c128")
    run_all_checks(x, uv, w, 6, "c64")


def test_empty_and_single_visibility():
    from paper_1903_04502_b200 import C128, PurifyOp
    n = 32
    x = synth.random_complex((n, n), seed=8)
    op = PurifyOp(n, 4, torch.empty((0, 2), dtype=torch.float64, device="cuda"), None, dtype=C128)
    y = op.degrid(dev(x))
    assert y.numel() == 0
    img = op.grid(y)
    assert float(img.abs().max()) == 0.0
    assert float(op.normal(dev(x)).abs().max()) == 0.0
    op.close()
    uv = np.array([[3.3, -7.7]])
    run_all_checks(x, uv, np.array([1.25]), 4, "c128")


def test_all_visibilities_in_one_cell():
    """Degenerate distribution: one cell holds every visibility (longest possible runs)."""
    n = 64
    x = synth.random_complex((n, n), seed=9)
    rng = synth.rng_for(9, 1)
    uv = np.stack([10 + rng.uniform(0, 1, 5000), -3 + rng.uniform(0, 1, 5000)], axis=1)
    run_all_checks(x, uv, rng.uniform(0.5, 1.5, 5000), 6, "c128", chunk=512)
    run_all_checks(x, uv, rng.uniform(0.5, 1.5, 5000), 4, "c64")


def test_errors():
    from paper_1903_04502_b200 import C64, C128, PurifyError, PurifyOp
    uv = torch.zeros((10, 2), dtype=torch.float64, device="cuda")
    for kw, code in [(dict(n=31, J=4), -1), (dict(n=32, J=5), -1), (dict(n=32, J=4, oversample=3), -2),
                     (dict(n=32, J=4, kernel_mode=7), -2), (dict(n=0, J=4), -1)]:
        with pytest.raises(PurifyError) as ei:
            PurifyOp(kw.pop("n"), kw.pop("J"), uv, None, dtype=C128, **kw)
        assert ei.value.status == code
    bad = uv.clone()
    bad[3, 1] = float("nan")
    with pytest.raises(PurifyError) as ei:
        PurifyOp(32, 4, bad, None, dtype=C128)
    assert ei.value.status == -3
    bad[3, 1] = float("inf")
    with pytest.raises(PurifyError) as ei:
        PurifyOp(32, 4, bad, None, dtype=C128)
    assert ei.value.status == -3
    with pytest.raises(ValueError):
        PurifyOp(32, 4, uv, None, dtype=C64)                 # wrong real dtype
    op = PurifyOp(32, 4, uv, None, dtype=C128)
    with pytest.raises(ValueError):
        op.degrid(torch.zeros((16, 16), dtype=torch.complex128, device="cuda"))
    op.close()
    # complex64 layout: native-order y must be 16-byte aligned (it is streamed by bulk copies)
    uv32 = torch.rand((100, 2), dtype=torch.float32, device="cuda") * 8 - 4
    op = PurifyOp(32, 4, uv32, None, dtype=C64)
    buf = torch.zeros(op.M_native + 1, dtype=torch.complex64, device="cuda")
    with pytest.raises(PurifyError) as ei:
        op.grid(buf[1:], native=True)
    assert ei.value.status == -1
    op.grid(buf[:-1], native=True)
    op.close()


def test_degrid_bit_reproducible_and_host_create():
    from paper_1903_04502_b200 import C64, PurifyOp
    cfg, x, uv, w = synth.make_problem(2, M=50_000)
    x, uv, w = cast_problem(x, uv, w, "c64")
    op = make_op(cfg.n, 4, uv, w, "c64")
    a = host(op.degrid(dev(x)))
    b = host(op.degrid(dev(x)))
    assert np.array_equal(a, b)
    op2 = PurifyOp(cfg.n, 4, torch.from_numpy(uv), torch.from_numpy(w), dtype=C64)   # host uv / w
    assert np.array_equal(host(op2.degrid(dev(x))), a)
    op.close()
    op2.close()


def test_hot_cells_and_layer_straddling_batches():
    """Batched complex64 layout: a handful of cells with hundreds of visibilities (several full units per cell,
    layers of different widths, batches that straddle layer boundaries and hold one cell twice -> the flagged
    flush path) on top of a sparse background."""
    rng = synth.rng_for(4242, synth.STREAM_UV)
    n, J = 64, 6
    K = 2 * n
    counts = [700, 333, 257, 256, 129, 128, 127, 65, 64, 63]          # around multiples of the unit capacity
    hot = rng.integers(-20, 20, size=(len(counts), 2)).astype(np.float64)
    parts = [h + rng.uniform(0.0, 1.0, size=(c, 2)) for h, c in zip(hot, counts)]
    parts.append(rng.uniform(-K / 2, K / 2, size=(3000, 2)))
    uv = np.concatenate(parts)
    uv = uv[rng.permutation(len(uv))]
    w = rng.uniform(0.5, 1.5, size=len(uv))
    x = synth.random_complex((n, n), seed=9)
    info = run_all_checks(x, uv, w, J, "c64")
    assert info["layout"] == 1
    run_all_checks(x, uv, w, J, "c128")


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_operator_norm_power_method(dtype):
    """f2: purify_op_norm against the oracle's power method, same start vector, same fixed number of
    iterations (rel_tol = 0), and the stopping rule with a tolerance; also the all-ones default start."""
    cfg, x, uv, w = synth.make_problem(1, M=4000)
    w = synth.rng_for(11, synth.STREAM_W).uniform(0.5, 1.5, size=len(uv))
    x0 = synth.random_complex((cfg.n, cfg.n), seed=21, dtype=dtype)
    _, uvc, wc = cast_problem(x, uv, w, dtype)
    op = make_op(cfg.n, cfg.J, uvc, wc, dtype)
    tol = TOL[dtype]
    for iters in (1, 7):
        lam_ref, _ = oracle.power_method(x0, uvc, wc, cfg.n, cfg.J, max_iter=iters, rel_tol=0.0, idx_prec=idx_prec(dtype))
        lam, its = op.norm(dev(x0), max_iter=iters, rel_tol=0.0)
        assert its == iters and abs(lam - lam_ref) <= tol * lam_ref, (iters, lam, lam_ref)
    lam_ref, its_ref = oracle.power_method(None, uvc, wc, cfg.n, cfg.J, max_iter=200, rel_tol=1e-4, idx_prec=idx_prec(dtype))
    lam, its = op.norm(None, max_iter=200, rel_tol=1e-4)
    assert abs(its - its_ref) <= 1 and abs(lam - lam_ref) <= 2e-4 * lam_ref
    # Rayleigh check with the operator itself: ||Phi^dagger Phi x|| <= lambda ||x|| (up to the convergence gap)
    xr = synth.random_complex((cfg.n, cfg.n), seed=22, dtype=dtype)
    lam_conv, _ = op.norm(dev(x0), max_iter=300, rel_tol=1e-7)
    z = host(op.normal(dev(xr)))
    assert np.linalg.norm(z) <= lam_conv * np.linalg.norm(xr) * (1 + 1e-3)
    with pytest.raises(Exception):
        op.norm(dev(np.zeros((cfg.n, cfg.n), dtype=synth.complex_dtype(dtype))), max_iter=3)
    op.close()


@pytest.mark.parametrize("dtype,unfused", [("c128", False), ("c64", False), ("c64", True)])
@pytest.mark.parametrize("case", ["outside", "inside", "eps0"])
def test_admm_fidelity_step(dtype, unfused, case):
    """f1 (Algorithm 1 lines 3-6): purify_admm_fidelity_step against the oracle - g, the updated dual
    variable and the residual norm; native-order vectors, garbage in the padding entries of y and s."""
    cfg, x, uv, w = synth.make_problem(2, M=30000, J=6)
    x, uv, w = cast_problem(x, uv, w, dtype)
    M = len(uv)
    op = make_op(cfg.n, 6, uv, w, dtype, admm_unfused=unfused)     # c64 default: the fused kernels
    y = synth.random_complex((M,), seed=51, dtype=dtype)
    s = (synth.random_complex((M,), seed=52, dtype=dtype) * 0.25).astype(y.dtype)
    v = oracle.degrid(x, uv, w, 6, idx_prec=idx_prec(dtype))
    nd = float(np.linalg.norm(v + s - y))
    eps = {"outside": 0.4 * nd, "inside": 5.0 * nd, "eps0": 0.0}[case]
    g_ref, s_ref, _, nrm_ref = oracle.admm_fidelity_step(x, y, s, uv, w, cfg.n, 6, eps, 0.9, idx_prec=idx_prec(dtype))
    perm = host(op.permutation())
    valid = perm >= 0
    y_nat = np.full(len(perm), np.nan + 1j * np.nan, dtype=y.dtype)      # padding holds NaN: must be ignored
    s_nat = np.full(len(perm), np.nan + 1j * np.nan, dtype=y.dtype)
    y_nat[valid], s_nat[valid] = y[perm[valid]], s[perm[valid]]
    s_dev = dev(s_nat)
    g, nrm = op.admm_fidelity_step(dev(x), dev(y_nat), s_dev, eps, 0.9)
    tol = TOL[dtype]
    ctx = dict(n=cfg.n, J=6, M=M, dtype=dtype, case=case, unfused=unfused)
    assert abs(nrm - nrm_ref) <= ADMM_NORM_FACTOR * tol * nrm_ref
    compare("ADMM g", host(g), g_ref, tol, l2_factor=ADMM_FACTOR, **ctx)
    s_out = host(s_dev)
    compare("ADMM s_new", s_out[valid], s_ref[perm[valid]], tol, l2_factor=ADMM_FACTOR, **ctx)
    assert not np.any(s_out[~valid])
    op.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_workspace_reuse_host_call_then_unfused_admm(dtype):
    """One handle: a host-buffer call (allocates the caller-order staging vector, M entries) followed by the unfused ADMM
    step (needs M_native >= M entries of the same workspace): the workspace must grow, not overflow."""
    cfg, x, uv, w = synth.make_problem(2, M=30000, J=6)
    x, uv, w = cast_problem(x, uv, w, dtype)
    M = len(uv)
    op = make_op(cfg.n, 6, uv, w, dtype, admm_unfused=True)
    assert op.M_native > M
    yh = op.degrid_host(torch.from_numpy(x).pin_memory()).numpy()
    y = synth.random_complex((M,), seed=51, dtype=dtype)
    s = (synth.random_complex((M,), seed=52, dtype=dtype) * 0.25).astype(y.dtype)
    eps = 0.4 * float(np.linalg.norm(yh + s - y))
    g_ref, s_ref, _, nrm_ref = oracle.admm_fidelity_step(x, y, s, uv, w, cfg.n, 6, eps, 0.9, idx_prec=idx_prec(dtype))
    perm = host(op.permutation())
    valid = perm >= 0
    y_nat = np.zeros(len(perm), dtype=y.dtype)
    s_nat = np.zeros(len(perm), dtype=y.dtype)
    y_nat[valid], s_nat[valid] = y[perm[valid]], s[perm[valid]]
    guard = torch.full((1 << 16,), 7.0, dtype=torch.float32, device="cuda")      # something to trample on, if it did overflow
    g, nrm = op.admm_fidelity_step(dev(x), dev(y_nat), dev(s_nat), eps, 0.9)
    compare("ADMM g after a host call", host(g), g_ref, TOL[dtype], l2_factor=ADMM_FACTOR, n=cfg.n, J=6, M=M, dtype=dtype)
    assert float(guard.min()) == 7.0 and float(guard.max()) == 7.0
    assert np.array_equal(op.degrid_host(torch.from_numpy(x).pin_memory()).numpy(), yh)
    op.close()


@pytest.mark.parametrize("seed", list(range(10)))
def test_fuzz_batched_layout(seed):
    """Random small problems for the complex64 batched layout: random grid side, taps, M, and a (u, v) mixture of a
    uniform background, a few very hot cells (many full units -> layers, flagged batches, several items per band),
    exact integers / half-integers and far-out-of-period points.  Phi, Phi^dagger (native order) and the ADMM step
    against the oracle."""
    rng = synth.rng_for(9000 + seed, synth.STREAM_UV)
    n = int(rng.choice([16, 24, 34, 50, 64, 80]))
    J = int(rng.choice([4, 6, 8]))
    K = 2 * n
    parts = [rng.uniform(-K / 2, K / 2, size=(int(rng.integers(1, 6000)), 2))]
    for _ in range(int(rng.integers(0, 5))):
        c = rng.integers(-K // 2, K // 2, size=2).astype(np.float64)
        parts.append(c + rng.uniform(0, 1, size=(int(rng.integers(1, 3000)), 2)))
    parts.append(rng.integers(-K, K, size=(int(rng.integers(0, 40)), 2)).astype(np.float64) * 0.5)
    parts.append(rng.uniform(-5 * K, 5 * K, size=(int(rng.integers(0, 40)), 2)))
    uv = np.concatenate(parts)
    uv = uv[rng.permutation(len(uv))].astype(np.float32)
    w = rng.uniform(0.5, 1.5, size=len(uv)).astype(np.float32)
    x = synth.random_complex((n, n), seed=seed, dtype="c64")
    M = len(uv)
    op = make_op(n, J, uv, w, "c64")
    perm = host(op.permutation())
    valid = perm >= 0
    assert sorted(perm[valid].tolist()) == list(range(M))
    y_ref = oracle.degrid(x, uv, w, J, idx_prec=32)
    ctx = dict(n=n, J=J, M=M, dtype="c64", seed=seed)
    y_nat = host(op.degrid(dev(x), native=True))
    compare("fuzz Phi", y_nat[valid], y_ref[perm[valid]], 1e-5, **ctx)
    yv = synth.random_complex((M,), seed=100 + seed, dtype="c64")
    img_ref = oracle.grid(yv, uv, w, n, J, idx_prec=32)
    yv_nat = np.zeros(len(perm), dtype=np.complex64)
    yv_nat[valid] = yv[perm[valid]]
    compare("fuzz Phi^dagger", host(op.grid(dev(yv_nat), native=True)), img_ref, 1e-5, **ctx)
    s = (synth.random_complex((M,), seed=200 + seed, dtype="c64") * np.float32(0.3)).astype(np.complex64)
    eps = 0.5 * float(np.linalg.norm(y_ref + s - yv))
    g_ref, s_ref, _, nrm_ref = oracle.admm_fidelity_step(x, yv, s, uv, w, n, J, eps, 0.7, idx_prec=32)
    s_nat = np.zeros(len(perm), dtype=np.complex64)
    s_nat[valid] = s[perm[valid]]
    s_dev = dev(s_nat)
    g, nrm = op.admm_fidelity_step(dev(x), dev(yv_nat), s_dev, eps, 0.7)
    assert abs(nrm - nrm_ref) <= ADMM_NORM_FACTOR * 1e-5 * nrm_ref
    compare("fuzz ADMM g", host(g), g_ref, 1e-5, l2_factor=ADMM_FACTOR, **ctx)
    compare("fuzz ADMM s_new", host(s_dev)[valid], s_ref[perm[valid]], 1e-5, l2_factor=ADMM_FACTOR, **ctx)
    op.close()


def test_ubench_fma_forms():
    """The committed issue-rate probe (csrc/ubench.cuh) behind DESIGN.md 5's 'which roofline binds': it runs, and the
    ordering it is quoted for holds - a Horner step (one register pair read) issues at the FMA pipe's rate of one
    packed instruction per 2 cycles per sub-partition, the degridding row-pass form (two register pairs read) needs more."""
    from paper_1903_04502_b200 import UBENCH_FORMS, ubench_fma
    rates = [ubench_fma(f, 16)[0] for f in range(len(UBENCH_FORMS))]
    assert all(0.9 < r < 8.0 for r in rates), rates
    assert 1.9 <= rates[3] <= 2.2, rates                 # Horner form: pipe-bound
    assert rates[1] >= rates[3] * 1.05, rates            # row-pass form: operand-bound
    assert rates[4] <= rates[1], rates                   # gridding form is the cheaper of the two MAC forms


def test_canaries_around_every_output_buffer():
    """compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md), so out-of-bounds writes are looked for
    directly: every output of the C ABI is a slice in the MIDDLE of a larger allocation whose flanks hold a canary
    pattern; after the call the flanks must be untouched.  Sizes chosen ragged (M and M_native not multiples of 32 x
    the chunk sizes, K not a power of two) so that the last chunk / item / batch / band of every kernel is partial."""
    from paper_1903_04502_b200 import C64, C128, PurifyOp
    GUARD = 4096

    def guarded(count, dtype):
        buf = torch.full((count + 2 * GUARD,), complex(7.25, -3.5), dtype=dtype, device="cuda")
        return buf, buf[GUARD:GUARD + count]

    def intact(buf, count):
        return bool((buf[:GUARD] == complex(7.25, -3.5)).all()) and bool((buf[GUARD + count:] == complex(7.25, -3.5)).all())

    rng = synth.rng_for(31337, synth.STREAM_UV)
    for dtype, dt, cdt in (("c64", C64, torch.complex64), ("c128", C128, torch.complex128)):
        for n, J, M in ((50, 6, 7001), (34, 4, 333), (64, 8, 5003)):
            K = 2 * n
            uv = np.concatenate([rng.uniform(-K / 2, K / 2, size=(M - 300, 2)), 3.0 + rng.uniform(0, 1, size=(300, 2))])
            uv = uv.astype(synth.real_dtype(dtype))
            w = rng.uniform(0.5, 1.5, size=M).astype(synth.real_dtype(dtype))
            op = PurifyOp(n, J, dev(uv), dev(w), dtype=dt)
            x = dev(synth.random_complex((n, n), seed=1, dtype=dtype))
            by, y = guarded(M, cdt)
            bn, yn = guarded(op.M_native, cdt)
            bx, xo = guarded(n * n, cdt)
            xo2 = xo.view(n, n)
            op.degrid(x, y)
            op.degrid(x, yn, native=True)
            op.grid(y, xo2)
            op.grid(yn, xo2, native=True)
            op.normal(x, xo2)
            op.normal(x, xo2)
            op.permute_to_native(y, yn)
            op.permute_from_native(yn, y)
            bs, s = guarded(op.M_native, cdt)
            s.zero_()
            op.admm_fidelity_step(x, yn, s, 0.5, 0.9, xo2)
            op.normal_dist(x, xo2, allreduce=lambda band: None, bands=7)
            torch.cuda.synchronize()
            assert intact(by, M) and intact(bn, op.M_native) and intact(bx, n * n) and intact(bs, op.M_native), (dtype, n, J, M)
            op.close()


def test_gridding_repeatable_under_stress_on_hot_cells():
    """The accumulator flush of the gridding kernel is the one place where lanes of a warp write overlapping
    shared-memory footprints; the steps are ordered by __syncwarp() (batched.cuh).  200 repetitions on the hot-cell
    input (flagged and unflagged batches, several items per band): every repetition within the tolerance of the
    oracle, and all repetitions within rounding of one another (a lost update would be an O(1) difference in a cell)."""
    rng = synth.rng_for(4242, synth.STREAM_UV)
    n, J = 64, 6
    K = 2 * n
    counts = [700, 333, 257, 256, 129, 128, 127, 65, 64, 63]
    hot = rng.integers(-20, 20, size=(len(counts), 2)).astype(np.float64)
    parts = [h + rng.uniform(0.0, 1.0, size=(c, 2)) for h, c in zip(hot, counts)]
    parts.append(rng.uniform(-K / 2, K / 2, size=(6000, 2)))
    uv = np.concatenate(parts).astype(np.float32)
    w = rng.uniform(0.5, 1.5, size=len(uv)).astype(np.float32)
    yv = synth.random_complex((len(uv),), seed=5, dtype="c64")
    op = make_op(n, J, uv, w, "c64")
    ref = oracle.grid_to_grid(yv, uv, w, K, J, idx_prec=32)
    yd = dev(yv)
    first = op.stage_gridded(yd)
    compare("stress: gridded", host(first), ref, 1e-5, n=n, J=J, M=len(uv), dtype="c64")
    scale = float(first.abs().max())
    worst = 0.0
    for _ in range(200):
        worst = max(worst, float((op.stage_gridded(yd) - first).abs().max()) / scale)
    assert worst <= 2e-6, worst                              # reduction order varies (atomics at L2): rounding only
    op.close()


@pytest.mark.parametrize("dtype", ["c64", "c128"])
def test_routed_permutation_is_the_permutation(dtype):
    """From 2^24 visibilities on the caller-order entry points permute in three routed passes (blocks of 8192 / 4096
    elements permuted in shared memory, runs written to coarse buckets, then to caller tiles of 4096, then inside the
    tile; kernels.cuh).  Index work: bit-exact against purify_op_permutation, both directions, at a ragged size (last
    block, last coarse bucket and last caller tile partial), with NaN canaries around the outputs."""
    from paper_1903_04502_b200 import C64, C128, PurifyOp
    M = (1 << 24) + 1234
    rng = np.random.default_rng(77)
    K = 512
    uv = rng.normal(0.0, K / 6, size=(M, 2)).clip(-K / 2 + 9, K / 2 - 9).astype(synth.real_dtype(dtype))
    op = PurifyOp(256, 4, torch.from_numpy(uv).cuda(), None, dtype=C64 if dtype == "c64" else C128)
    perm = op.permutation().cpu().numpy()
    Mn = op.M_native
    cd = synth.complex_dtype(dtype)
    real = perm >= 0
    assert real.sum() == M and np.array_equal(np.sort(perm[real]), np.arange(M))
    # native -> caller
    v_nat = synth.random_complex((Mn,), seed=5, dtype=dtype)
    buf = torch.full((M + 64,), complex(float("nan"), float("nan")), dtype=torch.from_numpy(v_nat).dtype, device="cuda")
    out = op.permute_from_native(torch.from_numpy(v_nat).cuda(), out=buf[32:32 + M])
    ref = np.empty(M, dtype=cd)
    ref[perm[real]] = v_nat[real]
    assert np.array_equal(out.cpu().numpy().view(np.uint8), ref.view(np.uint8))
    flank = torch.cat([buf[:32], buf[32 + M:]]).cpu().numpy()
    assert np.isnan(flank.real).all() and np.isnan(flank.imag).all()
    # caller -> native (padding slots become 0)
    v_call = synth.random_complex((M,), seed=6, dtype=dtype)
    buf2 = torch.full((Mn + 64,), complex(float("nan"), float("nan")), dtype=buf.dtype, device="cuda")
    out2 = op.permute_to_native(torch.from_numpy(v_call).cuda(), out=buf2[32:32 + Mn])
    ref2 = np.zeros(Mn, dtype=cd)
    ref2[real] = v_call[perm[real]]
    assert np.array_equal(out2.cpu().numpy().view(np.uint8), ref2.view(np.uint8))
    flank2 = torch.cat([buf2[:32], buf2[32 + Mn:]]).cpu().numpy()
    assert np.isnan(flank2.real).all() and np.isnan(flank2.imag).all()
    op.close()
