"""Pins of the CPU oracle against things that are NOT the oracle: the paper's printed
numbers, closed forms, scipy / numpy library routines, and a brute-force NUDFT written
here in numpy straight from PAPER.md Eq. (1).  (-m "not gpu")"""
import math
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.special

import oracle
from inputs import synth

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "constants.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])


def rel_l2(a, b):
    return float(np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b)))


def nudft(x, uv, w=None):
    """Brute force of PAPER.md Eq. (1) discretised with a == 1:
    y_k = w_k sum_{py,px} x[py,px] exp(-2 pi i (u_k p^x + v_k p^y) / K), p^ = p - n/2.
    Written with explicit phase matrices; no FFT, no kernel, nothing from oracle/."""
    n = x.shape[0]
    K = 2 * n
    p = np.arange(n) - n // 2
    y = np.empty(len(uv), dtype=np.complex128)
    for s in range(0, len(uv), 2048):
        u = uv[s:s + 2048, 0].astype(np.float64)
        v = uv[s:s + 2048, 1].astype(np.float64)
        Eu = np.exp(-2j * np.pi * np.outer(u, p) / K)       # [k, px]
        Ev = np.exp(-2j * np.pi * np.outer(v, p) / K)       # [k, py]
        y[s:s + 2048] = np.einsum("ky,yx,kx->k", Ev, x.astype(np.complex128), Eu, optimize=True)
    return y if w is None else y * w


# ------------------------------------------------------------------ kernel pieces
@pytest.mark.parametrize("J,key", [(4, "i0_beta_J4"), (6, "i0_beta_J6"), (8, "i0_beta_J8")])
def test_i0_series_vs_scipy_and_golden(J, key):
    beta = 2.34 * J
    assert oracle.i0(beta) == pytest.approx(GOLD[key], rel=1e-13)
    for z in [0.0, 1e-3, 0.5, 1.0, 3.3, beta / 2, beta]:
        assert oracle.i0(z) == pytest.approx(float(scipy.special.i0(z)), rel=2e-15)


@pytest.mark.parametrize("J", [4, 6, 8])
def test_kb_special_values(J):
    beta = 2.34 * J
    assert oracle.kb(0.0, J) == pytest.approx(1.0, abs=1e-15)
    assert oracle.kb(J / 2, J) == pytest.approx(1.0 / scipy.special.i0(beta), rel=1e-13)
    assert oracle.kb(J / 2 + 1e-9, J) == 0.0
    d = np.arange(-20, 21) * (J / 40.0)
    g = oracle.kb(d, J)
    assert np.allclose(g, g[::-1], rtol=0, atol=1e-15)       # even
    ref = scipy.special.i0(beta * np.sqrt(np.maximum(0, 1 - (2 * d / J) ** 2))) / scipy.special.i0(beta)
    assert np.allclose(g, ref, rtol=1e-13)
    assert np.all(np.diff(g[20:]) < 0)                      # decreasing away from 0


@pytest.mark.parametrize("J,key,flat", [(4, "ghat0_J4", 4e-4), (6, "ghat0_J6", 6e-6), (8, "ghat0_J8", 1e-7)])
def test_kernel_sum_closed_form(J, key, flat):
    """Poisson: sum_c g(delta - c) ~ g^(0) = J sinh(beta)/(beta I0(beta)), flat in delta."""
    beta = 2.34 * J
    closed = J * math.sinh(beta) / (beta * float(scipy.special.i0(beta)))
    assert closed == pytest.approx(GOLD[key], rel=1e-6)
    assert float(oracle.kb_ghat(0.0, J)) == pytest.approx(closed, rel=1e-13)
    for delta in np.linspace(0, 1, 11):
        taps = np.arange(-J, J + 1)
        s = float(np.sum(oracle.kb(delta - taps, J)))
        assert abs(s - closed) <= 1.5 * flat * closed


@pytest.mark.parametrize("J", [4, 6, 8])
def test_ghat_vs_quadrature(J):
    """g^(xi) = int g(d) cos(2 pi xi d) dd, checked by scipy quadrature of scipy's I0."""
    beta = 2.34 * J
    i0b = float(scipy.special.i0(beta))

    def g(d):
        return float(scipy.special.i0(beta * math.sqrt(max(0.0, 1 - (2 * d / J) ** 2)))) / i0b

    for xi in [0.0, 0.05, 0.125, 0.2, 0.25]:
        val, _ = scipy.integrate.quad(lambda d: g(d) * math.cos(2 * math.pi * xi * d), -J / 2, J / 2,
                                      epsabs=1e-13, epsrel=1e-13, limit=200)
        assert float(oracle.kb_ghat(xi, J)) == pytest.approx(val, rel=1e-9)


@pytest.mark.parametrize("J,lo,hi", [(4, 0.619, 1.004), (6, 0.503, 1.070), (8, 0.435, 1.212)])
def test_correction_vector(J, lo, hi):
    n = 128
    s = oracle.correction(n, J)
    p = np.arange(n) - n // 2
    assert np.allclose(s, 1.0 / oracle.kb_ghat(p / (2 * n), J), rtol=1e-14)
    assert s[n // 2] == pytest.approx(1.0 / float(oracle.kb_ghat(0.0, J)))
    assert np.allclose(s[1:], s[1:][::-1])                   # symmetric about the centre pixel
    # range printed in SURVEY.md O2 (normalised so that s[centre] ~ 1/g^(0))
    sn = s * float(oracle.kb_ghat(0.0, J))
    assert sn.min() == pytest.approx(1.0, abs=1e-12)
    assert s.max() / s.min() > 1.2


# ------------------------------------------------------------------ FFT
@pytest.mark.parametrize("K", [8, 32, 64, 12])
@pytest.mark.parametrize("sign", [-1, 1])
def test_fft_vs_numpy_and_direct(K, sign):
    a = synth.random_complex((K, K), seed=7, stream=K + sign)
    got = oracle.fft2(a, sign)
    ref = np.fft.fft2(a) if sign < 0 else np.fft.ifft2(a) * K * K
    assert rel_l2(got, ref) < 1e-14
    assert rel_l2(oracle.dft2_direct(a, sign), ref) < 1e-13
    # Parseval, unnormalised: ||B||^2 = K^2 ||b||^2
    assert np.linalg.norm(got) ** 2 == pytest.approx(K * K * np.linalg.norm(a) ** 2, rel=1e-13)


def test_fft_impulse_and_shift():
    K = 16
    a = np.zeros((K, K), complex)
    a[3, 5] = 1.0       # row (y) 3, col (x) 5
    B = oracle.fft2(a, -1)
    ky, kx = np.mgrid[0:K, 0:K]
    assert np.allclose(B, np.exp(-2j * np.pi * (3 * ky + 5 * kx) / K), atol=1e-14)


# ------------------------------------------------------------------ Phi vs brute-force NUDFT (Eq. 1)
@pytest.fixture(scope="module")
def tiny():
    cfg, x, uv, w = synth.make_problem(1)
    return cfg, x, uv, w


@pytest.mark.parametrize("J,tol_bj,tol_probe", [(4, 5e-3, 6e-4), (6, 1e-4, 7e-6), (8, 1e-5, 7e-8)])
def test_phi_vs_nudft_tiny(tiny, J, tol_bj, tol_probe):
    """BASELINE.json north_star: rel-L2 <= 5e-3 at J=4, <= 1e-5 at J=8 (oversample 2).
    tol_probe = 2x the error the proposed reading is known to reach."""
    cfg, x, uv, w = tiny
    y = oracle.degrid(x, uv, None, J)
    ref = nudft(x, uv)
    err = rel_l2(y, ref)
    assert err <= tol_bj
    assert err <= tol_probe


def test_phi_vs_nudft_noise_image_with_wrap():
    """White-noise image (every pixel, incl. image edges), uv over the FULL +-K/2 range
    including exact edges: pins R8 (periodic wrap) and the correction at all pixels."""
    n, J, K = 32, 4, 64
    x = synth.random_complex((n, n), seed=11)
    rng = synth.rng_for(11, 99)
    uv = rng.uniform(-K / 2, K / 2, size=(600, 2))
    uv[0] = (-K / 2, -K / 2)
    uv[1] = (K / 2 - 1e-9, K / 2 - 1e-9)
    uv[2] = (K / 2 - 1e-9, 0.25)
    uv[3] = (-K / 2 + 0.5, K / 2 - 0.5)
    uv[4] = (K / 2 + 3.25, -K / 2 - 7.5)        # outside the period: taken mod K
    w = rng.uniform(0.5, 1.5, size=600)
    y = oracle.degrid(x, uv, w, J)
    ref = nudft(x, uv, w)
    assert rel_l2(y, ref) < 1.5e-3
    edge = (np.abs(uv).max(axis=1) > K / 2 - J)
    assert edge.sum() > 20
    assert rel_l2(y[edge], ref[edge]) < 2e-3
    assert rel_l2(y[:5], ref[:5]) < 2e-3
    # J = 8 on the same inputs
    assert rel_l2(oracle.degrid(x, uv, w, 8), ref) < 5e-7


@pytest.mark.parametrize("J,eps", [(4, 8.3e-4), (6, 8.4e-6), (8, 1.2e-7)])
def test_centred_point_source(tiny, J, eps):
    """R6: unit delta at pixel (n/2, n/2) -> y_k = w_k (1 + e), |e| small (kernel accuracy)."""
    cfg, _, uv, _ = tiny
    x = np.zeros((cfg.n, cfg.n), complex)
    x[cfg.n // 2, cfg.n // 2] = 1.0
    w = synth.rng_for(3, 3).uniform(0.5, 1.5, size=len(uv))
    y = oracle.degrid(x, uv, w, J)
    assert np.max(np.abs(y / w - 1.0)) <= 1.3 * eps


def test_off_centre_point_source_axes_and_sign(tiny):
    """Delta of amplitude A at (py, px): y_k = A exp(-2 pi i (u p^x + v p^y)/K).
    Asymmetric offsets pin px<->u, py<->v and the sign of the exponent."""
    cfg, _, uv, _ = tiny
    n, K = cfg.n, cfg.K
    x = np.zeros((n, n), complex)
    py, px, A = n // 2 + 17, n // 2 - 5, 0.7 - 0.2j
    x[py, px] = A
    y = oracle.degrid(x, uv, None, 4)
    ref = A * np.exp(-2j * np.pi * (uv[:, 0] * (px - n // 2) + uv[:, 1] * (py - n // 2)) / K)
    assert rel_l2(y, ref) < 1e-3
    wrong_axes = A * np.exp(-2j * np.pi * (uv[:, 1] * (px - n // 2) + uv[:, 0] * (py - n // 2)) / K)
    assert rel_l2(y, wrong_axes) > 0.5
    assert rel_l2(y, np.conj(ref / A) * A) > 0.5


# ------------------------------------------------------------------ adjoint
@pytest.mark.parametrize("J,mode", [(4, "analytic"), (6, "analytic"), (8, "analytic"), (4, "table")])
def test_adjoint_identity(J, mode):
    """<Phi x, y> = <x, Phi^dagger y> to 1e-12 relative (north_star); R5: fails by K^2 if
    F^dagger carried a 1/K^2."""
    n, M = 64, 3000
    K = 2 * n
    x = synth.random_complex((n, n), seed=21)
    yv = synth.random_complex((M,), seed=22)
    rng = synth.rng_for(23, 0)
    uv = rng.uniform(-K / 2, K / 2, size=(M, 2))         # includes wrapped taps
    # R7: integer and half-integer coordinates (ties of the tap rule), alone and mixed with continuous ones
    uv[:200] = rng.integers(-K // 2, K // 2, size=(200, 2))
    uv[200:400] = rng.integers(-K, K, size=(200, 2)) * 0.5
    uv[400:500, 0] = rng.integers(-K // 2, K // 2, size=100)
    w = rng.uniform(0.5, 1.5, size=M)
    Px = oracle.degrid(x, uv, w, J, mode=mode)
    Pty = oracle.grid(yv, uv, w, n, J, mode=mode)
    lhs = np.vdot(Px, yv)
    rhs = np.vdot(x, Pty)
    assert abs(lhs - rhs) / (np.linalg.norm(Px) * np.linalg.norm(yv)) < 1e-12


def test_single_visibility_adjoint_closed_form():
    """Phi^dagger e_k ~ exp(+2 pi i (u p^x + v p^y)/K) (adjoint of the NUDFT row)."""
    n, J = 64, 4
    K = 2 * n
    uv = np.array([[13.37, -21.6]])
    img = oracle.grid(np.array([1.0 + 0j]), uv, None, n, J)
    p = np.arange(n) - n // 2
    ref = np.exp(2j * np.pi * (uv[0, 0] * p[None, :] + uv[0, 1] * p[:, None]) / K)
    assert rel_l2(img, ref) < 1.5e-3


def test_grid_footprint_and_tie_break():
    """R7 (convention, unpinned by the paper): taps are the integers in (u-J/2, u+J/2];
    at integer u the tap at distance +J/2 (below) is dropped, the one at -J/2 kept."""
    K, J = 32, 4
    for u, v, cols, rows in [(5.25, -3.5, [4, 5, 6, 7], [-5, -4, -3, -2]),
                             (6.0, 2.0, [5, 6, 7, 8], [1, 2, 3, 4])]:
        Bp = oracle.grid_to_grid(np.array([1.0 + 0j]), np.array([[u, v]]), None, K, J)
        nzr, nzc = np.nonzero(np.abs(Bp) > 0)
        assert sorted(set(nzc.tolist())) == sorted([c % K for c in cols])
        assert sorted(set(nzr.tolist())) == sorted([r % K for r in rows])
        # separable weights g(v - cy) g(u - cx)
        for r in rows:
            for c in cols:
                exp = float(oracle.kb(v - r, J)) * float(oracle.kb(u - c, J))
                assert Bp[r % K, c % K] == pytest.approx(exp, rel=1e-13)
    # kept tie tap has weight 1/I0(beta), not zero
    Bp = oracle.grid_to_grid(np.array([1.0 + 0j]), np.array([[6.0, 2.0]]), None, K, J)
    assert abs(Bp[2, 8]) == pytest.approx(1.0 / scipy.special.i0(2.34 * J), rel=1e-12)


@pytest.mark.parametrize("J", [4, 6, 8])
def test_degrid_footprint_and_tie_break_on_one_hot_grid(J):
    """R7 for W G on its own (not through G^dagger): with a one-hot Fourier grid B = e_(r,c) the degridded value is
    g(v - r) g(u - c) when (r, c) is one of the J x J taps - the integers in (v - J/2, v + J/2] x (u - J/2, u + J/2] -
    and 0 otherwise.  Integer, half-integer and generic coordinates; the tap set is written out here from the
    definition, the weights from scipy's I0."""
    K = 32
    beta = 2.34 * J

    def g(d):
        return float(scipy.special.i0(beta * math.sqrt(max(0.0, 1 - (2 * d / J) ** 2))) / scipy.special.i0(beta)) if abs(d) <= J / 2 else 0.0

    for u, v in [(5.0, -3.0), (6.5, 2.0), (-2.0, 7.5), (0.0, 0.0), (3.25, -4.75), (-7.5, -7.5)]:
        taps_x = [c for c in range(-K, K) if u - J / 2 < c <= u + J / 2]
        taps_y = [r for r in range(-K, K) if v - J / 2 < r <= v + J / 2]
        assert len(taps_x) == J and len(taps_y) == J
        for r in range(int(math.floor(v)) - J, int(math.floor(v)) + J + 1):
            for c in range(int(math.floor(u)) - J, int(math.floor(u)) + J + 1):
                B = np.zeros((K, K), complex)
                B[r % K, c % K] = 1.0
                y = oracle.degrid_from_grid(B, np.array([[u, v]]), None, J)[0]
                if r in taps_y and c in taps_x:
                    assert y == pytest.approx(g(v - r) * g(u - c), rel=1e-12, abs=1e-300), (u, v, r, c)
                else:
                    assert y == 0.0, (u, v, r, c)
    # the kept tie tap (distance exactly -J/2 from an integer u) carries 1/I0(beta), the dropped one (+J/2) nothing
    B = np.zeros((K, K), complex)
    B[2 % K, (6 + J // 2) % K] = 1.0
    assert oracle.degrid_from_grid(B, np.array([[6.0, 2.0]]), None, J)[0].real == pytest.approx(1.0 / scipy.special.i0(beta), rel=1e-12)
    B[:] = 0
    B[2 % K, (6 - J // 2) % K] = 1.0
    assert oracle.degrid_from_grid(B, np.array([[6.0, 2.0]]), None, J)[0] == 0.0


def test_stage_consistency_and_linearity(tiny):
    """Phi == W G . F . (Z S) composed from the stage entry points; Phi is linear."""
    cfg, x, uv, w = tiny
    J = 4
    uv, w = uv[:2000], synth.rng_for(5, 5).uniform(0.5, 1.5, size=2000)
    y = oracle.degrid(x, uv, w, J)
    B = oracle.fft2(oracle.pad(x, J), -1)
    assert rel_l2(oracle.degrid_from_grid(B, uv, w, J), y) < 1e-15
    x2 = synth.random_complex(x.shape, seed=31)
    assert rel_l2(oracle.degrid(x + 2j * x2, uv, w, J), y + 2j * oracle.degrid(x2, uv, w, J)) < 1e-13
    yv = synth.random_complex((2000,), seed=32)
    img = oracle.grid(yv, uv, w, cfg.n, J)
    img2 = oracle.crop(oracle.fft2(oracle.grid_to_grid(yv, uv, w, cfg.K, J), +1), J)
    assert rel_l2(img2, img) < 1e-15
    # permutation invariance of the gridded image / permutation equivariance of y
    perm = synth.shuffle_order(2000, 9)
    assert np.array_equal(oracle.degrid(x, uv[perm], w[perm], J), y[perm])
    assert rel_l2(oracle.grid(yv[perm], uv[perm], w[perm], cfg.n, J), img) < 1e-13


def test_pad_layout():
    """R6: centre pixel -> grid index 0; p^ mod K placement; zeros elsewhere."""
    n, J = 8, 4
    x = synth.random_complex((n, n), seed=41)
    b = oracle.pad(x, J)
    s = oracle.correction(n, J)
    K = 2 * n
    assert b[0, 0] == pytest.approx(s[n // 2] ** 2 * x[n // 2, n // 2])
    assert b[K - 1, 1] == pytest.approx(s[n // 2 - 1] * s[n // 2 + 1] * x[n // 2 - 1, n // 2 + 1])
    assert np.count_nonzero(b) == n * n
    assert np.all(b[n // 2:K - n // 2, :] == 0) and np.all(b[:, n // 2:K - n // 2] == 0)
    # crop is its adjoint: <pad x, c> = <x, crop c>
    c = synth.random_complex((K, K), seed=42)
    assert np.vdot(b, c) == pytest.approx(np.vdot(x, oracle.crop(c, J)), rel=1e-13)


# ------------------------------------------------------------------ table mode
def test_table_paper_statements():
    """2e5 samples/pixel -> zeroth-order lookup accurate to 1e-5; J=4 needs
    4e5 samples (table on [0, J/2], even symmetry).  Also the 25.6 GB / 48 B statements."""
    J, R = 4, int(GOLD["table_density_paper"])
    T = oracle.table(J, R)
    assert len(T) - 2 == int(GOLD["table_samples_J4_paper"])
    assert T[0] == 1.0 and T[-1] == 0.0
    rng = synth.rng_for(51, 0)
    d = rng.uniform(-J / 2, J / 2, size=4000)
    idx = np.floor(np.abs(d) * R + 0.5).astype(int)
    exact = oracle.kb(d, J)
    assert np.max(np.abs(T[idx] - exact)) <= GOLD["table_accuracy_paper"]
    # the operator's own lookup follows the same rule, for + and - distances
    for dd in d[:50]:
        c = 7
        assert oracle.kernel_weight(c + dd, c, J, "table", R, 64) == T[int(math.floor(abs((c + dd) - c) * R + 0.5))]
    # memory statements
    assert J * J * 1e8 * 16 == GOLD["stored_G_bytes_J4_M1e8"]
    assert 16 + 16 + 8 + 8 == GOLD["bytes_per_visibility_paper"]


def test_table_mode_operator_close_to_analytic():
    """R11: at R = 4096 the table-mode operator differs from the analytic one by
    ~4e-5..1e-4 rel-L2 (= max|g'|/(2R) scale), so parity must use the same mode."""
    cfg, x, uv, w = synth.make_problem(2, M=20000)
    ya = oracle.degrid(x, uv, w, 4, "analytic")
    yt = oracle.degrid(x, uv, w, 4, "table", 4096)
    e = rel_l2(yt, ya)
    assert 1e-6 < e < 2e-4
    assert rel_l2(oracle.degrid(x, uv, w, 4, "table", 200000), ya) < 4e-6


def test_table_index_precision_flag():
    """idx_prec=32 decides the lookup index in fp32 (C64 problems); for f32-representable
    u away from 0 the fp32 subtraction is exact and both precisions agree."""
    J, R = 4, 4096
    u32 = np.float32(1234.5678)
    for c in range(1233, 1237):
        assert oracle.kernel_weight(float(u32), c, J, "table", R, 32) == \
            oracle.kernel_weight(float(u32), c, J, "table", R, 64)


def test_table_index_fp32_branch_vs_exact_arithmetic():
    """R11, idx_prec = 32 (the branch the oracle takes for complex64 problems so that both sides decide the index in
    the storage precision).  Where every fp32 step is exact - u an f32 number with |u| >= 1, c an integer within J/2 + 1
    of it, R a power of two - the fp32 index must equal the index computed in exact rational arithmetic, and hence the
    fp64 branch; 1e5 random f32 coordinates over the range of config 5 (K = 8192).  At a density that is not a power of
    two (R = 1000) the fp32 product rounds: the two precisions may then differ by one sample on a small fraction of
    the inputs (reported in DESIGN.md R11) and never by more."""
    from fractions import Fraction
    rng = synth.rng_for(77, synth.STREAM_TEST)
    n = 100_000
    mag = np.exp(rng.uniform(0.0, math.log(4090.0), size=n))
    u = (mag * rng.choice([-1.0, 1.0], size=n)).astype(np.float32)
    u[np.abs(u) < 1.0] = np.float32(1.0)
    u[:1000] = np.round(u[:1000])                        # exact integers
    u[1000:2000] = np.round(u[1000:2000] * 2) / 2        # half-integers
    c = np.floor(u).astype(np.int64) + rng.integers(-3, 5, size=n)
    u64 = u.astype(np.float64)
    i32 = oracle.table_index(u64, c, 4096, 32)
    i64 = oracle.table_index(u64, c, 4096, 64)
    assert np.array_equal(i32, i64)
    for k in rng.integers(0, n, size=300).tolist() + list(range(0, 2000, 40)):       # exact arithmetic on a sample
        d = abs(Fraction(float(u[k])) - int(c[k]))
        assert int(i32[k]) == math.floor(d * 4096 + Fraction(1, 2)), (float(u[k]), int(c[k]))
    # numpy's own float64 evaluation of the same rule agrees everywhere
    assert np.array_equal(i64, np.floor(np.abs(u64 - c) * 4096 + 0.5).astype(np.int64))
    # not a power of two: |index difference| <= 1, on a small fraction of the inputs
    j32 = oracle.table_index(u64, c, 1000, 32)
    j64 = oracle.table_index(u64, c, 1000, 64)
    diff = np.abs(j32 - j64)
    assert diff.max() <= 1
    rate = float((diff > 0).mean())
    assert rate < 2e-3, rate
    # small |u| (< 1): the subtraction u - c itself rounds in fp32; still at most one sample apart at R = 4096
    us = rng.uniform(-1.0, 1.0, size=20000).astype(np.float32).astype(np.float64)
    cs = rng.integers(-3, 4, size=20000)
    assert np.abs(oracle.table_index(us, cs, 4096, 32) - oracle.table_index(us, cs, 4096, 64)).max() <= 1


def test_power_method_vs_dense_eigensolver():
    """f2: the oracle's power method against numpy's dense eigen-solver on a tiny operator whose
    matrix is assembled column by column (Phi applied to the n^2 basis images)."""
    n, J, M = 8, 4, 60
    rng = synth.rng_for(31, synth.STREAM_UV)
    uv = rng.uniform(-n + 0.01, n - 0.01, size=(M, 2))
    w = rng.uniform(0.5, 1.5, size=M)
    Phi = np.empty((M, n * n), dtype=np.complex128)
    for p in range(n * n):
        e = np.zeros(n * n, dtype=np.complex128)
        e[p] = 1.0
        Phi[:, p] = oracle.degrid(e.reshape(n, n), uv, w, J)
    lam_true = float(np.linalg.eigvalsh(Phi.conj().T @ Phi)[-1])
    assert abs(np.linalg.norm(Phi, 2) ** 2 - lam_true) <= 1e-10 * lam_true
    x0 = synth.random_complex((n, n), seed=3)
    lam, its = oracle.power_method(x0, uv, w, n, J, max_iter=3000, rel_tol=1e-13)
    assert abs(lam - lam_true) <= 1e-7 * lam_true, (lam, lam_true, its)
    # the iterates increase monotonically towards the eigenvalue (Phi^dagger Phi is positive semi-definite)
    lam5, _ = oracle.power_method(x0, uv, w, n, J, max_iter=5, rel_tol=0.0)
    lam50, _ = oracle.power_method(x0, uv, w, n, J, max_iter=50, rel_tol=0.0)
    assert lam5 <= lam50 * (1 + 1e-12) <= lam_true * (1 + 1e-9)
    # scaling: Phi -> 2 Phi (weights doubled) multiplies the eigenvalue by 4
    lam2, _ = oracle.power_method(x0, uv, 2 * w, n, J, max_iter=3000, rel_tol=1e-13)
    assert abs(lam2 - 4 * lam_true) <= 1e-6 * lam_true


def test_admm_fidelity_step_closed_forms(tiny):
    """f1: Algorithm 1 lines 3-6 with the projection of Eq. (23) - special cases
    with closed forms, and the defining properties of the projection."""
    cfg, x, uv, w = tiny
    M = 1500
    uv, w = uv[:M], w[:M] * 0 + synth.rng_for(5, synth.STREAM_W).uniform(0.5, 1.5, size=M)
    y = synth.random_complex((M,), seed=41)
    s = synth.random_complex((M,), seed=42) * 0.3
    v = oracle.degrid(x, uv, w, cfg.J)
    d = v + s - y
    nd = np.linalg.norm(d)
    # (i) inside the ball (huge epsilon): r = v + s, s_new = (1 - varrho) s, g = -varrho Phi^dagger s
    g, s_new, r, nrm = oracle.admm_fidelity_step(x, y, s, uv, w, cfg.n, cfg.J, epsilon=10 * nd, varrho=0.9)
    assert abs(nrm - nd) <= 1e-12 * nd
    assert np.allclose(r, v + s, rtol=0, atol=1e-13) and np.allclose(s_new, 0.1 * s, rtol=0, atol=1e-13)
    g_ref = -0.9 * oracle.grid(s, uv, w, cfg.n, cfg.J)
    assert np.linalg.norm(g - g_ref) <= 1e-12 * np.linalg.norm(g_ref)
    # (ii) epsilon = 0: r = y, s_new = s + varrho (v - y), g = Phi^dagger (v - y + s_new)
    g, s_new, r, _ = oracle.admm_fidelity_step(x, y, s, uv, w, cfg.n, cfg.J, epsilon=0.0, varrho=0.5)
    assert np.allclose(r, y, rtol=0, atol=1e-13) and np.allclose(s_new, s + 0.5 * (v - y), rtol=0, atol=1e-13)
    g_ref = oracle.grid(v - y + s_new, uv, w, cfg.n, cfg.J)
    assert np.linalg.norm(g - g_ref) <= 1e-12 * np.linalg.norm(g_ref)
    # (iii) outside the ball: r lies ON the sphere, on the segment from y to v + s, and is the nearest point of the ball
    eps = 0.37 * nd
    g, s_new, r, _ = oracle.admm_fidelity_step(x, y, s, uv, w, cfg.n, cfg.J, epsilon=eps, varrho=0.9)
    assert abs(np.linalg.norm(r - y) - eps) <= 1e-12 * eps
    t = np.vdot(d, r - y) / np.vdot(d, d)
    assert abs(t.imag) <= 1e-13 and abs(t.real - 0.37) <= 1e-12
    rng = synth.rng_for(77, synth.STREAM_TEST)
    for _ in range(20):                                   # random points of the ball are never closer to v + s
        q = synth.random_complex((M,), seed=int(rng.integers(1 << 30)))
        q = y + q / np.linalg.norm(q) * eps * rng.uniform(0, 1)
        assert np.linalg.norm(q - (v + s)) >= np.linalg.norm(r - (v + s)) * (1 - 1e-12)
    assert np.allclose(s_new, s + 0.9 * (v - r), rtol=0, atol=1e-13)
