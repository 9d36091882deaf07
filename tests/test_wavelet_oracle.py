"""Pins of the wavelet / DUALFB oracle (oracle/wavelets.py, f4) against things that are not the oracle: closed forms,
the defining properties of an orthonormal Daubechies filter bank, hand-computed values.  -m "not gpu" """
import math

import numpy as np
import pytest

from inputs import synth
from oracle import wavelets as W


def test_haar_and_db2_closed_forms():
    assert np.allclose(W.daubechies_lowpass(1), [1 / math.sqrt(2), 1 / math.sqrt(2)], rtol=0, atol=1e-15)
    s3 = math.sqrt(3.0)
    db2 = np.array([1 + s3, 3 + s3, 3 - s3, 1 - s3]) / (4 * math.sqrt(2.0))        # Daubechies' 4-tap filter, closed form
    assert np.allclose(W.daubechies_lowpass(2), db2, rtol=0, atol=1e-14)
    assert np.allclose(W.highpass(db2), [db2[3], -db2[2], db2[1], -db2[0]])


@pytest.mark.parametrize("N", range(1, 9))
def test_filter_is_an_orthonormal_daubechies_filter(N):
    """2N taps; sum = sqrt 2; double-shift orthonormality; N vanishing moments of the high-pass filter; minimum phase
    (every zero of H other than the N-fold one at -1 lies inside the unit circle); |H|^2 matches Daubechies' polynomial."""
    h = W.daubechies_lowpass(N)
    g = W.highpass(h)
    assert len(h) == 2 * N
    assert h.sum() == pytest.approx(math.sqrt(2.0), abs=1e-13)
    for m in range(N):
        dot = sum(h[k] * h[k + 2 * m] for k in range(2 * N - 2 * m))
        assert dot == pytest.approx(1.0 if m == 0 else 0.0, abs=1e-12)
        assert sum(h[k] * g[k + 2 * m] for k in range(2 * N - 2 * m)) == pytest.approx(0.0, abs=1e-12)
    k = np.arange(2 * N)
    for p in range(N):
        assert abs(np.sum(g * k.astype(float) ** p)) <= 1e-8 * max(1.0, float(np.sum(np.abs(g) * k.astype(float) ** p)))
    quo = h.copy()                                                 # divide the N-fold zero at -1 out: H(q) = (1+q)^N L(q)
    for _ in range(N):
        quo, rem = np.polydiv(quo, [1.0, 1.0])
        assert np.max(np.abs(rem)) <= 1e-9
    zeros = np.roots(quo[::-1])                                    # zeros of L in q = 1/z; minimum phase: zeros in z inside <=> |q| > 1
    assert len(zeros) == N - 1 and np.all(np.abs(zeros) > 1.0)
    for w in np.linspace(0.0, math.pi, 17):
        H = np.sum(h * np.exp(-1j * w * k))
        y = math.sin(w / 2) ** 2
        P = sum(math.comb(N - 1 + j, j) * y ** j for j in range(N))
        assert abs(H) ** 2 == pytest.approx(2.0 * math.cos(w / 2) ** (2 * N) * P, abs=1e-11)


def test_haar_by_hand_4x4():
    """One Haar level of a 4 x 4 image: 2 x 2 block sums / differences over 2, in the Mallat layout (along x first)."""
    x = np.arange(16, dtype=float).reshape(4, 4)
    a = W.basis_adjoint(x, 1, levels=1)
    for by in range(2):
        for bx in range(2):
            p, q, r, s = x[2 * by, 2 * bx], x[2 * by, 2 * bx + 1], x[2 * by + 1, 2 * bx], x[2 * by + 1, 2 * bx + 1]
            assert a[by, bx] == pytest.approx((p + q + r + s) / 2)               # low-low
            assert a[by, bx + 2] == pytest.approx((p - q + r - s) / 2)           # high along x, low along y
            assert a[by + 2, bx] == pytest.approx((p + q - r - s) / 2)           # low along x, high along y
            assert a[by + 2, bx + 2] == pytest.approx((p - q - r + s) / 2)
    assert np.allclose(W.basis_adjoint(x, 0), x)                                 # Dirac basis: identity


@pytest.mark.parametrize("n,levels", [(32, 3), (64, 3), (48, 2)])
def test_perfect_reconstruction_parseval_tight_frame_adjoint(n, levels):
    x = synth.random_complex((n, n), seed=5)
    alpha = W.psi_adjoint(x, levels)
    assert alpha.shape == (9, n, n)
    for b in range(W.N_BASES):
        assert np.abs(W.basis_forward(alpha[b], b, levels) - x).max() <= 1e-11 * np.abs(x).max()       # Psi_b Psi_b^dagger = I
        assert np.linalg.norm(alpha[b]) == pytest.approx(np.linalg.norm(x), rel=1e-12)                 # Parseval
    assert np.abs(W.psi_forward(alpha, levels) - 9.0 * x).max() <= 1e-10 * np.abs(x).max()             # Psi Psi^dagger = n_w I (W2)
    beta = np.stack([synth.random_complex((n, n), seed=20 + b) for b in range(9)])
    lhs = np.vdot(W.psi_forward(beta, levels), x)                                                      # <Psi beta, x> = <beta, Psi^dagger x>
    rhs = np.vdot(beta, alpha)
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(beta) * np.linalg.norm(x) * 3
    # a constant image has no detail coefficients at all (vanishing moments; periodic extension)
    c = W.basis_adjoint(np.ones((n, n)), 4, levels)
    m = n >> levels
    assert np.abs(c[m:, :]).max() <= 1e-10 and np.abs(c[:m, m:]).max() <= 1e-10
    assert np.allclose(c[:m, :m], 2.0 ** levels, atol=1e-10)


def test_soft_threshold_and_projection_hand_values():
    a = np.array([3.0, -3.0, 0.5, -0.5, 2.0, 3 + 4j, 0.3 + 0.4j, 1j * 2.5], dtype=complex)
    s = W.soft_threshold(a, 2.0)
    assert np.allclose(s, [1.0, -1.0, 0.0, 0.0, 0.0, (3 + 4j) * 3 / 5, 0.0, 0.5j])
    assert np.allclose(W.project_positive(np.array([1 + 2j, -1 + 2j, 0.25 - 1j])), [1.0, 0.0, 0.25])
    # prox property (Eq. 24): S_gamma(x) minimises gamma |v| + |v - x|^2 / 2 - checked against a brute-force scan
    for xv in (2.7, -0.4, 1.0):
        v = np.linspace(-4, 4, 80001)
        best = v[np.argmin(1.3 * np.abs(v) + 0.5 * (v - xv) ** 2)]
        assert W.soft_threshold(np.array([xv]), 1.3)[0].real == pytest.approx(best, abs=2e-4)


def test_dualfb_step_special_cases():
    n, levels = 32, 3
    z = synth.random_complex((n, n), seed=9)
    zb0 = W.project_positive(z)
    d0 = np.zeros((9, n, n), complex)
    # gamma = 0: S_0 is the identity, so d stays 0 and zbar = P_C(z)
    d, zb = W.dualfb_step(z, zb0, d0, 0.0, 1.0, levels)
    assert np.abs(d).max() <= 1e-14 and np.allclose(zb, zb0, rtol=0, atol=1e-12)
    # huge gamma: S_gamma(u) = 0, d = Psi^dagger zbar0 / eta, zbar = P_C(z - 9 zbar0 / eta)   (Psi Psi^dagger = 9 I)
    d, zb = W.dualfb_step(z, zb0, d0, 1e9, 18.0, levels)
    assert np.allclose(d, W.psi_adjoint(zb0, levels) / 18.0, atol=1e-13)
    assert np.allclose(zb, W.project_positive(z - 0.5 * zb0), atol=1e-11)
    # |d_i| <= gamma / eta always: (I - S_gamma) clips the modulus at gamma
    d, _ = W.dualfb_step(z, zb0, synth.random_complex((9, n, n), seed=10), 0.37, 2.0, levels)
    assert np.abs(d).max() <= 0.37 / 2.0 * (1 + 1e-12)
