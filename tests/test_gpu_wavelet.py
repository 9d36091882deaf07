"""f4 on the CUDA path (through the C ABI of include/purify_wavelet.h) against oracle/wavelets.py.  -m gpu"""
import numpy as np
import pytest
import torch

from inputs import synth
from oracle import wavelets as W
from parity_util import compare

pytestmark = pytest.mark.gpu
TOL = {"c128": 1e-12, "c64": 1e-5}


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make(n, levels, dtype):
    from paper_1903_04502_b200 import C64, C128, Wavelet
    return Wavelet(n, levels, C64 if dtype == "c64" else C128)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_filters_match_the_oracle_and_are_orthonormal(dtype):
    wl = make(64, 3, dtype)
    for N in range(1, 9):
        h = np.array(wl.filter(N))
        assert len(h) == 2 * N
        assert np.max(np.abs(h - W.daubechies_lowpass(N))) <= 2e-13        # two independent root finders
        for m in range(N):
            assert abs(sum(h[k] * h[k + 2 * m] for k in range(2 * N - 2 * m)) - (1.0 if m == 0 else 0.0)) <= 1e-12
    wl.close()


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("n,levels", [(64, 3), (96, 3), (256, 3), (40, 2), (16, 3), (128, 1)])
def test_psi_and_psi_dagger(dtype, n, levels):
    """n = 16 with 3 levels: the deepest level is 4 x 4, every filter longer than 4 taps wraps around several times."""
    wl = make(n, levels, dtype)
    cd = synth.complex_dtype(dtype)
    x = synth.random_complex((n, n), seed=n + levels, dtype=dtype)
    ctx = dict(n=n, levels=levels, dtype=dtype)
    alpha = wl.adjoint(dev(x))
    a_ref = W.psi_adjoint(x, levels)
    compare("Psi^dagger x", alpha.cpu().numpy(), a_ref, TOL[dtype], **ctx)
    for b in (0, 1, 4, 8):
        compare(f"Psi_{b}^dagger x", alpha[b].cpu().numpy(), a_ref[b], TOL[dtype], **ctx)
    beta = np.stack([synth.random_complex((n, n), seed=50 + b, dtype=dtype) for b in range(9)]).astype(cd)
    xs = wl.forward(dev(beta))
    compare("Psi alpha", xs.cpu().numpy(), W.psi_forward(beta, levels), TOL[dtype], **ctx)
    # tight frame on the GPU results themselves: Psi Psi^dagger x = 9 x; alpha untouched by the synthesis
    keep = alpha.clone()
    compare("Psi Psi^dagger x = 9 x", wl.forward(alpha).cpu().numpy(), 9.0 * x, TOL[dtype], **ctx)
    assert torch.equal(alpha, keep)
    # adjoint identity with GPU results
    lhs = np.vdot(xs.cpu().numpy().astype(np.complex128), x.astype(np.complex128))
    rhs = np.vdot(beta.astype(np.complex128), alpha.cpu().numpy().astype(np.complex128))
    assert abs(lhs - rhs) <= TOL[dtype] * np.linalg.norm(beta) * np.linalg.norm(x) * 3
    wl.close()


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("gamma,eta", [(0.0, 1.0), (0.4, 9.0), (1e9, 18.0), (0.05, 1.0)])
def test_dualfb_step(dtype, gamma, eta):
    n, levels = 128, 3
    wl = make(n, levels, dtype)
    cd = synth.complex_dtype(dtype)
    z = (synth.make_image(n, 1001, dtype) * 3 + synth.random_complex((n, n), seed=3, dtype=dtype) * 0.05).astype(cd)
    d0 = (np.stack([synth.random_complex((n, n), seed=70 + b, dtype=dtype) for b in range(9)]) * 0.02).astype(cd)
    zb0_ref = W.project_positive(z)
    zb0 = wl.project_positive(dev(z))
    assert np.array_equal(zb0.cpu().numpy(), zb0_ref.astype(cd))
    ctx = dict(n=n, dtype=dtype, gamma=gamma, eta=eta)
    # d = (I - S_gamma)(u) / eta is u clipped to modulus gamma: its rounding error is that of u = eta d + Psi^dagger zbar
    # (sums of O(max|u|) terms), so the element-wise deviation is measured against max|u| / eta, not against gamma / eta
    u_scale = float(np.abs(eta * d0 + W.psi_adjoint(zb0_ref, levels)).max()) / eta
    d_dev = dev(d0)
    zb1 = wl.dualfb_step(dev(z), zb0, d_dev, gamma, eta)
    d_ref, zb1_ref = W.dualfb_step(z, zb0_ref, d0, gamma, eta, levels)
    if gamma == 0.0:            # (I - S_0) = 0: d is zero up to the oracle's rounding of u (|u| - 0)/|u| - no relative comparison
        assert float(d_dev.abs().max()) <= 1e-6 * TOL[dtype] and np.abs(d_ref).max() <= 1e-13
    else:
        compare("DUALFB d", d_dev.cpu().numpy(), d_ref, TOL[dtype], scale=u_scale, **ctx)
    compare("DUALFB zbar", zb1.cpu().numpy(), zb1_ref, TOL[dtype], **ctx)
    assert float(zb1.real.min()) >= 0.0 and float(zb1.imag.abs().max()) == 0.0
    # a second pass from the GPU's own state, zbar written in place
    wl.dualfb_step(dev(z), zb1, d_dev, gamma, eta, zbar_out=zb1)
    d_ref2, zb2_ref = W.dualfb_step(z, zb1_ref, d_ref, gamma, eta, levels)
    if gamma > 0.0:
        compare("DUALFB d, second pass", d_dev.cpu().numpy(), d_ref2, TOL[dtype], scale=u_scale, **ctx)
    compare("DUALFB zbar, second pass", zb1.cpu().numpy(), zb2_ref, TOL[dtype], **ctx)
    wl.close()


def test_wavelet_errors():
    from paper_1903_04502_b200 import C64, PurifyError, Wavelet
    for n, levels in ((100, 3), (0, 3), (64, 0), (64, 9)):
        with pytest.raises(PurifyError) as ei:
            Wavelet(n, levels, C64)
        assert ei.value.status == -1
    wl = Wavelet(64, 3, C64)
    with pytest.raises(ValueError):
        wl.adjoint(torch.zeros((32, 32), dtype=torch.complex64, device="cuda"))
    with pytest.raises(PurifyError):
        wl.dualfb_step(wl.new_image(), wl.new_image(), wl.new_coefficients(), 0.1, 0.0)
    wl.close()
