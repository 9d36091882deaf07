"""Canaries around the outputs of the wavelet / DUALFB entry points (compute-sanitizer is closed on this pool).  -m gpu"""
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n,levels", [(40, 2), (96, 3), (16, 3)])
def test_wavelet_outputs_stay_inside_their_buffers(n, levels):
    from paper_1903_04502_b200 import C64, Wavelet
    GUARD = 4096
    wl = Wavelet(n, levels, C64)

    def guarded(count):
        buf = torch.full((count + 2 * GUARD,), complex(7.25, -3.5), dtype=torch.complex64, device="cuda")
        return buf, buf[GUARD:GUARD + count]

    def intact(buf, count):
        return bool((buf[:GUARD] == complex(7.25, -3.5)).all()) and bool((buf[GUARD + count:] == complex(7.25, -3.5)).all())

    x = torch.randn(n, n, dtype=torch.complex64, device="cuda")
    ba, a = guarded(9 * n * n)
    bx, xo = guarded(n * n)
    bd, d = guarded(9 * n * n)
    d.zero_()
    wl.adjoint(x, a.view(9, n, n))
    wl.forward(a.view(9, n, n), xo.view(n, n))
    wl.dualfb_step(x, x, d.view(9, n, n), 0.1, 9.0, zbar_out=xo.view(n, n))
    wl.project_positive(x, xo.view(n, n))
    torch.cuda.synchronize()
    assert intact(ba, 9 * n * n) and intact(bx, n * n) and intact(bd, 9 * n * n)
    wl.close()
