"""Comparison helper of the GPU parity tests: next to the rel-L2 over the whole output (BASELINE.json north_star:
<= 1e-12 complex128, <= 1e-5 complex64) every comparison also bounds the LARGEST element-wise deviation,

    max_i |a_i - ref_i|  <=  C_INF * tol * max_i |ref_i|,        C_INF = 1,

so that a handful of wrong elements cannot hide inside a norm (at M = 1e8 and tol 1e-5 about a hundred visibilities
could be off by 1 % and still pass the rel-L2).  Measured margins (profiles/parity_r2.md, all configs, both dtypes,
full sizes): rel-L2 <= 0.09 tol and max-abs <= 0.21 tol-units of max|ref| for every operator, composite ones
(Phi^dagger Phi, the ADMM step) included - so no operator gets a multiple of tol any more (round 1 allowed 2x - 4x).
Achieved errors are appended to gpurun_out/parity_r2.jsonl (when that directory exists); profiles/parity_r2.md is
written from it."""
import json
import os

import numpy as np

C_INF = 1.0
_LOG = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")


def errors(a, ref):
    """(rel-L2, max|a - ref| / max|ref|) blockwise (no M-sized complex128 temporaries)."""
    a = np.asarray(a).ravel()
    ref = np.asarray(ref).ravel()
    assert a.shape == ref.shape
    num = den = 0.0
    dmax = rmax = 0.0
    step = 1 << 24
    for i in range(0, max(len(ref), 1), step):
        rr = ref[i:i + step].astype(np.complex128)
        d = a[i:i + step].astype(np.complex128) - rr
        num += float(np.vdot(d, d).real)
        den += float(np.vdot(rr, rr).real)
        if len(rr):
            dmax = max(dmax, float(np.abs(d).max()))
            rmax = max(rmax, float(np.abs(rr).max()))
    if den == 0.0:
        return (0.0 if num == 0.0 else float("inf")), (0.0 if dmax == 0.0 else float("inf"))
    return (num / den) ** 0.5, dmax / rmax


def compare(label, a, ref, tol, l2_factor=1.0, scale=None, **ctx):
    """Assert both bounds; returns the rel-L2.  `l2_factor` (a multiple of tol) is 1 everywhere today.
    `scale`: magnitude the element-wise deviation is measured against when max|ref| is not the natural one (a clipped
    output whose inputs are much larger than its values)."""
    l2, linf = errors(a, ref)
    if scale is not None:
        linf = linf * float(np.abs(np.asarray(ref)).max()) / float(scale)
    if os.path.isdir(_LOG):
        with open(os.path.join(_LOG, "parity_r2.jsonl"), "a") as fh:
            fh.write(json.dumps(dict(label=label, rel_l2=l2, max_abs_over_max_ref=linf, tol=tol, l2_factor=l2_factor,
                                     elements=int(np.asarray(ref).size), **ctx)) + "\n")
    assert l2 <= l2_factor * tol, (label, "rel-L2", l2, tol, ctx)
    assert linf <= C_INF * l2_factor * tol, (label, "max-abs", linf, tol, ctx)
    return l2
