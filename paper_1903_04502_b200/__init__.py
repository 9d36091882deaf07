"""B200-native measurement operator Phi = W G F Z S / Phi^dagger of arXiv 1903.04502 (PURIFY).

    from paper_1903_04502_b200 import PurifyOp

`op` needs the built C-ABI library (`python -m paper_1903_04502_b200.build`) and fails loudly without it -
there is no CPU fallback.  The seeded input generators live outside the package, in `inputs/`.
"""
from .op import ANALYTIC, C64, C128, TABLE, UBENCH_FORMS, PurifyError, PurifyOp, load_library, ubench_fma  # noqa: F401
from .wavelet import Wavelet  # noqa: F401,E402
