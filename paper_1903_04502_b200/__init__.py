"""B200-native measurement operator Phi = W G F Z S / Phi^dagger of arXiv 1903.04502 (PURIFY).

    from paper_1903_04502_b200 import PurifyOp

`synth` (seeded input generators) is importable without CUDA; `op` needs the built C-ABI library
(`python -m paper_1903_04502_b200.build`) and fails loudly without it - there is no CPU fallback.
"""
from .op import ANALYTIC, C64, C128, TABLE, PurifyError, PurifyOp, load_library  # noqa: F401
