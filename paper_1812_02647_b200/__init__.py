"""paper_1812_02647_b200 — batched incoherent harmonic sum (arXiv 1812.02647, eqs. 1-4) for NVIDIA B200.

The product is the C-ABI library libhs.so (include/hs.h, csrc/); this package is its thin Python binding
(`binding`), the in-tree build step (`build`) and the batch partition used for multi-GPU runs (`shard`).
Attribute access is lazy so that `python -m paper_1812_02647_b200.build` works before libhs.so exists; touching
any binding name without the library raises ImportError (there is no CPU fallback).
"""
_BINDING_NAMES = ("ALGOS", "HS_ALGO_AUTO", "HS_ALGO_DIRECT", "HS_ALGO_TILED", "HS_ALGO_TWOPHASE", "HS_FREQBIN", "HS_GREEDY", "HS_MAX",
                  "HS_OUT_BOTH", "HS_OUT_FULL", "HS_OUT_REDUCED", "HS_STANDARD", "LIB_PATH", "OUT_MODES", "VARIANTS",
                  "HsError", "Plan", "hs_plan_create", "lib")


def __getattr__(name):
    if name in _BINDING_NAMES:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
