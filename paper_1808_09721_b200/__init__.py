"""B200-native IMEX SSP2(222) step for resistive / two-fluid special-relativistic MHD.

The product path is the CUDA library ``librmhd.so`` (C-ABI in include/rmhd.h) reached through
:mod:`paper_1808_09721_b200.binding`; there is no CPU fallback.  :mod:`paper_1808_09721_b200.synth`
holds the seeded input generators only.
"""
__all__ = ["binding", "synth", "build"]
