"""B200-native hot path of SOC's Monte Carlo radiative transfer (arXiv:1812.06632).

`paper_1812_06632_b200.soc` is the thin ctypes binding over the C-ABI library (include/soc.h);
`paper_1812_06632_b200.inputs` manufactures the seeded synthetic inputs.  Nothing here falls back to
a CPU implementation: using the binding without the built CUDA library raises.
"""
__all__ = ["soc", "inputs"]
