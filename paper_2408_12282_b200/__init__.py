"""sssgs: B200-native forward relighting render path of SSS-GS (arXiv 2408.12282).

`scenes` (numpy input generators) imports without the CUDA library; the renderer
binding (`paper_2408_12282_b200.binding`) loads `libsssgs.so` and fails loudly if it
is missing -- there is no CPU fallback.
"""
__all__ = ["scenes"]
