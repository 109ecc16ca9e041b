"""sledge-b200: B200-native hot path of sledgehamr (arXiv 2404.02950).

The CUDA library is loaded lazily by `paper_2404_02950_b200.sledge`; importing the package (or
`paper_2404_02950_b200.inputs`) does not need a GPU.  There is no CPU fallback: every compute call
fails loudly if libsledge.so is missing or no CUDA device is present.
"""
__all__ = ["inputs", "sledge"]
