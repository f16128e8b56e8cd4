"""B200-native batched exact division of midsize unsigned integers (arxiv/paper_2606_06386).

The product is the C-ABI library ``libmpdiv.so`` (include/mpdiv.h) built from the CUDA sources
under ``csrc/``; ``binding`` marshals arguments to it, ``inputs`` draws the seeded workloads.
Nothing here falls back to a CPU path: calling an op without the built library raises.
"""
__all__ = ["binding", "inputs", "build"]
