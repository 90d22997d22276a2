"""paper_2502_21231_b200 — B200-native hot path of ByteScale's HDP step (arXiv 2502.21231):
packed varlen / zigzag-CP causal attention (fwd, LSE merge, bwd) behind a C-ABI library.

``from paper_2502_21231_b200 import binding`` loads csrc/libbytescale_attn.so and fails loudly
if it is missing; ``paper_2502_21231_b200.synth`` (seeded inputs) imports no native CUDA code.
"""
__all__ = ["binding", "synth"]
