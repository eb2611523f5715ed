"""B200-native MLP-Splatting forward render (arxiv/paper_2606_03877).

`synth` (seeded inputs) imports nothing heavy; the CUDA binding is loaded on
first use of `paper_2606_03877_b200.api`.
"""
__all__ = ["synth"]
