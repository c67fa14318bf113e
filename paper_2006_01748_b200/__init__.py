"""gg-b200: B200-native explicit finite-volume step for the anisotropic, heterogeneous
Gatenby-Gawlinski tumour-invasion model (Mascia, Pera, Simeoni, arXiv 2006.01748).

The product is the C-ABI library `libgg.so` (include/gg.h, csrc/) -- hand-written CUDA for
sm_100a.  `paper_2006_01748_b200.binding` is its thin ctypes binding (argument marshalling only);
`paper_2006_01748_b200.workloads` builds the seeded synthetic inputs.  Nothing here imports the
CPU oracle under oracle/, and there is no CPU fallback: the binding raises if the CUDA library is
missing.
"""
__all__ = ["binding", "workloads"]
