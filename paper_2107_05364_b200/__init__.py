"""paper_2107_05364_b200 — B200-native hot path of MagTense (arxiv 2107.05364).

`binding` is the thin ctypes layer over the C-ABI library (include/mt.h, csrc/*.cu);
`workloads` holds the seeded synthetic inputs; `build` compiles the library in-tree.
Importing the package does not load the CUDA library; `binding.load()` does, and fails loudly
when it is missing — there is no CPU fallback.
"""
from . import binding, workloads  # noqa: F401

__all__ = ["binding", "workloads"]
