"""kappagen for B200: the hot path of arXiv 2602.05606 (approximate Kappa generator, Table I).

`paper_2602_05606_b200.kappagen` is the thin ctypes binding over the C-ABI library libkappagen
(include/kappagen.h); `paper_2602_05606_b200.workloads` builds the seeded synthetic inputs.
Importing this package does not load the CUDA library; the first call through the binding does,
and fails loudly if it has not been built (python -c "import __graft_entry__ as g; g.build()").
"""
__all__ = ["kappagen", "workloads"]
