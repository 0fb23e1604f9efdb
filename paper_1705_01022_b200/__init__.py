"""B200-native engine for the domain-decomposed random-sequential sweep of the 2+1-d octahedron model
(arXiv 1705.01022).  The product is the C-ABI library built from ``csrc/`` (declared in
``include/oct.h``); ``binding`` is argument marshalling only.  Nothing here imports ``oracle``.

Importing the package is cheap; the CUDA library is loaded on first use of ``binding``.
"""
__all__ = ["binding", "workloads", "build"]
