"""paper_2606_18600_b200 — B200-native forward pass of one ShuntServe pipeline stage (arxiv/paper_2606_18600).

The product is ``libshuntstage.so`` (hand-written CUDA for sm_100a behind the C-ABI of ``include/shuntstage.h``);
``binding`` is the thin ctypes layer with the same names, ``synth`` the seeded input generators, ``estimator``
the paper's Eq. 1 / Table 2 closed form printed beside measurements.  Importing this package does not load CUDA.
"""
__all__ = ["binding", "synth", "estimator", "build"]
