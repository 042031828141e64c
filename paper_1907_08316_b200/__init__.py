"""sldg-b200: B200-native SLDG translation sweep / Vlasov-Poisson Strang step (arXiv:1907.08316).

`paper_1907_08316_b200.sldg` is the Python binding of the C-ABI library (include/sldg.h);
`paper_1907_08316_b200.workloads` holds the seeded input generators (no method arithmetic).
Importing this package does not load CUDA; importing `.sldg` loads libsldg.so and fails
loudly if it has not been built (python -c "import __graft_entry__ as g; g.build()").
"""
__all__ = ["workloads"]
