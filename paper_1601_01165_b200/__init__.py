"""dedisp-b200: brute-force incoherent dedispersion (arXiv 1601.01165) for sm_100a.

The Python side is a thin binding over the C-ABI library (include/dedisp.h).
Import `paper_1601_01165_b200.dedisp` for the calls; `workloads` holds the
observational setups and seeded synthetic inputs.
"""
__version__ = "0.1.0"
