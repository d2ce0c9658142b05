"""avm — microscopic electron-avalanche transport (null-collision Monte Carlo) on one B200.

Layout: `gen/` seeded input generators (gas tables, field maps, primaries; shared with the tests' oracle
as *inputs* only), `csrc/` the hand-written sm_100a CUDA kernels behind the C ABI of include/avm.h,
`avm.py` the thin ctypes binding (argument marshalling only).  Importing the package does not load the
CUDA library; `paper_2509_15377_b200.avm` does, and fails loudly when it is missing.
"""
__all__ = ["gen"]
