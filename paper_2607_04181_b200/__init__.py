"""cocoscale-b200: the replicated decoder-layer hot path of CoCoScale (arxiv/paper_2607_04181)
as hand-written sm_100a CUDA behind a C ABI (include/cocoscale.h).

`paper_2607_04181_b200.binding` is the thin ctypes layer over libcocoscale.so (argument
marshalling only); `paper_2607_04181_b200.inputs` holds the seeded synthetic-input recipe and
none of the method's arithmetic.  Importing the package does not load the CUDA library; using
`binding` without the built library raises (there is no CPU fallback).
"""
__all__ = ["binding", "inputs", "build"]
