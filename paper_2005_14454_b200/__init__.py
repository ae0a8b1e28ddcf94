"""paper_2005_14454_b200 — Abelian-Higgs leapfrog hot path on one B200 (sm_100a).

`inputs` (seeded generators, numpy only) can be imported without the CUDA
library; everything in `binding` needs the built C-ABI library and raises
loudly if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "inputs", "replicas"]
