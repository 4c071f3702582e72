"""ptfock -- B200-native plane-wave Fock exchange (hot path of arXiv:1905.01348, Eq. 3 / Alg. 2).

``paper_1905_01348_b200.binding`` is the thin Python face of the C-ABI library declared in
``include/ptfock.h`` (argument marshalling only); ``paper_1905_01348_b200.synth`` makes the seeded
synthetic inputs.  Importing the package does not load the CUDA library; using ``binding`` without it
raises (there is no CPU fallback).
"""
__all__ = ["binding", "synth"]
