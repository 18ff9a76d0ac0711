"""B200-native MONC advection source terms (arxiv 2009.12850's GPU offload).

The product is the C-ABI library declared in include/monc_adv.h, built from
csrc/ for sm_100a.  `paper_2009_12850_b200.binding` is the thin ctypes binding
(argument marshalling only); `paper_2009_12850_b200.synth` holds the seeded
synthetic inputs.  Nothing is loaded at package import: the CUDA library is
opened on first use of the binding and fails loudly when it is missing.
"""
__all__ = ["binding", "synth", "build"]
