"""B200-native plate-level RAM Metropolis-within-Gibbs sampler (hot path of arXiv 2105.08026).

`paper_2105_08026_b200.binding` is the thin ctypes binding of the C-ABI library
(`include/cudahm.h`, built from `csrc/`); `paper_2105_08026_b200.synth` holds the seeded
synthetic inputs.  Nothing here imports the CPU oracle.
"""
__all__ = ["binding", "synth"]
