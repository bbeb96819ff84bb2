"""B200-native Count-Sketch heavy-hitter pass for N-body particles (arXiv 1711.00975).

`paper_1711_00975_b200.binding` is the thin ctypes binding over the C-ABI library `libcs.so`
(include/cs.h); `paper_1711_00975_b200.synth` holds the seeded synthetic streams.  Importing the
package does not load the CUDA library; `binding` loads it on first use and fails loudly if it is missing.
"""
__all__ = ["binding", "synth"]
