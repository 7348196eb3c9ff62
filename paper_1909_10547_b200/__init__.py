"""fkconv: B200-native Fast-Kernel (FK) table convolution (arXiv:1909.10547, Eq. (1)).

`paper_1909_10547_b200.fkconv` is the thin ctypes binding over the C-ABI library
(`include/fkconv.h`); importing it fails loudly if `libfkconv.so` has not been built.
`paper_1909_10547_b200.synth` holds the seeded input generators (no method arithmetic).
Nothing here imports `oracle/`.
"""
__all__ = ["fkconv", "synth"]
