"""B200-native direct J/K and J/K-gradient engine (hot path of arxiv 2407.09700).

`workloads` holds the seeded input generators (no method arithmetic).
`eri` is the thin ctypes binding over the C-ABI library `liberi_b200.so` (include/eri.h);
it is imported lazily so that the generators can be used without the CUDA build.
"""

__all__ = ["workloads", "eri"]
