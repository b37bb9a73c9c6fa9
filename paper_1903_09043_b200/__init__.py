"""ark-b200: B200-native (sm_100a) hot path of the ARK all-Mach, well-balanced finite-volume solver
(arXiv 1903.09043).  `binding` is the thin ctypes layer over the C-ABI library (include/ark.h);
`inputs` holds the seeded synthetic workloads.  Nothing is imported eagerly: importing `inputs`
must not require the CUDA extension, and `binding` fails loudly if the extension is missing."""
__all__ = ["binding", "inputs"]
