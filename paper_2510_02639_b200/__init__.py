"""B200-native image-centred ray shooting (ICRS) hot path of arxiv 2510.02639.

`binding` is the thin ctypes layer over the C ABI in include/ulens.h (CUDA only, no CPU fallback);
`inputs` holds the seeded synthetic workloads C0..C4; `build` compiles the library for sm_100a.
"""
