"""B200-native photon-packet transport (Heymann & Siebenmorgen, arxiv 1203.2941) behind a C ABI.

``binding`` holds the thin ctypes layer over libmcrt_b200.so (same names as include/mcrt.h);
``workloads`` holds the seeded synthetic input generators.  Importing the package loads nothing.
"""
__all__ = ["binding", "workloads"]
