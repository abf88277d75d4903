"""B200-native nested slice sampling hot path (arxiv 2509.24949) behind a C-ABI CUDA library.

`paper_2509_24949_b200.nss` is the thin ctypes binding over `csrc/libnss.so` (argument marshalling
only); `paper_2509_24949_b200.inputs` holds the seeded synthetic workloads (no method arithmetic).
Importing the package does not load the CUDA library; the binding loads it on first use and
raises if it is missing (there is no CPU fallback).
"""
__all__ = ["inputs", "nss"]
