"""B200-native SPH hot path of CCAKE 2.0 (arxiv 2511.22852): CUDA kernels behind the C ABI of include/ccake.h.

`paper_2511_22852_b200.binding` is the thin ctypes layer over libccake.so (argument marshalling only);
`paper_2511_22852_b200.workloads` holds the seeded input generators.  The CUDA library is loaded on first use
of the binding and raises loudly when it is missing — there is no CPU fallback.
"""
__all__ = ["binding", "workloads", "build"]
