"""B200-native parallel tempering for the 3D Random Field Ising Model (arxiv 1508.06268).

The product is the C-ABI library ``librfimpt.so`` (declared in ``include/rfim_pt.h``,
sources under ``csrc/``); ``binding`` is the thin ctypes layer above it.  Importing this
package does not load the library; the first call through ``binding`` does, and fails
loudly if the CUDA extension has not been built.
"""
__all__ = ["binding", "workloads", "build"]
