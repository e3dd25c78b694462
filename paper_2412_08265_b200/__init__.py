"""B200-native hot path of RUBIX's IFU forward model (arXiv 2412.08265, §3 L40).

``synth``   seeded synthetic workloads (shared with the oracle tests; no method arithmetic)
``binding`` thin ctypes layer over the C-ABI library ``librubix_b200.so`` (include/rubix.h)
``build``   nvcc invocation that produces the library in-tree

Nothing here falls back to the CPU: importing ``binding`` without the built library, or calling
it without a CUDA device, raises.
"""
__all__ = ["synth", "binding", "build", "replicas"]
