"""caee-b200: the CAEE (Cost-Aware Expert Execution, arxiv 2606.29982) per-layer MoE
decode hot path for NVIDIA B200 (sm_100a).

`workloads` holds the seeded synthetic inputs; `binding` is the thin ctypes layer over
the C-ABI library `libcaee.so` (built from csrc/ by `build.build()`), and raises at import
if that library is missing: there is no CPU fallback.
"""
__all__ = ["workloads"]
