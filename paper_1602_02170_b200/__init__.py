"""B200-native RPY / wall-RPY blob mobility matvec (hot path of arXiv:1602.02170).

``u = M lambda`` by direct O(N_b^2) summation with M the RPY tensor,
Eq. (9), plus the single-wall Rotne-Prager-Blake correction
(PAPER.md:148).  All arithmetic runs in hand-written sm_100a CUDA kernels behind the
C ABI declared in ``include/rpy_matvec.h``; this package is the thin Python binding
(argument marshalling only).  There is no CPU fallback: calling a matvec without the
built CUDA library, or without a CUDA device, raises.

The native library is loaded on first use, so importing ``workloads`` (seeded input
generators, no method arithmetic) works on a CPU-only box.
"""
from __future__ import annotations

__all__ = [
    "rpy_wall_matvec", "rpy_free_matvec", "rpy_wall_matvec_host", "rpy_free_matvec_host",
    "rpy_matvec_workspace_bytes", "rpy_matvec_host_scratch_bytes", "rpy_wall_count_below",
    "rpy_matvec_launch_plan",
    "rpy_wall_matvec_shard", "rpy_free_matvec_shard", "rpy_wall_matvec_rect", "rpy_free_matvec_rect", "rpy_matvec_rect_workspace_bytes", "rpy_flow_subdivide",
    "rpy_status_string", "RpyError", "load_library", "library_path",
]


def __getattr__(name):
    if name in __all__:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
