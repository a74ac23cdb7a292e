"""B200-native Lagrangian particle step + binning (hot path of arxiv/paper_0912_3223).

CUDA kernels for sm_100a behind the C ABI of include/lpm.h (csrc/, built into liblpm_b200.so by
`python -m paper_0912_3223_b200.build`) and a thin ctypes binding with the same entry points.
Importing the package is light; the shared library is loaded on first use and its absence is an
error (there is no CPU fallback).
"""
from .binding import (LEDGER_NAMES, box_muller_kernel, curand_philox_kernel, LpmError, Simulation, load, normals_kernel, philox_kernel, probe, sample_kernel, sample_static,  # noqa: F401
                      schedule_born, status_string, version, workspace_bytes)
