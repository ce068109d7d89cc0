"""B200-native nodal DG + multidimensional HABC time stepper (arXiv 1610.05023) behind a C ABI.

`Solver` wraps `include/dg_habc.h` (libdg_habc.so, hand-written CUDA for sm_100a).  There is no CPU fallback."""
from .binding import DgError, Solver, dg_mesh_counts, dg_reference_element, lib  # noqa: F401

__all__ = ["Solver", "DgError", "dg_reference_element", "dg_mesh_counts", "lib"]
