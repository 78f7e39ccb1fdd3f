"""B200-native DOCTORS hot path (arXiv 1910.11335): the discrete-ordinates transport sweep of
Eq. (2) inside the multigroup source iteration, as a C-ABI CUDA library (sm_100a) plus this thin
binding.  See DESIGN.md.  No CPU fallback: the library must be built (`build.build()`)."""
from .binding import (Problem, DoctorsError, problem_from_workload, load_library, wavefront_size,
                      host_level_symmetric, host_schedule, host_projection_tables, EXPORTS, LIB_PATH,
                      OK, INVALID_ARG, BAD_STATE, ALLOC, CUDA, NOT_CONVERGED, NOT_RETAINED)

__all__ = ["Problem", "DoctorsError", "problem_from_workload", "load_library", "wavefront_size",
           "host_level_symmetric", "host_schedule", "host_projection_tables", "EXPORTS", "LIB_PATH"]
