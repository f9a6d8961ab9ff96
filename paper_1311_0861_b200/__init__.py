"""B200-native hot path of GPUPEGAS (arXiv:1311.0861): one explicit Godunov + FIIC timestep.

`Simulation` wraps the C-ABI library libgpupegas.so (include/gpupegas.h); `workloads` holds the
seeded synthetic inputs.  Importing the package loads nothing; the first call into the library
fails loudly if it has not been built or no CUDA device is present.
"""
from . import workloads  # noqa: F401
from .binding import (FIELDS, GAS_FIELDS, STAR_FIELDS, GP_BC_OUTFLOW, GP_BC_PERIODIC, GP_ERR_STATE, GP_GAS,  # noqa: F401
                      GP_POISSON_ISOLATED, GP_POISSON_NONE, GP_POISSON_PERIODIC, GP_STARS, GpError, Simulation, lib, fp64_rate_selftest, math_selftest)
