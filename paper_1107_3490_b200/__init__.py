"""B200-native replica-exchange Monte Carlo of a bead-spring homopolymer (arxiv 1107.3490).

The product is the C-ABI library ``libpt_b200.so`` (include/pt_b200.h, csrc/); this package
is its thin Python binding plus the seeded synthetic-input generators (``synth``).
Importing the package does not load the library; ``binding.lib()`` does, and fails loudly
if it cannot be built -- there is no CPU fallback.
"""
from .binding import (PT_F32, PT_F64, PT_RANDOM_PICK, PT_SEQUENTIAL, ParallelTempering, PtError,
                      PtParams, lib, lib_path, make_params, pt_fma_peak, pt_workspace_bytes)

__all__ = ["PT_F32", "PT_F64", "PT_RANDOM_PICK", "PT_SEQUENTIAL", "ParallelTempering", "PtError",
           "PtParams", "lib", "lib_path", "make_params", "pt_fma_peak", "pt_workspace_bytes"]
