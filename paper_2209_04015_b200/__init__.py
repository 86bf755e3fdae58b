"""B200-native batched phaseless-AFQMC local energy (arXiv 2209.04015, single-determinant trials).

Thin Python binding over the C-ABI shared library ``libafqmc.so`` (include/afqmc.h).  Importing this package
does not load the library; the first use does, and fails loudly if it has not been built
(``python -c "import __graft_entry__ as g; g.build()"``).  There is no CPU fallback.
"""
from .binding import (AfqmcError, LocalEnergy, fp64_peak_tflops, library_path, load_library, log_overlap_static, phaseless_weights,
                      plan, sample_fields)  # noqa: F401
from .build import build_library  # noqa: F401
from .parallel import gather_walker_results, max_over_ranks, walker_shard  # noqa: F401
