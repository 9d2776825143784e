"""paper_2111_11687_b200 -- B200-native voxel Monte Carlo dose engine for annihilation photons
(the hot path of ARCHER-NM, arxiv 2111.11687).  The product is libanm.so (include/anm.h, csrc/);
this package is its thin Python binding.  There is no CPU fallback: `load()` raises if the CUDA
library is missing or no GPU is usable."""
from .binding import Simulation, AnmError, load, lib_path, ANM_SYMBOLS, organ_summary_static  # noqa: F401
