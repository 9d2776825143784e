"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This module holds INPUT DATA generators only: materials, photon cross-section
tables and voxel phantoms (material / density / activity / organ labels) for the
five BASELINE.json configs.  It contains none of the method's arithmetic (no
source sampling, no transport, no tally, no statistics) and imports neither
`oracle/` nor `paper_2111_11687_b200/`.  Both sides receive its arrays as plain
inputs (north_star: "shares no code with the GPU path (only the generated
material and cross-section data files)").

Stand-in notice: the paper's patient PET/CT and its 27 organ
contours are private clinical data; the phantoms here are
synthetic with the shapes and value ranges BASELINE.json `configs` state.
"""
from .materials import MATERIALS, MATERIAL_IDS, electrons_per_gram  # noqa: F401
from .tables import make_tables, sigma_kn_per_electron, E0_MEV  # noqa: F401
from .phantoms import make_config, make_patient_on_grid, ORGAN_NAMES, CONFIG_NAMES  # noqa: F401
from .images import DEFAULT_HU_RAMP, make_ct_pet, density_to_hu  # noqa: F401
from .electrons import make_electron_tables, bethe_collision_stopping, ELECTRON_CUTOFF_MEV  # noqa: F401
