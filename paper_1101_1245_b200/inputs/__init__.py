"""Seeded synthetic input generators (tables, phantoms, spectra, the five configs).

Data only: nothing here takes part in the transport arithmetic; the CUDA
library and the CPU oracle both receive these arrays as plain inputs.
"""
from .configs import (ELECTRON, PENCIL, PHASE_SPACE, PHOTON, RECTANGLE, Source, Workload, make_config,  # noqa: F401
                      make_paper_geometry)
from .phase_space import synthetic_phase_space  # noqa: F401
from .tables import TableBundle, build_tables  # noqa: F401
