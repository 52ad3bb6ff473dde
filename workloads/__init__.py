"""Seeded synthetic inputs and config definitions shared by the oracle-side and CUDA-side
tests and by bench.py.  Holds none of the method's arithmetic (no field, tensor, FFT or LLG
code): only random numbers, the five BASELINE.json configs and the error metric."""
from .configs import (CONFIGS, PAPER_DEMAG_MS, PAPER_MESHES, SWEEP_MESHES, Config,  # noqa: F401
                      get_config)
from .generators import (box_filter_renormalise, in_plane_state, normal_field,  # noqa: F401
                         random_unit_vectors, sample_cells, sparse_sources)
from .metrics import field_errors, traj_error  # noqa: F401
