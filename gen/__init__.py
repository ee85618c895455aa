"""Seeded synthetic workload generator (inputs only; none of the solver's arithmetic).

Shared by the fp64 oracle (`oracle/`) and the CUDA path (`paper_2606_05687_b200/`):
both consume the same fp32-rounded arrays.  See DESIGN.md "Input recipe".
"""
from .workload import CONFIGS, SWEEP_B, SWEEP_N, Workload, make_workload, make_config, subset, centroidal_view  # noqa: F401
