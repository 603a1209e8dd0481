"""B200-native batched drone-environment step of arxiv/paper_2606_08039 (MuJoCo-Drones-Gym).

The product is the CUDA library behind `include/mdg.h` (built in-tree as `libmdg.so`); this package is
its thin Python binding plus the seeded workload recipes.  Importing the package does not load CUDA;
using `Env` without the built library or without a GPU raises.
"""
from . import workloads
from .binding import Env, MdgError, default_params, lib, mdg_params, measure_fp32_peak

__all__ = ["Env", "MdgError", "default_params", "lib", "mdg_params", "measure_fp32_peak", "workloads"]
