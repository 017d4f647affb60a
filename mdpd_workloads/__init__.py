"""Seeded synthetic input generators for the mDPD hot path (configs 0-4 of BASELINE.json).

This module is shared by the fp64 oracle (``oracle/``) and the CUDA path
(``paper_1903_10134_b200/``).  It holds NONE of the method's arithmetic: no weight
function, no force, no hash, no integrator, no cell list.  It only draws particle
positions / velocities / types and voxel masks from ``numpy.random.default_rng(seed)``
and names the parameter values each configuration uses.

Recipe: seed = 190310134 + config
index; positions are float32 values in [0, L) so that the oracle (which upcasts them to
fp64) and the GPU path (fp32) start from bit-identical coordinates.  These inputs stand
in for the paper's workloads (Fig. 3 box, L141 slab, L180 porous cell,
L247 FIB-SEM pore) whose data files are not available.
"""
from .generators import (  # noqa: F401
    BASE_SEED,
    default_params,
    make_liquid,
    make_slab,
    make_poiseuille,
    make_pore_network,
    make_species_mixture,
    make_liquid_vacuum,
    make_slit_wetting,
    make_config,
    quantise_positions,
    maxwell_velocities,
)
