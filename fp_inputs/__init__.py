"""Seeded synthetic inputs for the FourPhonon hot path (crystals, harmonic phonons, anharmonic IFC lists).

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2510_00518_b200/`).  It prepares inputs ("harmonic properties ... inherently on
the CPU") and holds none of the scattering-rate arithmetic: no momentum/energy filter, no broadening, no matrix
element, no occupation factor, no rate sum.
"""
from .generate import (  # noqa: F401
    Crystal, Inputs, diamond_crystal, sc8_crystal, sc1_crystal, spring_fc2, phonons, clusters, random_ifc,
    make_config, make_tiny, qpoint_index, qpoint_coords, CONFIG_NAMES, PAPER_MESHES,
)
