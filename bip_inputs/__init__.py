"""Seeded synthetic inputs for BiP-PRISM (arxiv/paper_2607_00756).

This package is the ONLY code shared by the fp64 CPU oracle (``oracle/``) and the
CUDA path (``paper_2607_00756_b200/``).  It holds no arithmetic of the method:
it only manufactures *problem data* -- specimen transmission functions ``T_j``
(PAPER.md:51), transition-potential windows ``H_n``, ionised-atom
sites snapped to (slice, pixel), scan positions and the
scalar microscope parameters -- with the shapes of the paper's workloads
(BASELINE.json ``configs``; recipe in DESIGN.md §4).  Beam sets, parent selection,
interpolation weights, probe coefficients, scattering matrices and everything
downstream are computed separately by each side.
"""
from .physics import electron_wavelength, interaction_constant
from .specimen import Workload, make_workload, CONFIGS

__all__ = ["electron_wavelength", "interaction_constant", "Workload", "make_workload", "CONFIGS"]
