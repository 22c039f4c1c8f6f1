"""Seeded synthetic inputs shaped like the paper's workloads.

This package holds NO arithmetic of the method (no projection, binning, DFT, peak pick): it only
produces ion clouds, ion types, material-point centres and the scalar parameters of each config.
Both the CPU oracle (``oracle/``) and the CUDA path (``paper_2009_00735_b200/``) are fed from here;
neither imports the other.
"""
from .lattices import (fcc_basis, bcc_basis, random_rotation, lattice_in_box, lattice_in_ball,
                       jitter_thin_shuffle)
from .configs import CONFIGS, make_config, window_for, Workload

__all__ = ["fcc_basis", "bcc_basis", "random_rotation", "lattice_in_box", "lattice_in_ball",
           "jitter_thin_shuffle", "CONFIGS", "make_config", "window_for", "Workload"]
