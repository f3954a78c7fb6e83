"""Seeded synthetic inputs and workload shapes for the five configurations of BASELINE.json.

This module serves BOTH the CPU oracle's tests and the CUDA library's tests / bench and
therefore holds none of the method's arithmetic: no differentiation matrix, no spin-weighted
harmonic, no filter, no Jacobian.  It only (a) names the grid sizes and the tensor layout of
each configuration and (b) draws smooth random scalar functions on the grid (each stored
Cartesian component is an independent scalar field), using its own textbook
recurrence for ordinary normalised associated Legendre functions and Chebyshev polynomials.
The paper's workload (the 50-field GHG state of a single black hole) is
not a public dataset; these fields take its SHAPE and stand in for it.
"""
from .configs import CONFIGS, config, ghg_tensors, wave_tensors, tensor_ncomp  # noqa: F401
from .fields import make_state, scalar_basis, white_state  # noqa: F401
from .wave import wave_exact  # noqa: F401
from .ghg import grid_xyz, kerr_schild_metric, minkowski_metric, perturbed_ghg_state  # noqa: F401
