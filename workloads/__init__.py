"""Seeded synthetic workloads (harness only).

This package holds the five BASELINE.json configurations and the seeded input
generators that feed BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2308_07277_b200/``) with the same data.  It contains none of the
method's arithmetic: no G-sphere enumeration for wavefunctions, no Hamiltonian
term, no FFT of a wavefunction.  Callers pass in whatever geometry the
generators need (Miller indices, reciprocal vectors) from their own side.
"""
from .configs import CONFIGS, Config, get_config, cell_for  # noqa: F401
from .generators import (  # noqa: F401
    SEED, make_kpoints, make_psi, make_vloc, make_beta, make_dmatrix, rng_for,
)
