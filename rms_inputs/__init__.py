"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path.

This package holds NO arithmetic of the method (no random walk, no permeation
probability, no phase, no reduction): only label lattices, physical parameter
tables, gradient waveforms and direction sets, i.e. the *arguments* of the
three C-ABI calls.  Recipes are stated in DESIGN.md ("Input recipe") and follow
BASELINE.json:configs / SURVEY.md section 8(d).  The paper's own substrate (an EM
segmentation of 227 mouse corpus-callosum axons) is not
available; `axon_substrate` stands in for it.
"""
from .substrates import (  # noqa: F401
    Substrate,
    single_cylinder,
    packed_cylinders,
    axon_substrate,
    plates,
    slabs,
    random_lattice,
    uniform_lattice,
)
from .sequences import pgse_wave, pgse_gamp, one_hot_wave, fibonacci_dirs, Sequence, pgse_sequence  # noqa: F401
from .configs import make_config, CONFIG_NAMES  # noqa: F401
