"""Seeded synthetic particle sets for the CRKSPH hot path (test/bench tooling).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2202_02840_b200``).  It holds none of the method's arithmetic: no SPH
kernel, no volumes, no reproducing-kernel coefficients, no forces.  It only
draws positions / velocities / energies from seeded counter-based streams
(numpy Philox; the paper uses counter-based Threefry for the same reason,
PAPER.md:338) and assigns a support radius ``h`` from *generator-side*
knowledge of the number density (lattice spacing, k-th neighbour distance, or
the Zel'dovich Jacobian) -- never from the oracle or the CUDA path.

Recipes follow BASELINE.json ``configs`` / SURVEY.md section 8(d); every reading
is listed in DESIGN.md ("Input recipe").  All outputs are float32 SoA arrays,
positions in [0, box), box = 1, gamma = 5/3, equal masses m = 1/N,
n_h = 2.4  (h is the SUPPORT radius: W = 0 for r >= h).
"""
from .generators import (  # noqa: F401
    ParticleSet,
    N_H,
    tiny_uniform,
    blast_wave,
    clustered_plummer,
    zeldovich,
    make_config,
    select_window,
    CONFIG_NAMES,
)
