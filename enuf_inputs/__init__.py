"""Seeded synthetic workloads for the ENUF reciprocal-space path.

This module holds *inputs only*: positions, charges and the literal plan
parameters of the five BASELINE.json configs.  It holds none
of the method's arithmetic (no window, no Ewald kernel, no FFT) and imports
neither the CUDA package nor ``oracle/``; both sides read the same arrays.

Stand-ins: the paper's own inputs (the +-1 lattice of PAPER.md:467, the DPD
electrolyte of PAPER.md:471-483, the coarse-grained ionic liquids of
PAPER.md:523) are not available; these seeded generators reproduce their
shape, size, charge pattern and density structure.

Random numbers: SplitMix64 used as a counter-based generator,
``x_i = mix(seed + (i + 1) * GOLDEN)``, ``U = (x >> 11) * 2**-53`` in [0, 1);
Gaussians by Box-Muller.  Values are drawn particle-major, dimension-minor,
generated in fp64 and rounded once to the config's precision.
"""
from .workloads import (  # noqa: F401
    CONFIGS,
    Workload,
    make_workload,
    splitmix64,
    uniform01,
    displaced_positions,
    random_neutral_gas,
)
