"""nbgen -- seeded synthetic star-cluster inputs (shared by the oracle tests and the CUDA path).

This module only SYNTHESISES inputs: particle masses, positions, velocities, block levels,
reference times, active-index blocks and neighbour radii with the shapes of the paper's
workloads (Plummer / King models, Kroupa IMF, 5 % binaries as centre-of-mass bodies, deep
hierarchical block steps -- PAPER.md P:89; BASELINE.json configs 1-5).

It holds NONE of the method's arithmetic: no predictor, no pairwise force / jerk / potential
sum, no neighbour classification.  It imports neither ``oracle`` nor the CUDA package, and
neither of those imports the other.  Where a config needs method results as *inputs*
(config 1: a0/j0 from a full direct sum, h^2 from the 48th nearest neighbour at the predicted
positions) the caller computes them with whichever side it is testing and passes them in.

Every random draw comes from ``numpy.random.Generator(Philox)`` keyed by (seed, stream) so
that changing one piece never shifts the others.
"""
from .cluster import (  # noqa: F401
    STREAMS,
    substream,
    plummer_positions,
    plummer_velocities,
    plummer_model,
    plummer_smooth_field,
    plummer_number_density,
    kroupa_masses,
    merge_binaries,
    KingModel,
    king_sample,
    block_levels_uniform,
    block_levels_powerlaw,
    t0_from_levels,
    h2_from_density,
    knn_radius2,
    center_of_mass_frame,
)
from .configs import make_config, finish_config1, active_block, CONFIG_NAMES, shard_active_block  # noqa: F401
