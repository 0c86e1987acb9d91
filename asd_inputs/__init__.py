"""Seeded synthetic inputs for the atomistic spin-dynamics (ASD) window of arXiv 2502.02236.

This module serves BOTH the fp64 oracle (oracle/) and the CUDA library (paper_2502_02236_b200/):
it produces lattice descriptions, grain maps, temperature / field profiles, initial spins and the
drive schedule as plain numpy arrays.  It holds NONE of the method's arithmetic (no LLG, no field
evaluation, no Philox, no Box-Muller, no cone sampling) and imports neither side.

The inputs stand in for the paper's workload (a 60 nm-wide granular FePt track of 8 nm Voronoi
grains written with 20 nm bits under a moving Gaussian laser spot);
the paper's own track realisation is not available.  The recipes are BASELINE.json configs[0..4]
with the readings Q7-Q13 of SURVEY.md section 8(c), restated in DESIGN.md section 4.
"""
from .workloads import (  # noqa: F401
    shell_ell_table,
    GAMMA_E, MU_B, K_B, SC, L10, Workload, voronoi_grain_map, laser_temperature, tilted_spins,
    make_config, small_film, ShiftSchedule, planes_for_shift, nrz_bits, field_scale_at,
)
from .two_track import TwoTrack, two_track_film, drive_pass, read_tracks  # noqa: F401
from . import multiscale  # noqa: F401
from .multiscale import (  # noqa: F401
    Multiscale, multiscale_film, apply_multiscale, cell_grain_map, MultiscaleWrite, multiscale_write, drive_multiscale_write,
)
