"""Seeded synthetic workload generators (test/bench infrastructure).

This package holds NONE of the multigrid arithmetic: it only produces the input
buffers (density rho, right-hand side rhs, and for config 1 the known solution)
that are handed, unchanged, to both the CPU oracle (`oracle/`) and the CUDA path
(`paper_2605_30082_b200/`).  Neither of those imports the other; both are fed
from here.

Recipes: SURVEY.md §8(d) (configs 1-5 of BASELINE.json), standing in for the
paper's FS3D fields (PAPER.md:75-77 drop + film + air box, PAPER.md:190
oscillating droplet, PAPER.md:196/218 512^3 cells per device), which are not
available.
"""
from .configs import (  # noqa: F401
    CONFIGS,
    Workload,
    make_workload,
    sequence_density,
    splitmix64_uniform,
    velocity_field,
)
