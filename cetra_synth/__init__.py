"""Seeded synthetic inputs for the CETRA hot path (tests, bench, smoke).

This module serves both the CPU oracle and the CUDA path and therefore holds
NONE of the method's arithmetic (no weights, no windowed sums, no folding):
it only draws light curves, builds the tabulated transit profile that the
library takes as an *input*, and lays out the trial grids.  The recipe is the
one SURVEY.md §8(d) fixes for BASELINE.json's five configs; it is restated in
DESIGN.md §"Input recipe".

No TESS files, Batman models or TLS grids are in the container: these inputs
stand in for them (PAPER.md:65-69 for the model, PAPER.md:226 for the cadences).
"""
from .lightcurves import (  # noqa: F401
    SearchProblem,
    transit_profile,
    tabulate_template,
    make_config,
    make_survey_batch,
    make_irregular_batch,
    duration_grid,
    period_grid_uniform_frequency,
    CONFIG_NAMES,
)
