"""Seeded synthetic inputs for the COMET seed x hit scan (arXiv 1911.09340).

This module only *makes inputs*: a stand-in drift-chamber geometry, truth
electrons on a closed-form helix, drift-radius hits with left/right ghosts and
the seed grids of BASELINE.json's five configs.  It holds none of the method's
arithmetic (no RKN stepping, no closest-point search, no RSS): both the CPU
oracle (`oracle/`) and the CUDA path (`paper_1911_09340_b200/`) consume what it
produces, and neither imports the other.

Units: cm, MeV/c, Tesla, charge in units of e.
"""
from .geometry import cdc_geometry, CDCGeometry
from .helix import Helix, KAPPA
from .events import (Event, Partition, make_event, make_config, config_spec,
                     seed_grid, event_seeds, truth_seed, CONFIG_SPECS,
                     seed_axes, pack_axes, grid_from_axes, event_axes)
from .fieldmap import solenoid_map, uniform_map, hough_tables

__all__ = [
    "cdc_geometry", "CDCGeometry", "Helix", "KAPPA", "Event", "Partition",
    "make_event", "make_config", "config_spec", "seed_grid", "event_seeds", "seed_axes", "pack_axes", "grid_from_axes", "event_axes",
    "truth_seed", "CONFIG_SPECS", "solenoid_map", "uniform_map", "hough_tables",
]
