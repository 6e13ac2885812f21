"""Seeded synthetic inputs for the ZDA zone solver (shared by oracle and CUDA path; inputs only)."""
from .zone_inputs import DensityMap, ZoneInputs  # noqa: F401
from .configs import (config1, config2, config3, config4, config5_zones, config6_thin_wedge, config7_first_zone, cut_down,  # noqa: F401
                      courant_dt, courant_dt_one_phi_cell, cpml_sigma_max, focal_point_weights, gaussian_pulse_table, plane_wave_sheet, window)
