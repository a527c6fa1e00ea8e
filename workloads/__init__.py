"""Seeded synthetic input generators shared by the oracle tests and the CUDA path (no DG arithmetic)."""
from .configs import (CONFIGS, SWEEP5, SEED0, TABLE1, base_params, config1, config2, config3, config4, config5,
                      conserved, lgl_nodes, min_node_spacing, node_coords, sound_speed_max)
