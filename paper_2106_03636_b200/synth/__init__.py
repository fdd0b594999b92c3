"""Seeded synthetic inputs shared by the CPU oracle tests and the CUDA path (no tracker arithmetic)."""
from .params import KB, N_ROWS, SECTORS_PER_SIDE, V_DRIFT, TpcParams, default_row_x
from .generator import (Event, config0, config1, config2, config3, config4, make_config, single_helix,
                        choose_cells)
from .digitizer import Digits, digitize

__all__ = ["KB", "N_ROWS", "SECTORS_PER_SIDE", "V_DRIFT", "TpcParams", "default_row_x", "Event", "config0",
           "config1", "config2", "config3", "config4", "make_config", "single_helix", "choose_cells", "Digits", "digitize"]
