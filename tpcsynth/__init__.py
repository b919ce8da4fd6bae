"""Seeded synthetic TPC event generator (inputs only; shared by oracle tests and the CUDA path)."""
from .events import (CONFIGS, KB, N_ROWS, NOISE_ID, STREAM_BASE_SEED, Event, EventConfig, Geometry,
                     generate_event, generate_stream, row_x_table)

__all__ = ["CONFIGS", "KB", "N_ROWS", "NOISE_ID", "STREAM_BASE_SEED", "Event", "EventConfig", "Geometry",
           "generate_event", "generate_stream", "row_x_table"]
