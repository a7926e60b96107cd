"""Seeded synthetic inputs (random streams, Plummer sampler, the five configs).  Shared by tests,
bench.py and smoke(); holds none of the method's arithmetic."""
from .configs import Case, config1, config2, config3, config4, config5, sample_positions, SEED0
from .plummer import HENON_A, mean_field, plummer
from .rng import Streams, integers, permutation

__all__ = ["Case", "config1", "config2", "config3", "config4", "config5", "sample_positions",
           "SEED0", "HENON_A", "mean_field", "plummer", "Streams", "integers", "permutation"]
