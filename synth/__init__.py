"""Seeded synthetic inputs (filterbanks, config shapes) shared by oracle tests and CUDA tests/bench.
Holds none of the search method's arithmetic."""
from . import configs, filterbank  # noqa: F401
