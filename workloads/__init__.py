"""Seeded synthetic input generators shared by the oracle and the CUDA path (no method arithmetic here)."""
from .configs import make_problem, loss_and_seed, rest_length, subset, FULL_SIZES  # noqa: F401
