"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

Holds none of the method's arithmetic (see configs.py).
"""
from . import rng  # noqa: F401
from .configs import *  # noqa: F401,F403
from .networks import *  # noqa: F401,F403
