"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

Holds no step arithmetic; see workloads/model.py.
"""
from .model import *  # noqa: F401,F403
from . import configs  # noqa: F401
