"""Seeded synthetic inputs shared by the oracle tests and the CUDA path (no method arithmetic here)."""
from . import configs, meshes, prng, states  # noqa: F401
from .configs import MODEL_CRN98, MODEL_STEWART, MODEL_TP06, Problem, Stimulus, make  # noqa: F401
from .meshes import TetMesh, TriMesh  # noqa: F401
