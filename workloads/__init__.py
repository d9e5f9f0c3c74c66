"""Seeded synthetic inputs for the epoch-substitution-model hot path.

This package is the ONLY artefact shared by the CPU oracle (``oracle/``) and the
CUDA product (``paper_1309_3075_b200/``).  It holds input generators and nothing
of the method's arithmetic: no matrix exponential, no segmenter, no pruning.
It imports neither of the two.
"""
from .problem import EpochProblem
from .configs import make_config, CONFIG_NAMES, config_seed
from . import models, trees

__all__ = ["EpochProblem", "make_config", "CONFIG_NAMES", "config_seed", "models", "trees"]
