"""morphgen -- seeded synthetic inputs shared by the oracle tests and the CUDA path.

Holds none of the Hines method's arithmetic: topology (parent arrays) and
coefficient draws only.  Neither ``oracle/`` nor ``paper_1810_12742_b200/``
imports the other; both are fed from here.
"""
from . import rng
from .morphology import Morphology, cables, complete_binary, random_trees, concat
from .coefficients import coefficients, rhs, system, global_parent
from .configs import make_config, CONFIG_NAMES, Q_SPLIT

__all__ = ["rng", "Morphology", "cables", "complete_binary", "random_trees", "concat",
           "coefficients", "rhs", "system", "global_parent", "make_config", "CONFIG_NAMES",
           "Q_SPLIT"]
