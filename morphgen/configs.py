"""The five BASELINE.json workloads as seeded synthetic morphologies.

``scale`` shrinks the number of cells (configs 0-3) or the number of levels is
left alone and only cells are scaled; ``scale=1`` is the full BASELINE size.
The recipe (levels, split probability q, length ranges) is the one calibrated in
SURVEY.md §8(d) against BASELINE.json's stated sizes; see DESIGN.md.
"""
from __future__ import annotations

import numpy as np

from . import rng
from .morphology import Morphology, cables, complete_binary, random_trees

Q_SPLIT = 0.40

CONFIG_NAMES = {
    0: "cfg0: 64 cells x balanced binary dendrite, 15 branches x 5 compartments",
    1: "cfg1: 10,000 unbranched cables x 1,000 compartments",
    2: "cfg2: 10,000 random dendrites (13 levels, q=0.40, branch length U{1..40})",
    3: "cfg3: 65,536 heterogeneous cells (80% small ~200, 20% large ~10,000 unknowns)",
    4: "cfg4: 1 cell, complete binary branch tree of 17 levels x 10 compartments",
}


def _scaled(n: int, scale: float) -> int:
    return max(1, int(round(n * scale)))


def make_config(cfg: int, scale: float = 1.0, seed: int = rng.BASE_SEED) -> Morphology:
    if cfg == 0:
        m = complete_binary(_scaled(64, scale), 4, 5)
    elif cfg == 1:
        m = cables(_scaled(10_000, scale), 1000)
    elif cfg == 2:
        m = random_trees(_scaled(10_000, scale), 13, Q_SPLIT, 40, seed, name="cfg2")
    elif cfg == 3:
        nc = _scaled(65_536, scale)
        cls = rng.uniform01(seed, rng.STREAM_CLASS, np.arange(nc, dtype=np.uint64)) < 0.2
        nlevels = np.where(cls, 13, 7)
        maxlen = np.where(cls, 100, 16)
        m = random_trees(nc, nlevels, Q_SPLIT, maxlen, seed + 3, name="cfg3")
        m.meta["large"] = cls
    elif cfg == 4:
        m = complete_binary(1, 17, 10)
    else:
        raise ValueError(f"unknown config {cfg}")
    m.name = CONFIG_NAMES[cfg] + (f" [scale {scale:g}]" if scale != 1.0 else "")
    m.meta["cfg"] = cfg
    m.meta["scale"] = scale
    return m
