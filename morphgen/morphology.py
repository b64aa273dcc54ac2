"""Seeded synthetic dendrite morphologies (topology only: parent arrays).

Stand-in for the paper's ring-network benchmark (§7: "all dendritic
trees are created with a specific number of levels. On each level branches are
split into two child branches with a predefined probability. If a branch does
not split it will just continue on the next level"), which is not available.
Numbering follows PAPER.md:44-50 / :149: branches breadth-first from the root,
compartments contiguous per branch and ordered by distance from the root, so
each branch is one tridiagonal block and ``parent[i] < i``.

``parent`` holds CELL-LOCAL indices (root = -1); cells are concatenated and
delimited by ``cell_offsets`` (int64, ncells+1).

Nothing in here performs any step of the Hines solve.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import rng


@dataclass
class Morphology:
    parent: np.ndarray            # int32 [N], cell-local, root -1
    cell_offsets: np.ndarray      # int64 [ncells+1]
    # generator-side branch table (what the generator intended; the canonical
    # branch rule of the plan may merge a single child numbered right after its
    # parent, reading S4) -- used only by tests of the generator.
    gen_branch_len: np.ndarray | None = None      # int32 [nbranches]
    gen_branch_cell: np.ndarray | None = None     # int64 [nbranches]
    gen_branch_level: np.ndarray | None = None    # int32 [nbranches]
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.cell_offsets[-1])

    @property
    def ncells(self) -> int:
        return len(self.cell_offsets) - 1


def cables(ncells: int, length: int) -> Morphology:
    """Unbranched cables: p[i] = i-1 (config 1, the degenerate single-branch case)."""
    one = np.arange(-1, length - 1, dtype=np.int32)
    parent = np.tile(one, ncells)
    offs = np.arange(ncells + 1, dtype=np.int64) * length
    return Morphology(parent, offs,
                      gen_branch_len=np.full(ncells, length, np.int32),
                      gen_branch_cell=np.arange(ncells, dtype=np.int64),
                      gen_branch_level=np.zeros(ncells, np.int32),
                      name=f"cables_{ncells}x{length}")


def complete_binary(ncells: int, nlevels: int, branch_len: int) -> Morphology:
    """Complete binary branch tree, ``nlevels`` levels (2^nlevels - 1 branches),
    every branch ``branch_len`` compartments (configs 0 and 4)."""
    nb = (1 << nlevels) - 1
    n = nb * branch_len
    j = np.arange(nb, dtype=np.int64)
    parent = np.arange(-1, n - 1, dtype=np.int64)
    # first compartment of branch j>0 hangs off the last compartment of branch (j-1)//2
    parent[j[1:] * branch_len] = ((j[1:] - 1) // 2) * branch_len + (branch_len - 1)
    parent = parent.astype(np.int32)
    level = np.floor(np.log2(j + 1)).astype(np.int32)
    offs = np.arange(ncells + 1, dtype=np.int64) * n
    return Morphology(np.tile(parent, ncells), offs,
                      gen_branch_len=np.full(nb * ncells, branch_len, np.int32),
                      gen_branch_cell=np.repeat(np.arange(ncells, dtype=np.int64), nb),
                      gen_branch_level=np.tile(level, ncells),
                      name=f"binary_{ncells}x{nlevels}lv x{branch_len}")


def random_trees(ncells: int, nlevels, q: float, maxlen, seed: int = rng.BASE_SEED,
                 cell_id_base: int = 0, name: str = "random") -> Morphology:
    """Random dendrites by the paper's split-or-continue recipe.

    Every cell has ``nlevels[c]`` levels (depth 0 .. nlevels-1).  A branch at depth
    < nlevels-1 gets two children with probability ``q`` and one child (it
    "continues on the next level") otherwise.  Branch lengths are U{1..maxlen[c]}.
    ``nlevels`` and ``maxlen`` may be scalars or per-cell arrays.
    Decisions are keyed by (cell id, heap-style node id), so a cell's tree does not
    depend on how many other cells are generated.
    """
    nlevels = np.broadcast_to(np.asarray(nlevels, dtype=np.int64), (ncells,))
    maxlen = np.broadcast_to(np.asarray(maxlen, dtype=np.int64), (ncells,))
    lmax = int(nlevels.max())

    # frontier of the current level, kept sorted by (cell, position in level)
    cell = np.arange(ncells, dtype=np.int64)
    node = np.ones(ncells, dtype=np.int64)            # heap-style id, root = 1
    pref = np.full(ncells, -1, dtype=np.int64)        # index into the previous level's arrays
    lv_cell, lv_node, lv_pref = [], [], []
    for lev in range(lmax):
        lv_cell.append(cell); lv_node.append(node); lv_pref.append(pref)
        if lev == lmax - 1 or cell.size == 0:
            break
        key = ((cell + cell_id_base) << np.int64(32)) | node
        r = rng.uniform01(seed, rng.STREAM_TOPOLOGY, key)
        nchild = np.where(r < q, 2, 1).astype(np.int64)
        nchild[lev >= nlevels[cell] - 1] = 0
        idx = np.repeat(np.arange(cell.size, dtype=np.int64), nchild)
        first = np.cumsum(nchild) - nchild                        # first child slot per parent
        which = np.arange(idx.size, dtype=np.int64) - first[idx]  # 0 or 1
        cell, node, pref = cell[idx], 2 * node[idx] + which, idx

    nper = [a.size for a in lv_cell]
    base = np.concatenate([[0], np.cumsum(nper)])[:-1]
    all_cell = np.concatenate(lv_cell)
    all_node = np.concatenate(lv_node)
    all_level = np.concatenate([np.full(n, l, np.int64) for l, n in enumerate(nper)])
    all_pold = np.concatenate([np.where(p >= 0, p + (base[l - 1] if l > 0 else 0), -1)
                               for l, p in enumerate(lv_pref)])
    # breadth-first numbering per cell: order by (cell, level, position); positions are
    # already in order inside each level, so a stable sort by (cell, level) does it.
    order = np.argsort(all_cell * lmax + all_level, kind="stable")
    inv = np.empty_like(order); inv[order] = np.arange(order.size)
    b_cell = all_cell[order]; b_node = all_node[order]; b_level = all_level[order]
    b_parent = np.where(all_pold[order] >= 0, inv[np.maximum(all_pold[order], 0)], -1)  # global branch id

    key = ((b_cell + cell_id_base) << np.int64(32)) | b_node
    ul = rng.uniform01(seed, rng.STREAM_LENGTH, key)
    b_len = 1 + np.floor(ul * maxlen[b_cell]).astype(np.int64)
    b_len = np.minimum(b_len, maxlen[b_cell])

    b_start = np.cumsum(b_len) - b_len                              # global compartment index
    n = int(b_len.sum())
    cell_size = np.bincount(b_cell, weights=b_len, minlength=ncells).astype(np.int64)
    offs = np.concatenate([[0], np.cumsum(cell_size)]).astype(np.int64)

    comp_cell_off = np.repeat(offs[:-1], cell_size)
    parent = np.arange(n, dtype=np.int64) - 1 - comp_cell_off       # local i-1
    del comp_cell_off
    nonroot = b_parent >= 0
    pb = b_parent[nonroot]
    parent[b_start[nonroot]] = (b_start[pb] + b_len[pb] - 1) - offs[b_cell[nonroot]]
    parent[b_start[~nonroot]] = -1
    return Morphology(parent.astype(np.int32), offs,
                      gen_branch_len=b_len.astype(np.int32),
                      gen_branch_cell=b_cell, gen_branch_level=b_level.astype(np.int32),
                      name=name)


def concat(morphs, name="concat") -> Morphology:
    parent = np.concatenate([m.parent for m in morphs])
    sizes = np.concatenate([np.diff(m.cell_offsets) for m in morphs])
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    return Morphology(parent, offs, name=name)
