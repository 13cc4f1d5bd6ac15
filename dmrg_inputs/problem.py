"""Plain containers for a superblock problem in the LR strategy.

An operator of an enlarged block is kept as a list of dense blocks
``A_{q_i -> q_j}``: block ``b`` maps sector ``src[b]`` to sector
``dst[b]`` and has shape ``dims[dst[b]] x dims[src[b]]`` (row-major).
No arithmetic of the method lives here.
"""
from __future__ import annotations
from dataclasses import dataclass, field
from typing import Dict, List
import numpy as np

HEISENBERG = "heisenberg"
HUBBARD = "hubbard"


@dataclass
class Sectors:
    """Quantum-number sectors of one enlarged block."""
    labels: np.ndarray  # [n_sectors, n_labels] int32 (1 label: Sz units; 2 labels: N_up, N_dn)
    dims: np.ndarray    # [n_sectors] int32, >= 0

    def __post_init__(self):
        self.labels = np.ascontiguousarray(np.asarray(self.labels, dtype=np.int32).reshape(len(self.dims), -1))
        self.dims = np.ascontiguousarray(np.asarray(self.dims, dtype=np.int32))

    @property
    def n_sectors(self) -> int:
        return int(self.dims.shape[0])

    @property
    def n_labels(self) -> int:
        return int(self.labels.shape[1])

    @property
    def total_dim(self) -> int:
        return int(self.dims.sum())


@dataclass
class BlockOp:
    """Sector-blocked operator: dense blocks ``A_{src->dst}``."""
    src: List[int] = field(default_factory=list)
    dst: List[int] = field(default_factory=list)
    blocks: List[np.ndarray] = field(default_factory=list)

    def add(self, src: int, dst: int, block: np.ndarray) -> None:
        self.src.append(int(src))
        self.dst.append(int(dst))
        self.blocks.append(np.ascontiguousarray(block, dtype=np.float64))

    @property
    def n_blocks(self) -> int:
        return len(self.blocks)

    def n_elements(self) -> int:
        return int(sum(b.size for b in self.blocks))


@dataclass
class Problem:
    """Everything `dmrg_plan_create` is told (include/dmrg_b200.h, struct dmrg_problem).

    Heisenberg operator names: H_L, H_R, Sz_L, Sp_L, Sz_R, Sp_R  (S- = (S+)^T implied).
    Hubbard operator names:    H_L, H_R, Cup_L, Cdn_L, Cup_R, Cdn_R (c^dagger of the
    boundary site with block-local strings; c = transpose implied) and optional
    D_L, D_R (sum_j n_up n_dn of the block, entering as U*(D_L (x) I + I (x) D_R)).
    """
    model: str
    J: float
    Delta: float
    t: float
    U: float
    left: Sectors
    right: Sectors
    ops: Dict[str, BlockOp]
    target: np.ndarray  # [n_labels] int32

    def __post_init__(self):
        self.target = np.ascontiguousarray(np.asarray(self.target, dtype=np.int32).reshape(-1))

    def op(self, name: str) -> BlockOp:
        return self.ops.get(name, BlockOp())
