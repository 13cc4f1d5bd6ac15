"""O-BLK: exact (untruncated) left/right blocks cut into per-sector dense blocks.  TEST INFRASTRUCTURE.

Left block = first l sites, right block = last r sites of the open chain.  H_L, H_R are
the model on those sites alone; the boundary operators act on the LAST site of L and
the FIRST site of R, with fermionic strings inside their own block only (reading A6).
The product basis of each block is sorted by label (stable in the basis index) and every
operator is cut into dense blocks A_{q_i -> q_j}.
"""
from __future__ import annotations
import numpy as np
from dmrg_inputs.problem import Sectors, BlockOp, Problem, HEISENBERG, HUBBARD
from . import ed


def _sort_basis(labels: np.ndarray):
    """labels [dim, n_labels] -> permutation (stable, lexicographic ascending), sector list."""
    dim = labels.shape[0]
    keys = [tuple(int(v) for v in labels[a]) for a in range(dim)]
    perm = sorted(range(dim), key=lambda a: keys[a])  # Python's sort is stable
    uniq, dims = [], []
    for a in perm:
        if not uniq or uniq[-1] != keys[a]:
            uniq.append(keys[a])
            dims.append(0)
        dims[-1] += 1
    return np.array(perm), np.array(uniq, dtype=np.int32).reshape(len(uniq), -1), np.array(dims, dtype=np.int32)


def _cut(O: np.ndarray, perm: np.ndarray, dims: np.ndarray, tol: float = 0.0) -> BlockOp:
    Os = O[np.ix_(perm, perm)]
    off = np.concatenate([[0], np.cumsum(dims)])
    op = BlockOp()
    for s in range(len(dims)):
        for d in range(len(dims)):
            blk = Os[off[d]:off[d + 1], off[s]:off[s + 1]]
            if np.any(np.abs(blk) > tol):
                op.add(s, d, blk.copy())
    return op


def heisenberg_exact(l: int, r: int, J: float = 1.0, Delta: float = 1.0, target_twice_sz: int = 0) -> Problem:
    """Config 1 of BASELINE.json for l = r = 6.  Labels are 2*S_z (integers for any l)."""
    sides = {}
    for name, n, site in (("L", l, l), ("R", r, 1)):
        lab = ed.heisenberg_twice_sz(n).reshape(-1, 1)
        perm, uniq, dims = _sort_basis(lab)
        sides[name] = (Sectors(uniq, dims),
                       _cut(ed.heisenberg_H(n, J, Delta), perm, dims),
                       _cut(ed.embed(ed.S_Z, site, n), perm, dims),
                       _cut(ed.embed(ed.S_PLUS, site, n), perm, dims))
    (sl, HL, SzL, SpL), (sr, HR, SzR, SpR) = sides["L"], sides["R"]
    return Problem(HEISENBERG, J, Delta, 0.0, 0.0, sl, sr,
                   {"H_L": HL, "H_R": HR, "Sz_L": SzL, "Sp_L": SpL, "Sz_R": SzR, "Sp_R": SpR},
                   np.array([target_twice_sz]))


def hubbard_exact(l: int, r: int, t: float = 1.0, U: float = 4.0, target=None, fold_U: bool = False) -> Problem:
    """Exact Hubbard blocks.  Labels (N_up, N_dn).  With ``fold_U`` the on-site term sits inside
    H_L/H_R and D_L/D_R are absent; otherwise H_L/H_R are the U = 0 blocks and D_L/D_R carry
    sum_j n_up n_dn so that the caller's U multiplies them (reading A7)."""
    sides = {}
    for name, n, site in (("L", l, l), ("R", r, 1)):
        nu, nd = ed.hubbard_counts(n)
        perm, uniq, dims = _sort_basis(np.stack([nu, nd], axis=1))
        H = ed.hubbard_H(n, t, U if fold_U else 0.0)
        ops = dict(H=_cut(H, perm, dims),
                   Cup=_cut(ed.hubbard_mode_op(ed.C_DAG, site, 1, n), perm, dims),
                   Cdn=_cut(ed.hubbard_mode_op(ed.C_DAG, site, 0, n), perm, dims))
        if not fold_U:
            ops["D"] = _cut(ed.hubbard_double_occupancy(n), perm, dims)
        sides[name] = (Sectors(uniq, dims), ops)
    (sl, ol), (sr, orr) = sides["L"], sides["R"]
    ops = {"H_L": ol["H"], "H_R": orr["H"], "Cup_L": ol["Cup"], "Cdn_L": ol["Cdn"],
           "Cup_R": orr["Cup"], "Cdn_R": orr["Cdn"]}
    if not fold_U:
        ops["D_L"], ops["D_R"] = ol["D"], orr["D"]
    N = l + r
    if target is None:
        target = (N // 2, N // 2)
    return Problem(HUBBARD, 0.0, 0.0, t, U, sl, sr, ops, np.array(target))


def block_basis_order(labels: np.ndarray) -> np.ndarray:
    """Permutation used by the builders above (exposed for the RNG-free H*1 pin)."""
    return _sort_basis(labels)[0]
