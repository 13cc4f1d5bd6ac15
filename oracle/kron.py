"""O-KRON: the definition.  TEST INFRASTRUCTURE.

H_SB = sum_alpha c_alpha  A_alpha (x) B_alpha   (Eq. 9), composite index
a*m_R + b (left index slow: reading A1), restricted to the target sector Q
(PAPER.md:L94, L118).  Dense; for m_L*m_R up to ~2e4.
"""
from __future__ import annotations
import numpy as np
from dmrg_inputs.problem import Problem, BlockOp, Sectors, HEISENBERG, HUBBARD


def dense_op(op: BlockOp, sec: Sectors) -> np.ndarray:
    """Scatter the sector blocks of one operator into a dense m x m matrix."""
    off = np.concatenate([[0], np.cumsum(sec.dims)])
    m = int(off[-1])
    O = np.zeros((m, m))
    for s, d, blk in zip(op.src, op.dst, op.blocks):
        assert blk.shape == (sec.dims[d], sec.dims[s])
        O[off[d]:off[d + 1], off[s]:off[s + 1]] += blk
    return O


def state_labels(sec: Sectors) -> np.ndarray:
    return np.repeat(sec.labels, sec.dims, axis=0)


def terms_dense(p: Problem):
    """(c_alpha, A_alpha, B_alpha) of Eq. 9 -- the enumeration the paper leaves implicit (A3).

    Heisenberg (Eq. 1 split at the L|R bond, overall J: A2):
        H_L (x) I,  I (x) H_R,  J/2 S+_L (x) S-_R,  J/2 S-_L (x) S+_R,  J*Delta Sz_L (x) Sz_R.
    Hubbard (Eq. 4 split at the bond; A6): a right-block operator carries the Phi-string over
    the whole left block, c_R^full = P_L (x) c_R with P_L = (-1)^{N_L}, hence
        -t (c+_L P_L) (x) c_R   and its transpose  -t (P_L c_L) (x) c+_R   per polarisation;
    optional  U D_L (x) I,  U I (x) D_R  (A7)."""
    L, R = p.left, p.right
    IL, IR = np.eye(L.total_dim), np.eye(R.total_dim)
    HL, HR = dense_op(p.op("H_L"), L), dense_op(p.op("H_R"), R)
    out = [(1.0, HL, IR), (1.0, IL, HR)]
    if p.model == HEISENBERG:
        SpL, SpR = dense_op(p.op("Sp_L"), L), dense_op(p.op("Sp_R"), R)
        SzL, SzR = dense_op(p.op("Sz_L"), L), dense_op(p.op("Sz_R"), R)
        out += [(0.5 * p.J, SpL, SpR.T), (0.5 * p.J, SpL.T, SpR), (p.J * p.Delta, SzL, SzR)]
    elif p.model == HUBBARD:
        PL = np.diag((-1.0) ** state_labels(L).sum(axis=1))
        for nm in ("Cup", "Cdn"):
            cL, cR = dense_op(p.op(nm + "_L"), L), dense_op(p.op(nm + "_R"), R)
            out += [(-p.t, cL @ PL, cR.T), (-p.t, PL @ cL.T, cR)]
        if p.op("D_L").n_blocks:
            out.append((p.U, dense_op(p.op("D_L"), L), IR))
        if p.op("D_R").n_blocks:
            out.append((p.U, IL, dense_op(p.op("D_R"), R)))
    else:
        raise ValueError(p.model)
    return out


def H_full(p: Problem) -> np.ndarray:
    """Eq. 9 on the whole m_L*m_R product space."""
    mL, mR = p.left.total_dim, p.right.total_dim
    H = np.zeros((mL * mR, mL * mR))
    for c, A, B in terms_dense(p):
        H += c * np.kron(A, B)
    return H


def target_index(p: Problem) -> np.ndarray:
    """Composite indices a*m_R + b of the target sector in the canonical flat-vector order:
    pairs (i,k) ascending in (left sector, right sector) index, inside a pair the d_i x d_k
    segment row-major, left index slow (A1, A5)."""
    L, R = p.left, p.right
    offL = np.concatenate([[0], np.cumsum(L.dims)])
    offR = np.concatenate([[0], np.cumsum(R.dims)])
    mR = R.total_dim
    idx = []
    for i in range(L.n_sectors):
        for k in range(R.n_sectors):
            if np.array_equal(L.labels[i] + R.labels[k], p.target) and L.dims[i] > 0 and R.dims[k] > 0:
                a = np.arange(offL[i], offL[i + 1])
                b = np.arange(offR[k], offR[k + 1])
                idx.append((a[:, None] * mR + b[None, :]).ravel())
    return np.concatenate(idx) if idx else np.zeros(0, dtype=np.int64)


def H_sector(p: Problem):
    """(P_Q H P_Q^T, leakage) where leakage = max |H| element connecting the target sector to
    its complement (must be 0: H is block-diagonal in Q)."""
    H = H_full(p)
    idx = target_index(p)
    comp = np.setdiff1d(np.arange(H.shape[0]), idx)
    leak = float(np.abs(H[np.ix_(idx, comp)]).max()) if comp.size and idx.size else 0.0
    return H[np.ix_(idx, idx)], leak


def apply_kron(p: Problem, x: np.ndarray) -> np.ndarray:
    Hs, _ = H_sector(p)
    return Hs @ x
