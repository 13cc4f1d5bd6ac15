"""O-REC: block-wise projection, one operation record at a time.  TEST INFRASTRUCTURE.

X'_jl += c * A_{alpha,i->j} X_ik B_{alpha,k->l}^T     (Eq. 11)
over every term alpha and every admissible transition pair (L165), with library matmul.
Also diag(H_SB) for the Davidson preconditioner (A14) and the FLOP convention (A24).
Written independently of oracle.kron (per-block coefficients instead of a dense P_L).
"""
from __future__ import annotations
import numpy as np
from dmrg_inputs.problem import Problem, BlockOp, HEISENBERG, HUBBARD


class Layout:
    """Flat-vector layout of the target sector (A1, A5): pairs sorted by (left, right) sector
    index; each segment row-major d_i x d_k."""

    def __init__(self, p: Problem):
        L, R = p.left, p.right
        self.pairs, self.offset = [], []
        self.index = {}
        n = 0
        for i in range(L.n_sectors):
            for k in range(R.n_sectors):
                if L.dims[i] > 0 and R.dims[k] > 0 and np.array_equal(L.labels[i] + R.labels[k], p.target):
                    self.index[(i, k)] = len(self.pairs)
                    self.pairs.append((i, k))
                    self.offset.append(n)
                    n += int(L.dims[i]) * int(R.dims[k])
        self.n = n
        self.dl, self.dr = L.dims, R.dims

    def seg(self, x: np.ndarray, i: int, k: int) -> np.ndarray:
        o = self.offset[self.index[(i, k)]]
        return x[o:o + int(self.dl[i]) * int(self.dr[k])].reshape(int(self.dl[i]), int(self.dr[k]))


def _identity_like(n_sectors) -> list:
    return [(s, s, None) for s in range(n_sectors)]


def _blocks(op: BlockOp) -> list:
    return list(zip(op.src, op.dst, op.blocks))


def _transposed(op: BlockOp) -> list:
    return [(d, s, b.T) for s, d, b in zip(op.src, op.dst, op.blocks)]


def block_terms(p: Problem):
    """List of (coef_fn(i, j), A_blocks, B_blocks): blocks are (src, dst, matrix|None=identity);
    coef_fn gets the left input/output sector so the fermion sign of A6 is a per-record scalar:
    -t*(-1)^{N(q_i)} for c+_L c_R (input left sector), -t*(-1)^{N(q_j)} for its h.c. (output)."""
    nL, nR = p.left.n_sectors, p.right.n_sectors
    one = lambda i, j: 1.0
    T = [(one, _blocks(p.op("H_L")), _identity_like(nR)), (one, _identity_like(nL), _blocks(p.op("H_R")))]
    if p.model == HEISENBERG:
        half = lambda i, j: 0.5 * p.J
        T.append((half, _blocks(p.op("Sp_L")), _transposed(p.op("Sp_R"))))
        T.append((half, _transposed(p.op("Sp_L")), _blocks(p.op("Sp_R"))))
        T.append((lambda i, j: p.J * p.Delta, _blocks(p.op("Sz_L")), _blocks(p.op("Sz_R"))))
    elif p.model == HUBBARD:
        NL = p.left.labels.sum(axis=1)
        s_in = lambda i, j: -p.t * (1.0 if NL[i] % 2 == 0 else -1.0)
        s_out = lambda i, j: -p.t * (1.0 if NL[j] % 2 == 0 else -1.0)
        for nm in ("Cup", "Cdn"):
            T.append((s_in, _blocks(p.op(nm + "_L")), _transposed(p.op(nm + "_R"))))
            T.append((s_out, _transposed(p.op(nm + "_L")), _blocks(p.op(nm + "_R"))))
        uu = lambda i, j: p.U
        if p.op("D_L").n_blocks:
            T.append((uu, _blocks(p.op("D_L")), _identity_like(nR)))
        if p.op("D_R").n_blocks:
            T.append((uu, _identity_like(nL), _blocks(p.op("D_R"))))
    else:
        raise ValueError(p.model)
    return T


def records(p: Problem, lay: Layout | None = None):
    """Operation records: (c, A|None, B|None, (i,k) input, (j,l) output)."""
    lay = lay or Layout(p)
    recs = []
    for coef, Ab, Bb in block_terms(p):
        for (i, j, A) in Ab:
            for (k, l, B) in Bb:
                if (i, k) in lay.index and (j, l) in lay.index:
                    recs.append((coef(i, j), A, B, (i, k), (j, l)))
    return recs


def apply_blockwise(p: Problem, x: np.ndarray, lay: Layout | None = None, recs=None) -> np.ndarray:
    """y = H_SB x by Eq. 11, record by record."""
    lay = lay or Layout(p)
    recs = recs if recs is not None else records(p, lay)
    y = np.zeros(lay.n)
    for c, A, B, (i, k), (j, l) in recs:
        X = lay.seg(x, i, k)
        T = X if A is None else A @ X
        T = T if B is None else T @ B.T
        lay.seg(y, j, l)[...] += c * T
    return y


def diag_H(p: Problem, lay: Layout | None = None) -> np.ndarray:
    """diag(H_SB) on the target sector (A14): only records with (i,k) == (j,l) contribute,
    D[(i,k)][a,b] += c * A_aa * B_bb (identity factor -> 1)."""
    lay = lay or Layout(p)
    D = np.zeros(lay.n)
    for c, A, B, (i, k), (j, l) in records(p, lay):
        if (i, k) != (j, l):
            continue
        da = np.ones(int(lay.dl[i])) if A is None else np.diag(A).copy()
        db = np.ones(int(lay.dr[k])) if B is None else np.diag(B).copy()
        lay.seg(D, i, k)[...] += c * np.outer(da, db)
    return D


def flop_count(p: Problem, lay: Layout | None = None) -> int:
    """Algorithmic FLOP per apply (A24): per record min over the two association orders;
    identity-factor records are one GEMM."""
    lay = lay or Layout(p)
    tot = 0
    for c, A, B, (i, k), (j, l) in records(p, lay):
        di, dk, dj, dl_ = int(lay.dl[i]), int(lay.dr[k]), int(lay.dl[j]), int(lay.dr[l])
        if A is None:
            tot += 2 * di * dk * dl_
        elif B is None:
            tot += 2 * dj * di * dk
        else:
            tot += min(2 * dj * di * dk + 2 * dj * dk * dl_, 2 * di * dk * dl_ + 2 * dj * di * dl_)
    return tot
