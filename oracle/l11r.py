"""O-L11R: the l-1-1-r strategy (Eq. 12-13; Alg. 2).  TEST INFRASTRUCTURE.

    H_SB = sum_alpha A_alpha^(l) (x) a_alpha (x) b_alpha (x) B_alpha^(r)                 (Eq. 12)
    X'   = sum_alpha ProjectX_l11r(A_alpha, a_alpha, b_alpha, B_alpha, X)                (Eq. 13)

with l, r the (un-enlarged) blocks and a, b operators of the two single sites between them.  `project_l11r` is Alg. 2
written out step by step in the paper's order (reshapes in the paper's column-major convention: the index of the RIGHTMOST
Kronecker factor is the fastest, reading A1); line 8 of the listing is lost in the source ("X_3' = X_3 A^T" by the pattern of
lines 3-6).  The operator quadruplets of the spin-1/2 Heisenberg chain (Eq. 1 with the overall J of reading A2) are
enumerated in `terms` (the paper does not list them, reading A3/A35):
    H_l 1 1 1,   1 1 1 H_r,
    J/2 (S+_l S- 1 1 + S-_l S+ 1 1) + J Delta Sz_l Sz 1 1          (bond block l - site 1)
    J/2 (1 S+ S- 1 + 1 S- S+ 1)     + J Delta 1 Sz Sz 1            (bond site 1 - site 2)
    J/2 (1 1 S+ S-_r + 1 1 S- S+_r) + J Delta 1 1 Sz Sz_r          (bond site 2 - block r)
Layout of the target-sector vector (A36): left composite sectors (s, sigma1) in the order index = 2 s + sigma1 (down = 0,
up = 1), right composite sectors (sigma2, s') in the order index = sigma2 * n_r + s'; segments = admissible pairs sorted by
(left index, right index), each the row-major d_l(s) x d_r(s') block -- the LR convention (A5) on the finer sectors.
"""
from __future__ import annotations
import numpy as np
from .kron import dense_op
from .renorm import Block

SZ = np.diag([-0.5, 0.5])                       # site basis (down, up) = labels (-1, +1)
SP = np.array([[0.0, 0.0], [1.0, 0.0]])         # S+ |down> = |up>
I2 = np.eye(2)


def project_l11r(A, B, C, D, X):
    """Alg. 2: X' = (A (x) B (x) C (x) D) X for one matrix quadruplet, by mode products."""
    Ac, Bc, Cc, Dc = A.shape[1], B.shape[1], C.shape[1], D.shape[1]
    Ar, Br, Cr, Dr = A.shape[0], B.shape[0], C.shape[0], D.shape[0]
    # line 2: X1 = reshape(X) as [D^col, C^col, B^col, A^col]   (column-major: D's index fastest)
    X1 = np.reshape(X, (Dc, Cc, Bc, Ac), order="F")
    # line 3: for each (i, j): X1'(:, :, i, j) = D X1(:, :, i, j)
    X1p = np.empty((Dr, Cc, Bc, Ac))
    for i in range(Bc):
        for j in range(Ac):
            X1p[:, :, i, j] = D @ X1[:, :, i, j]
    # line 4: for each (i, j): X1''(:, :, i, j) = X1'(:, :, i, j) C^T
    X1pp = np.empty((Dr, Cr, Bc, Ac))
    for i in range(Bc):
        for j in range(Ac):
            X1pp[:, :, i, j] = X1p[:, :, i, j] @ C.T
    # line 5: X2 = reshape(X1'') as [D^row C^row, B^col, A^col];  line 6: for each i: X2'(:, :, i) = X2(:, :, i) B^T
    X2 = np.reshape(X1pp, (Dr * Cr, Bc, Ac), order="F")
    X2p = np.empty((Dr * Cr, Br, Ac))
    for i in range(Ac):
        X2p[:, :, i] = X2[:, :, i] @ B.T
    # line 7: X3 = reshape(X2') as [D^row C^row B^row, A^col];  line 8: X3' = X3 A^T
    X3 = np.reshape(X2p, (Dr * Cr * Br, Ac), order="F")
    X3p = X3 @ A.T
    # line 9: X' = reshape(X3') as [D^row C^row B^row A^row]
    return np.reshape(X3p, (Dr * Cr * Br * Ar,), order="F")


def terms(l: Block, r: Block, J: float, Delta: float):
    """(coefficient, A^(l), a, b, B^(r)) of Eq. 12 for the Heisenberg chain, dense."""
    Hl, Szl, Spl = dense_op(l.H, l.sectors), dense_op(l.Sz, l.sectors), dense_op(l.Sp, l.sectors)
    Hr, Szr, Spr = dense_op(r.H, r.sectors), dense_op(r.Sz, r.sectors), dense_op(r.Sp, r.sectors)
    Il, Ir = np.eye(Hl.shape[0]), np.eye(Hr.shape[0])
    h = 0.5 * J
    return [(1.0, Hl, I2, I2, Ir), (1.0, Il, I2, I2, Hr),
            (h, Spl, SP.T, I2, Ir), (h, Spl.T, SP, I2, Ir), (J * Delta, Szl, SZ, I2, Ir),
            (h, Il, SP, SP.T, Ir), (h, Il, SP.T, SP, Ir), (J * Delta, Il, SZ, SZ, Ir),
            (h, Il, I2, SP, Spr.T), (h, Il, I2, SP.T, Spr), (J * Delta, Il, I2, SZ, Szr)]


class Layout4:
    """Target sector in the l-1-1-r product basis (A36)."""

    def __init__(self, l: Block, r: Block, target_twice_sz: int):
        nl, nr = l.sectors.n_sectors, r.sectors.n_sectors
        self.dl = np.repeat(l.sectors.dims, 2)                                     # left composite index 2 s + sigma
        self.labl = np.repeat(l.sectors.labels[:, 0], 2) + np.tile([-1, 1], nl)
        self.dr = np.tile(r.sectors.dims, 2)                                       # right composite index sigma * n_r + s'
        self.labr = np.tile(r.sectors.labels[:, 0], 2) + np.repeat([-1, 1], nr)
        self.pairs, self.offset, n = [], [], 0
        for i in range(2 * nl):
            for k in range(2 * nr):
                if self.dl[i] and self.dr[k] and self.labl[i] + self.labr[k] == target_twice_sz:
                    self.pairs.append((i, k)); self.offset.append(n); n += int(self.dl[i]) * int(self.dr[k])
        self.n = n
        self.ml, self.mr = l.sectors.total_dim, r.sectors.total_dim
        self.offl = np.concatenate([[0], np.cumsum(l.sectors.dims)]); self.offr = np.concatenate([[0], np.cumsum(r.sectors.dims)])
        self.nl, self.nr = nl, nr

    def scatter(self, x):
        """Target-sector vector -> the full tensor X[a_l, sigma1, sigma2, b_r] (zero outside the target sector)."""
        X = np.zeros((self.ml, 2, 2, self.mr))
        for (i, k), o in zip(self.pairs, self.offset):
            s, s1, s2, sp = i // 2, i % 2, k // self.nr, k % self.nr
            X[self.offl[s]:self.offl[s + 1], s1, s2, self.offr[sp]:self.offr[sp + 1]] = x[o:o + int(self.dl[i]) * int(self.dr[k])].reshape(int(self.dl[i]), int(self.dr[k]))
        return X

    def gather(self, X):
        x = np.zeros(self.n)
        mask = np.ones(X.shape, dtype=bool)
        for (i, k), o in zip(self.pairs, self.offset):
            s, s1, s2, sp = i // 2, i % 2, k // self.nr, k % self.nr
            x[o:o + int(self.dl[i]) * int(self.dr[k])] = X[self.offl[s]:self.offl[s + 1], s1, s2, self.offr[sp]:self.offr[sp + 1]].ravel()
            mask[self.offl[s]:self.offl[s + 1], s1, s2, self.offr[sp]:self.offr[sp + 1]] = False
        assert np.max(np.abs(X[mask]), initial=0.0) <= 1e-12 * max(1.0, np.max(np.abs(X), initial=0.0)), "leakage out of the target sector"
        return x


def apply(l: Block, r: Block, J: float, Delta: float, lay: Layout4, x: np.ndarray) -> np.ndarray:
    """Eq. 13 on the target sector: scatter, sum of Alg. 2 over the quadruplets, gather."""
    X = lay.scatter(x).reshape(-1)          # C order of [a_l, s1, s2, b_r] = the paper's column-major [D, C, B, A] order
    Y = np.zeros_like(X)
    for c, A, a, b, B in terms(l, r, J, Delta):
        Y += c * project_l11r(A, a, b, B, X)
    return lay.gather(Y.reshape(lay.ml, 2, 2, lay.mr))


def diag(l: Block, r: Block, J: float, Delta: float, lay: Layout4) -> np.ndarray:
    """diag(H_SB) on the target sector (A14), from the definition: products of the factors' diagonals."""
    D = np.zeros((lay.ml, 2, 2, lay.mr))
    for c, A, a, b, B in terms(l, r, J, Delta):
        D += c * np.einsum("a,s,t,b->astb", np.diag(A), np.diag(a), np.diag(b), np.diag(B))
    out = np.zeros(lay.n)
    for (i, k), o in zip(lay.pairs, lay.offset):
        s, s1, s2, sp = i // 2, i % 2, k // lay.nr, k % lay.nr
        out[o:o + int(lay.dl[i]) * int(lay.dr[k])] = D[lay.offl[s]:lay.offl[s + 1], s1, s2, lay.offr[sp]:lay.offr[sp + 1]].ravel()
    return out
