"""O-REN: the steps either side of the Davidson hot path in one infinite-lattice DMRG iteration.  TEST INFRASTRUCTURE.

PAPER.md:L100-110 (Alg. 1): "1 Load a left and a right block.  2 Form the superblock configuration.  3 Compute the lowest
eigenstate of H_SB (Davidson).  4 for each block: 5 Construct the density matrix for the given block from the lowest
eigenstate.  6 Compute the eigenvalues of the density matrix.  7 Renormalize the basis of the block by keeping states with
high eigenvalues."  L112/L120: two-site procedure, both blocks are enlarged by one site per iteration, starting from
single-site blocks; LR strategy: the superblock is formed from the two ENLARGED blocks (L124).

The paper gives no formulas for lines 5-7 (it refers to [1-3]); the textbook definitions are written out here, dense and slow:
  line 2   enlarged block = block (x) site (left) or site (x) block (right); H_e = H_b + bond term of Eq. 1 (A2/A3) between
           the block's boundary site and the new site; the new site becomes the boundary site;
  line 5   rho_L = Tr_R |psi><psi| : with Psi[a, b] the wave function as a (dim_L x dim_R) matrix, rho_L = Psi Psi^T,
           rho_R = Psi^T Psi.  U(1) symmetry makes rho block diagonal in the sector label: rho_i = sum_k X_ik X_ik^T
           (left), rho_k = sum_i X_ik^T X_ik (right);
  line 6   all eigenpairs of every rho_i (the paper uses Lanczos; any symmetric eigensolver gives the same pairs);
  line 7   keep the m eigenvectors with the largest eigenvalues over ALL sectors (A33: ties broken by sector index, then by
           position in the ascending LAPACK order; eigenvalues <= 0 are never kept); new sector dims m_i; every operator block
           is rotated, O'_{s->d} = U_d^T O_{s->d} U_s; discarded weight = 1 - sum of kept eigenvalues.
"""
from __future__ import annotations
from dataclasses import dataclass
from typing import List
import numpy as np
from dmrg_inputs.problem import Sectors, BlockOp, Problem, HEISENBERG
from . import ed
from .blocks import _sort_basis, _cut
from .kron import dense_op
from .rec import Layout


@dataclass
class Block:
    """A block of the chain in its current (possibly truncated) basis: H of the block and the boundary-site operators."""
    sectors: Sectors
    H: BlockOp
    Sz: BlockOp
    Sp: BlockOp
    n_sites: int


def single_site_block() -> Block:
    """L120: 'each block contains a single spin'.  Labels are 2 S_z; basis ordered by label (down, up)."""
    sec = Sectors(np.array([[-1], [1]]), np.array([1, 1]))
    H, Sz, Sp = BlockOp(), BlockOp(), BlockOp()
    Sz.add(0, 0, np.array([[-0.5]])); Sz.add(1, 1, np.array([[0.5]]))
    Sp.add(0, 1, np.array([[1.0]]))
    return Block(sec, H, Sz, Sp, 1)


def enlarge(b: Block, side: str, J: float, Delta: float) -> Block:
    """Alg. 1 line 2 for one block (Heisenberg, Eq. 1-3 with the overall J of reading A2)."""
    sec = b.sectors
    Hb, Szb, Spb = dense_op(b.H, sec), dense_op(b.Sz, sec), dense_op(b.Sp, sec)
    lab_b = np.repeat(sec.labels[:, 0], sec.dims)
    m = Hb.shape[0]
    Ib, Is = np.eye(m), np.eye(2)
    # site basis ordered (down, up) = labels (-1, +1): S+ |down> = |up>
    Szs, Sps = np.diag([-0.5, 0.5]), np.array([[0.0, 0.0], [1.0, 0.0]])
    lab_s = np.array([-1, 1])
    if side == "left":      # block (x) site, block index slow
        H = np.kron(Hb, Is) + 0.5 * J * (np.kron(Spb, Sps.T) + np.kron(Spb.T, Sps)) + J * Delta * np.kron(Szb, Szs)
        Sz, Sp = np.kron(Ib, Szs), np.kron(Ib, Sps)
        lab = (lab_b[:, None] + lab_s[None, :]).reshape(-1)
    else:                   # site (x) block, site index slow
        H = np.kron(Is, Hb) + 0.5 * J * (np.kron(Sps, Spb.T) + np.kron(Sps.T, Spb)) + J * Delta * np.kron(Szs, Szb)
        Sz, Sp = np.kron(Szs, Ib), np.kron(Sps, Ib)
        lab = (lab_s[:, None] + lab_b[None, :]).reshape(-1)
    perm, uniq, dims = _sort_basis(lab.reshape(-1, 1))
    return Block(Sectors(uniq, dims), _cut(H, perm, dims), _cut(Sz, perm, dims), _cut(Sp, perm, dims), b.n_sites + 1)


def superblock(L: Block, R: Block, J: float, Delta: float, target_twice_sz: int = 0) -> Problem:
    """Alg. 1 line 2: the LR superblock of two enlarged blocks (what dmrg_plan_create is told)."""
    return Problem(HEISENBERG, J, Delta, 0.0, 0.0, L.sectors, R.sectors,
                   {"H_L": L.H, "H_R": R.H, "Sz_L": L.Sz, "Sp_L": L.Sp, "Sz_R": R.Sz, "Sp_R": R.Sp}, np.array([target_twice_sz]))


def reduced_density_matrices(p: Problem, lay: Layout, x: np.ndarray, side: str) -> List[np.ndarray]:
    """Alg. 1 line 5: one d x d matrix per sector of the chosen side (zero matrix for a sector without a pair)."""
    sec = p.left if side == "left" else p.right
    rho = [np.zeros((int(d), int(d))) for d in sec.dims]
    for (i, k) in lay.pairs:
        X = lay.seg(x, i, k)
        if side == "left":
            rho[i] += X @ X.T
        else:
            rho[k] += X.T @ X
    return rho


def truncation_basis(rho: List[np.ndarray], m: int):
    """Alg. 1 lines 6-7.  Returns (U per sector [d_s x m_s, columns by descending weight], kept weights per sector,
    discarded weight)."""
    cand = []
    eig = []
    for s, r in enumerate(rho):
        if r.shape[0] == 0:
            eig.append((np.zeros(0), np.zeros((0, 0))))
            continue
        w, Uv = np.linalg.eigh(0.5 * (r + r.T))
        eig.append((w, Uv))
        for j in range(len(w) - 1, -1, -1):          # descending weight inside the sector
            if w[j] > 0.0:
                cand.append((-w[j], s, len(w) - 1 - j, j))
    cand.sort()                                       # by weight, then sector, then rank inside the sector (A33)
    keep = cand[:m]
    U, kept = [], []
    for s, (w, Uv) in enumerate(eig):
        cols = [j for (_, ss, _, j) in keep if ss == s]
        U.append(Uv[:, cols] if cols else np.zeros((Uv.shape[0], 0)))
        kept.append(w[cols] if cols else np.zeros(0))
    total = sum(float(np.trace(r)) for r in rho)
    return U, kept, total - sum(float(kw.sum()) for kw in kept)


def rotate_op(op: BlockOp, U: List[np.ndarray]) -> BlockOp:
    """O'_{s->d} = U_d^T O_{s->d} U_s (sector indices are kept; sectors may end up with dimension 0)."""
    out = BlockOp()
    for s, d, blk in zip(op.src, op.dst, op.blocks):
        if U[s].shape[1] and U[d].shape[1]:
            out.add(s, d, U[d].T @ blk @ U[s])
    return out


def renormalise(b: Block, U: List[np.ndarray]) -> Block:
    """Alg. 1 line 7 for one enlarged block."""
    dims = np.array([u.shape[1] for u in U], dtype=np.int32)
    return Block(Sectors(b.sectors.labels.copy(), dims), rotate_op(b.H, U), rotate_op(b.Sz, U), rotate_op(b.Sp, U), b.n_sites)


def infinite_dmrg(N: int, m: int, J: float = 1.0, Delta: float = 1.0, solve=None):
    """Alg. 1 looped from the four-site configuration up to N sites (N even).  `solve(problem) -> (E, x)` is line 3
    (default: dense diagonalisation of the target sector via oracle.kron).  Returns one record per superblock size."""
    from . import kron
    if solve is None:
        def solve(p):
            Hs, _ = kron.H_sector(p)
            w, v = np.linalg.eigh(Hs)
            return float(w[0]), v[:, 0]
    L, R = single_site_block(), single_site_block()
    out = []
    while True:
        L, R = enlarge(L, "left", J, Delta), enlarge(R, "right", J, Delta)
        p = superblock(L, R, J, Delta, 0)
        E, x = solve(p)
        lay = Layout(p)
        UL, _, dL = truncation_basis(reduced_density_matrices(p, lay, x, "left"), m)
        UR, _, dR = truncation_basis(reduced_density_matrices(p, lay, x, "right"), m)
        out.append(dict(n_sites=L.n_sites + R.n_sites, energy=E, discarded=(dL, dR), dim=(L.sectors.total_dim, R.sectors.total_dim), n=lay.n))
        if L.n_sites + R.n_sites >= N:
            return out
        L, R = renormalise(L, UL), renormalise(R, UR)
