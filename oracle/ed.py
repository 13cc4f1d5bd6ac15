"""O-ED: site-level exact Hamiltonians by explicit Kronecker products.  TEST INFRASTRUCTURE.

Heisenberg XXZ chain: PAPER.md:L43-54 (Eq. 1-3).  Spin-1/2 Hubbard chain: PAPER.md:L66-82
(Eq. 4-8) with F = 1/2.  Independent of any block/sector structure.
"""
from __future__ import annotations
from functools import reduce
import numpy as np

I2 = np.eye(2)
# Eq. 3: basis index 0 = up, 1 = down.
S_PLUS = np.array([[0.0, 1.0], [0.0, 0.0]])
S_MINUS = np.array([[0.0, 0.0], [1.0, 0.0]])
S_Z = 0.5 * np.array([[1.0, 0.0], [0.0, -1.0]])
# Eq. 7-8: [1;0] = empty, [0;1] = occupied (L62).
PHI = np.array([[1.0, 0.0], [0.0, -1.0]])
C_DAG = np.array([[0.0, 0.0], [1.0, 0.0]])
C_ANN = np.array([[0.0, 1.0], [0.0, 0.0]])


def kron_all(mats):
    return reduce(np.kron, mats, np.eye(1))


def embed(op: np.ndarray, j: int, N: int) -> np.ndarray:
    """Eq. 2 (L48): O_j = I^{(j-1)} (x) O (x) I^{(N-j)}, j = 1..N."""
    assert 1 <= j <= N
    return kron_all([I2] * (j - 1) + [op] + [I2] * (N - j))


def heisenberg_H(N: int, J: float = 1.0, Delta: float = 1.0) -> np.ndarray:
    """Eq. 1 (L43) with an overall J (reading A2): open chain, nearest neighbours."""
    H = np.zeros((2 ** N, 2 ** N))
    for j in range(1, N):
        H += 0.5 * (embed(S_PLUS, j, N) @ embed(S_MINUS, j + 1, N) + embed(S_MINUS, j, N) @ embed(S_PLUS, j + 1, N))
        H += Delta * (embed(S_Z, j, N) @ embed(S_Z, j + 1, N))
    return J * H


def embed_bond(op2: np.ndarray, j: int, N: int) -> np.ndarray:
    """O_j O'_{j+1} of two Eq.-2 embeddings = I^{(j-1)} (x) (O (x) O') (x) I^{(N-j-1)} (mixed-product
    property); op2 is the 4x4 two-site matrix.  Same operator as the product of two `embed`s,
    without the 2^N x 2^N matmul (tests check the two agree for N <= 8)."""
    assert 1 <= j < N
    return kron_all([I2] * (j - 1) + [op2] + [I2] * (N - j - 1))


def heisenberg_H_bond(N: int, J: float = 1.0, Delta: float = 1.0) -> np.ndarray:
    """Eq. 1 assembled bond by bond with `embed_bond` (usable up to N = 12)."""
    h = 0.5 * (np.kron(S_PLUS, S_MINUS) + np.kron(S_MINUS, S_PLUS)) + Delta * np.kron(S_Z, S_Z)
    H = np.zeros((2 ** N, 2 ** N))
    for j in range(1, N):
        H += embed_bond(h, j, N)
    return J * H


def heisenberg_twice_sz(N: int) -> np.ndarray:
    """Diagonal of 2*S_z^tot = sum_j 2 S^z_j (integer quantum number, L88)."""
    d = np.zeros(2 ** N)
    for j in range(1, N + 1):
        d += np.diag(embed(2.0 * S_Z, j, N))
    return np.rint(d).astype(np.int64)


# ---- Hubbard, F = 1/2: modes are site-major, sigma = -1/2 (index 0) before +1/2 (index 1) -------------
def hubbard_mode_op(op: np.ndarray, j: int, s: int, N: int) -> np.ndarray:
    """Eq. 5-6 (L72-76): Phi on every mode preceding (site j, polarisation s), identity after.
    j = 1..N, s = 0 (sigma=-1/2, "down") or 1 (sigma=+1/2, "up").  The upper limits printed in
    Eq. 5 do not add up to F'N factors (reading A27): identities fill all following modes."""
    assert 1 <= j <= N and s in (0, 1)
    p = 2 * (j - 1) + s
    M = 2 * N
    return kron_all([PHI] * p + [op] + [I2] * (M - p - 1))


def hubbard_number(j: int, s: int, N: int) -> np.ndarray:
    c = hubbard_mode_op(C_ANN, j, s, N)
    return hubbard_mode_op(C_DAG, j, s, N) @ c


def hubbard_H(N: int, t: float = 1.0, U: float = 4.0) -> np.ndarray:
    """Eq. 4 (L66) with F = 1/2: (U/2) sum_{sigma != sigma'} n n = U n_up n_dn per site."""
    dim = 4 ** N
    H = np.zeros((dim, dim))
    for j in range(1, N):
        for s in (0, 1):
            hop = hubbard_mode_op(C_DAG, j, s, N) @ hubbard_mode_op(C_ANN, j + 1, s, N)
            H += -t * (hop + hop.T)
    for j in range(1, N + 1):
        n0, n1 = hubbard_number(j, 0, N), hubbard_number(j, 1, N)
        H += 0.5 * U * (n0 @ n1 + n1 @ n0)
    return H


def hubbard_counts(N: int):
    """Diagonals of (N_up, N_dn) = (sum_j n_{j,+1/2}, sum_j n_{j,-1/2}) as integers."""
    nu = sum(np.diag(hubbard_number(j, 1, N)) for j in range(1, N + 1))
    nd = sum(np.diag(hubbard_number(j, 0, N)) for j in range(1, N + 1))
    return np.rint(nu).astype(np.int64), np.rint(nd).astype(np.int64)


def hubbard_double_occupancy(N: int) -> np.ndarray:
    """D = sum_j n_{j,up} n_{j,dn} (dense, diagonal)."""
    dim = 4 ** N
    D = np.zeros((dim, dim))
    for j in range(1, N + 1):
        D += hubbard_number(j, 0, N) @ hubbard_number(j, 1, N)
    return D


def lowest_in_sector(H: np.ndarray, mask: np.ndarray):
    """Lowest eigenpair of H restricted to the basis states selected by ``mask``."""
    idx = np.nonzero(mask)[0]
    w, v = np.linalg.eigh(H[np.ix_(idx, idx)])
    return w, v, idx
