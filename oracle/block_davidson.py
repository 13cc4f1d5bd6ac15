"""O-BDAV: block Davidson (Davidson-Liu) for the lowest `b` eigenpairs.  TEST INFRASTRUCTURE.

PAPER.md:L247 names the method only ("block extension ... the so called Davidson-Liu, to determine a few of the
lowest eigenvalues, where more than one candidate vectors are added at once resulting in BLAS level 3 operations")
and gives no listing, so this is the textbook method written in the notation and line order of the paper's own
Alg. 3 (L201-237), with b columns wherever Alg. 3 has one -- every reading A13-A19 of DESIGN.md is applied column by
column, and at b = 1 a step is `oracle.davidson.davidson_step` to the last bit (pinned in tests/test_oracle_block.py).

State: V, W (n x k_max, column-contiguous), G = V^T W (k_max x k_max; the paper's B), k = basis vectors held,
na = how many of the newest columns still lack their projection W = H V.

Readings made here (A29-A32):
  A29  one step = project the `na` newest basis vectors, Rayleigh-Ritz for the lowest b pairs, residuals, then one
       correction vector per NOT yet converged pair (a converged pair, ||r_i|| <= tol, adds nothing);
  A30  converged = all of the lowest b residual norms <= tol (A17 per pair);
  A31  restart when the corrections would not fit (k + na_new > k_max): collapse to the b Ritz vectors (A15 per column);
  A32  the corrections are orthogonalised against V by `reorth` classical Gram-Schmidt passes (A16), then among
       themselves, in pair order, by modified Gram-Schmidt with two passes -- i.e. the unique thin QR factor with a
       positive diagonal; a correction whose norm after projection is zero or not finite is a breakdown.
"""
from __future__ import annotations
from dataclasses import dataclass
import numpy as np
from .davidson import small_eig, precondition  # noqa: F401  (precondition: A14, shared column by column)


@dataclass
class BlockState:
    V: np.ndarray
    W: np.ndarray
    G: np.ndarray
    k: int
    na: int          # newest columns V(:, k-na .. k-1) not yet projected


def orthonormalise_columns(T: np.ndarray) -> np.ndarray:
    """A32: thin QR with positive diagonal by two passes of modified Gram-Schmidt, in column order."""
    Q = np.array(T, dtype=np.float64, order="F", copy=True)
    for _ in range(2):
        for j in range(Q.shape[1]):
            for i in range(j):
                Q[:, j] -= (Q[:, i] @ Q[:, j]) * Q[:, i]
            nrm = float(np.linalg.norm(Q[:, j]))
            if not np.isfinite(nrm) or nrm == 0.0:
                raise FloatingPointError("block Davidson breakdown: dependent start/correction vectors")
            Q[:, j] /= nrm
    return Q


def init_state(X0: np.ndarray, k_max: int) -> BlockState:
    """Step 0 (Alg. 3 'Require', L204, with b columns): V(:,1:b) = orthonormalised X0."""
    n, b = X0.shape
    assert b <= k_max
    V = np.zeros((n, k_max), order="F")
    W = np.zeros((n, k_max), order="F")
    V[:, :b] = orthonormalise_columns(X0)
    return BlockState(V, W, np.zeros((k_max, k_max)), b, b)


def small_eig_block(Gk: np.ndarray, b: int):
    """Line 4 with b pairs (A18 per column): the b lowest eigenpairs of the symmetrised k x k matrix, ascending; each
    vector's largest-|y_p| component made positive (lowest index on ties)."""
    w, Y = np.linalg.eigh(0.5 * (Gk + Gk.T))
    Y = Y[:, :b].copy()
    for c in range(Y.shape[1]):
        p = int(np.argmax(np.abs(Y[:, c])))
        if Y[p, c] < 0:
            Y[:, c] = -Y[:, c]
    return w[:b].copy(), Y


def block_step(st: BlockState, apply, D: np.ndarray, b: int, tol: float, reorth: int = 1):
    """One block iteration.  Returns dict(theta (b), resnorm (b), converged, Y, k_used, X (when converged))."""
    V, W, G = st.V, st.W, st.G
    k, k_max = st.k, V.shape[1]
    # line 2 for every new column: W(:,j) = H_SB V(:,j)
    for j in range(k - st.na, k):
        W[:, j] = apply(V[:, j])
    # line 3: G(1:k, new) = V^T W(:, new), mirrored (A18)
    for j in range(k - st.na, k):
        col = V[:, :k].T @ W[:, j]
        G[:k, j] = col
        G[j, :k] = col
    st.na = 0
    # line 4
    nb = min(b, k)
    theta, Y = small_eig_block(G[:k, :k], nb)
    # lines 5-7
    X = V[:, :k] @ Y
    WY = W[:, :k] @ Y
    R = WY - X * theta[None, :]
    rho = np.linalg.norm(R, axis=0)
    out = dict(theta=theta, resnorm=rho, converged=False, Y=Y, k_used=k)
    active = [i for i in range(nb) if not rho[i] <= tol]
    if not active:
        out["converged"] = True
        out["X"] = X / np.linalg.norm(X, axis=0)[None, :]
        return out
    # restart (A31): collapse to the Ritz vectors, no extra apply
    if k + len(active) > k_max:
        nx = np.linalg.norm(X, axis=0)
        V[:, :nb] = X / nx[None, :]
        W[:, :nb] = WY / nx[None, :]
        G[:, :] = 0.0
        G[np.arange(nb), np.arange(nb)] = theta
        k = nb
    # line 10, one correction per unconverged pair
    T = np.stack([precondition(R[:, i], float(theta[i]), D) for i in active], axis=1)
    # lines 12-13 against the basis (A16), then among themselves (A32)
    for _ in range(reorth):
        S = V[:, :k].T @ T
        T = T - V[:, :k] @ S
    Q = orthonormalise_columns(T)
    # line 14
    V[:, k:k + len(active)] = Q
    st.k = k + len(active)
    st.na = len(active)
    return out


def block_solve(apply, D: np.ndarray, X0: np.ndarray, k_max: int, tol: float, max_iter: int, reorth: int = 1):
    """Driver: iterate until the lowest b = X0.shape[1] pairs are converged or max_iter block iterations are spent."""
    b = X0.shape[1]
    st = init_state(X0, k_max)
    hist, res, applies = [], None, 0
    for it in range(1, max_iter + 1):
        applies += st.na
        res = block_step(st, apply, D, b, tol, reorth)
        hist.append((res["theta"].copy(), res["resnorm"].copy()))
        if res["converged"]:
            return dict(theta=res["theta"], X=res["X"], resnorm=res["resnorm"], iters=it, applies=applies,
                        converged=True, history=hist, state=st)
    return dict(theta=res["theta"], X=None, resnorm=res["resnorm"], iters=max_iter, applies=applies,
                converged=False, history=hist, state=st)


def start_lowest_diag(D: np.ndarray, b: int) -> np.ndarray:
    """Deterministic block start (A19 (D) with b columns): unit vectors at the b smallest D_pp (stable order)."""
    idx = np.argsort(D, kind="stable")[:b]
    X = np.zeros((D.shape[0], b))
    X[idx, np.arange(b)] = 1.0
    return X
