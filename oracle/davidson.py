"""O-DAV: textbook Davidson following PAPER.md Alg. 3 (L201-237) line by line.  TEST INFRASTRUCTURE.

Line numbering per reading A13; every choice the paper leaves open is tagged with its
reading (A14-A19) in DESIGN.md.  State: V, W (n x k_max, column-contiguous), B (k_max x k_max),
k = number of basis vectors held, D = diag(H_SB).
"""
from __future__ import annotations
from dataclasses import dataclass, field
import numpy as np

GUARD = 1e-8  # A14: |lambda - D_pp| floor of the diagonal preconditioner


@dataclass
class DavidsonState:
    V: np.ndarray
    W: np.ndarray
    B: np.ndarray
    k: int
    history: list = field(default_factory=list)


def init_state(x0: np.ndarray, k_max: int) -> DavidsonState:
    """Step 0 (L204): V(:,1) = x0/||x0|| (A19), k = 1."""
    n = x0.shape[0]
    V = np.zeros((n, k_max), order="F")
    W = np.zeros((n, k_max), order="F")
    V[:, 0] = x0 / np.linalg.norm(x0)
    return DavidsonState(V, W, np.zeros((k_max, k_max)), 1)


def small_eig(Bk: np.ndarray):
    """Line 4 (L212; A18): lowest eigenpair of the symmetric k x k matrix; sign convention:
    the largest-|y_p| component positive (lowest index on ties)."""
    w, Y = np.linalg.eigh(0.5 * (Bk + Bk.T))
    y = Y[:, 0].copy()
    p = int(np.argmax(np.abs(y)))  # argmax returns the lowest index on ties
    if y[p] < 0:
        y = -y
    return float(w[0]), y


def precondition(r: np.ndarray, lam: float, D: np.ndarray) -> np.ndarray:
    """Line 10 "correct r" (L223; A14): t_p = r_p / g(lambda - D_pp)."""
    delta = lam - D
    small = np.abs(delta) < GUARD
    g = np.where(small, np.where(np.signbit(delta), -GUARD, GUARD), delta)
    return r / g


def davidson_step(st: DavidsonState, apply, D: np.ndarray, tol: float, reorth: int = 1):
    """One call of Alg. 3.  Returns dict(lam, resnorm, converged, x (only when converged), y)."""
    V, W, B = st.V, st.W, st.B
    k = st.k
    k_max = V.shape[1]
    # line 2 (L206): W(:,k) = H_SB V(:,k)
    W[:, k - 1] = apply(V[:, k - 1])
    # line 3 (L209): B(1:k,k) = V(:,1:k)^T W(:,k), mirrored into row k (A18)
    col = V[:, :k].T @ W[:, k - 1]
    B[:k, k - 1] = col
    B[k - 1, :k] = col
    # line 4 (L212)
    lam, y = small_eig(B[:k, :k])
    # lines 5-6 (L213-215): x = V y ; r = W y - lambda x
    x = V[:, :k] @ y
    wy = W[:, :k] @ y
    r = wy - lam * x
    # lines 7-8 (L217-219; A17)
    rho = float(np.linalg.norm(r))
    out = dict(lam=lam, resnorm=rho, converged=False, y=y, k_used=k)
    if rho <= tol:
        out["converged"] = True
        out["x"] = x / np.linalg.norm(x)
        return out
    # restart at the basis limit (L271; A15): collapse to the Ritz vector, no extra apply
    if k == k_max:
        nx = np.linalg.norm(x)
        V[:, 0] = x / nx
        W[:, 0] = wy / nx
        B[:, :] = 0.0
        B[0, 0] = lam
        k = 1
    # line 10 (L223; A14)
    t = precondition(r, lam, D)
    # lines 12-13 (L227-231; A16): classical Gram-Schmidt, all k coefficients from the same t
    for _ in range(reorth):
        s = V[:, :k].T @ t
        t = t - V[:, :k] @ s
    # line 14 (L233)
    tau = float(np.linalg.norm(t))
    if not np.isfinite(tau) or tau == 0.0:
        raise FloatingPointError("Davidson breakdown: correction vector has zero/non-finite norm")
    V[:, k] = t / tau
    st.k = k + 1
    return out


def davidson_solve(apply, D: np.ndarray, x0: np.ndarray, k_max: int, tol: float, max_iter: int, reorth: int = 1):
    """Driver (L217-235): loop Alg. 3 until ||r|| <= tol or max_iter applies."""
    st = init_state(x0, k_max)
    hist = []
    res = None
    for it in range(1, max_iter + 1):
        res = davidson_step(st, apply, D, tol, reorth)
        hist.append((res["lam"], res["resnorm"]))
        if res["converged"]:
            return dict(lam=res["lam"], x=res["x"], resnorm=res["resnorm"], iters=it, converged=True, history=hist, state=st)
    # not converged: best Ritz pair from the last step
    y = res["y"]
    return dict(lam=res["lam"], x=None, resnorm=res["resnorm"], iters=max_iter, converged=False, history=hist, state=st)


def start_argmin_diag(D: np.ndarray) -> np.ndarray:
    """Deterministic start (D) of A19: unit vector at argmin_p D_pp (lowest index on ties)."""
    x = np.zeros_like(D)
    x[int(np.argmin(D))] = 1.0
    return x
