"""Pins of oracle/block_davidson.py (O-BDAV, Davidson-Liu) against things other than itself:
reduction to the single-vector Alg. 3 oracle at b = 1, LAPACK eigenpairs of small dense matrices, an exactly
doubly-degenerate spectrum, the library QR factor, and the invariants of a Rayleigh-Ritz iteration."""
import numpy as np
import pytest

from dmrg_inputs import random_vector, make_config
from oracle import blocks, kron, rec, davidson as odav, block_davidson as obd


def _dense(name):
    p = {"cfg1": lambda: blocks.heisenberg_exact(6, 6, 1.0, 1.0),
         "hub33": lambda: blocks.hubbard_exact(3, 3, 1.0, 4.0),
         "cfg2_m60": lambda: make_config("cfg2", 60)}[name]()
    H, _ = kron.H_sector(p)
    return p, H


def test_qr_factor_is_the_library_one():
    rng = np.random.default_rng(5)
    T = rng.standard_normal((200, 4))
    Q = obd.orthonormalise_columns(T)
    Qn, Rn = np.linalg.qr(T)
    Qn = Qn * np.sign(np.diag(Rn))[None, :]          # positive diagonal of R makes the factor unique
    assert np.max(np.abs(Q - Qn)) <= 1e-13
    assert np.max(np.abs(Q.T @ Q - np.eye(4))) <= 1e-15 * 50
    with pytest.raises(FloatingPointError):
        obd.orthonormalise_columns(np.stack([T[:, 0], 2.0 * T[:, 0] - T[:, 0] * 2.0], axis=1))


@pytest.mark.parametrize("name,k_max,reorth", [("cfg1", 16, 1), ("cfg1", 4, 2), ("hub33", 7, 1)])
def test_block_size_one_is_algorithm_3(name, k_max, reorth):
    """b = 1: every step equals oracle.davidson.davidson_step (lambda, ||r||, the basis), through restarts."""
    p, H = _dense(name)
    n = H.shape[0]
    D = np.diag(H).copy()
    x0 = random_vector(n, 77)
    s1 = odav.init_state(x0, k_max)
    sb = obd.init_state(x0.reshape(-1, 1), k_max)
    apply = lambda v: H @ v
    for it in range(40):
        r1 = odav.davidson_step(s1, apply, D, 1e-11, reorth)
        rb = obd.block_step(sb, apply, D, 1, 1e-11, reorth)
        assert abs(r1["lam"] - rb["theta"][0]) <= 1e-13 * max(1.0, abs(r1["lam"]))
        assert abs(r1["resnorm"] - rb["resnorm"][0]) <= 1e-12 * max(1.0, r1["resnorm"])
        assert r1["converged"] == rb["converged"]
        if r1["converged"]:
            break
        assert s1.k == sb.k
        # the appended vectors agree up to the rounding of one extra normalisation (A32 runs two MGS passes)
        assert np.max(np.abs(s1.V[:, :s1.k] - sb.V[:, :sb.k])) <= 1e-6   # (the iteration amplifies last-bit differences, A20)
    assert it >= 10


@pytest.mark.parametrize("name,b,k_max", [("cfg1", 2, 16), ("cfg1", 4, 12), ("hub33", 3, 12), ("cfg2_m60", 4, 16)])
def test_converges_to_lapack_lowest_pairs(name, b, k_max):
    p, H = _dense(name)
    n = H.shape[0]
    D = np.diag(H).copy()
    w, U = np.linalg.eigh(H)
    rng = np.random.default_rng(11)
    res = obd.block_solve(lambda v: H @ v, D, rng.standard_normal((n, b)), k_max, 1e-10, 3000)
    assert res["converged"]
    assert np.max(np.abs(res["theta"] - w[:b])) <= 1e-9
    X = res["X"]
    # recomputed residuals and Rayleigh quotients with the matrix itself
    for i in range(b):
        assert np.linalg.norm(H @ X[:, i] - res["theta"][i] * X[:, i]) <= 2e-10
        assert abs(X[:, i] @ H @ X[:, i] - res["theta"][i]) <= 1e-12 * max(1.0, abs(w[0]))
    # the spanned subspace is the LAPACK one wherever the b-th and (b+1)-th eigenvalues are separated
    if w[b] - w[b - 1] > 1e-6:
        Pw = U[:, :b] @ U[:, :b].T
        assert np.max(np.abs(Pw @ X - X)) <= 1e-6
    # basis invariants of the final state
    st = res["state"]
    Vk = st.V[:, :st.k - st.na]
    assert np.max(np.abs(Vk.T @ Vk - np.eye(Vk.shape[1]))) <= 1e-12
    assert np.max(np.abs(st.W[:, :Vk.shape[1]] - H @ Vk)) <= 1e-11 * np.max(np.abs(H))
    assert np.max(np.abs(st.G[:Vk.shape[1], :Vk.shape[1]] - Vk.T @ H @ Vk)) <= 1e-11 * np.max(np.abs(H))


def test_exactly_degenerate_ground_state_is_found_twice():
    """H = blockdiag(A, A): every eigenvalue is doubly degenerate; the block method with b = 2 returns the lowest one
    twice with two orthogonal vectors (what a single-vector iteration cannot do)."""
    rng = np.random.default_rng(3)
    A = rng.standard_normal((40, 40)); A = A + A.T + np.diag(np.arange(40.0))
    H = np.zeros((80, 80)); H[:40, :40] = A; H[40:, 40:] = A
    w = np.linalg.eigvalsh(A)
    res = obd.block_solve(lambda v: H @ v, np.diag(H).copy(), rng.standard_normal((80, 2)), 12, 1e-10, 2000)
    assert res["converged"]
    assert np.max(np.abs(res["theta"] - w[0])) <= 1e-9
    X = res["X"]
    assert abs(X[:, 0] @ X[:, 1]) <= 1e-9


def test_monotone_ritz_values_and_restart_is_exercised():
    p, H = _dense("cfg1")
    n = H.shape[0]
    D = np.diag(H).copy()
    res = obd.block_solve(lambda v: H @ v, D, obd.start_lowest_diag(D, 3), 7, 1e-10, 2000)
    assert res["converged"] and res["iters"] > 6          # k_max = 7, b = 3: a restart every other step
    th = np.array([h[0] for h in res["history"]])
    for i in range(3):                                      # Ritz values never rise (Cauchy interlacing; restart keeps them)
        assert np.all(np.diff(th[:, i]) <= 1e-11)
    assert np.max(np.abs(th[-1] - np.linalg.eigvalsh(H)[:3])) <= 1e-9
    X0 = obd.start_lowest_diag(D, 3)
    assert np.array_equal(X0.sum(axis=0), np.ones(3)) and set(np.argmax(X0, axis=0)) == set(np.argsort(D, kind="stable")[:3])
