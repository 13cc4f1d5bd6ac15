"""Parity of the block path (Davidson-Liu) with the CPU oracle O-BDAV:
dmrg_apply_H_multi against O-REC column by column, block steps in lock step with oracle.block_davidson.block_step
(theta, ||r||, the new columns of G, the appended orthonormal vectors), converged lowest-nb eigenpairs against LAPACK /
the oracle's own block run, and nb = 1 against the single-vector path."""
import numpy as np
import pytest

from dmrg_inputs import random_vector
from oracle import rec, kron, block_davidson as obd
from gpu_common import small_problems, full_config, oracle_apply, rel_maxnorm, to_dev, HPSI_RTOL, LAMBDA_ATOL, OVERLAP_DEF

pytestmark = pytest.mark.gpu
SMALL = small_problems()


@pytest.fixture(scope="module")
def lib():
    import torch
    assert torch.cuda.is_available()
    import paper_1309_5571_b200 as lib
    lib.load_library()
    return lib


def _block(n, nb, seed):
    return np.stack([random_vector(n, seed + r) for r in range(nb)], axis=0)      # (nb, n): rows = vectors


@pytest.mark.parametrize("name", ["cfg1", "heis_syn_m300_ragged", "hub_syn_m60", "cfg4_m243", "heis_syn_m517"])
@pytest.mark.parametrize("nrhs", [2, 3, 4])
def test_apply_multi_matches_oracle_and_single(lib, name, nrhs):
    import torch
    p = SMALL[name]()
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=8, max_rhs=4)
    X = _block(lay.n, nrhs, 4100)
    ld = lay.n + 3                                   # odd column stride: the scalar store path of the epilogue
    for ldx in (None, ld):
        Xd = torch.zeros((nrhs, ldx or (lay.n + 15) // 16 * 16), dtype=torch.float64, device="cuda")
        Xd[:, :lay.n] = to_dev(X)
        Yd = torch.full_like(Xd, float("nan"))
        plan.apply_H_multi(Xd, Yd)
        Y2 = plan.apply_H_multi(Xd)
        torch.cuda.synchronize()
        apply_o = oracle_apply(p, lay)
        for r in range(nrhs):
            assert rel_maxnorm(Yd[r, :lay.n].cpu().numpy(), apply_o(X[r])) <= HPSI_RTOL
            # same bits as the single-vector launch (same units, same order of operations per right-hand side)
            assert torch.equal(Yd[r, :lay.n], plan.apply_H(Xd[r, :lay.n].contiguous()))
            assert torch.equal(Yd[r, :lay.n], Y2[r, :lay.n])
    with pytest.raises(lib.DmrgError):
        lib.Plan(p, k_max=8, max_rhs=2).apply_H_multi(torch.zeros((3, lay.n + 1), dtype=torch.float64, device="cuda"))
    plan.close()


def test_apply_multi_full_config_cfg3(lib):
    import torch
    p = full_config("cfg3")
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=8, max_rhs=4)
    X = _block(lay.n, 4, 4200)
    Xd = torch.zeros((4, (lay.n + 15) // 16 * 16), dtype=torch.float64, device="cuda"); Xd[:, :lay.n] = to_dev(X)
    Y = plan.apply_H_multi(Xd)
    apply_o = oracle_apply(p, lay)
    for r in (0, 3):
        assert rel_maxnorm(Y[r, :lay.n].cpu().numpy(), apply_o(X[r])) <= HPSI_RTOL
    plan.close()


def _lockstep_block(lib, p, nb, k_max, steps, X0, reorth=1, tol=1e-10):
    import torch
    lay = rec.Layout(p)
    n = lay.n
    apply_o = oracle_apply(p, lay)
    D = rec.diag_H(p, lay)
    plan = lib.Plan(p, k_max=k_max, tol=tol, reorth=reorth, max_rhs=4)
    V, W = plan.new_basis()
    X0d = torch.zeros((nb, V.stride(0)), dtype=torch.float64, device="cuda"); X0d[:, :n] = to_dev(X0)
    k, na = plan.block_init(V, W, X0d)
    # the start block is the unique QR factor of X0 (A32)
    Q0 = obd.orthonormalise_columns(X0.T)
    assert np.max(np.abs(V[:nb, :n].cpu().numpy().T - Q0)) <= 1e-12
    worst = dict(theta=0.0, rho=0.0, G=0.0, v=0.0)
    conv = False
    for it in range(steps):
        G0, _ = plan.block_get_small(nb)
        Vh = np.asfortranarray(V[:, :n].cpu().numpy().T); Wh = np.asfortranarray(W[:, :n].cpu().numpy().T)
        st = obd.BlockState(Vh, Wh, G0.copy(), k, na)
        ores = obd.block_step(st, apply_o, D, nb, tol, reorth)
        k_prev, na_prev = k, na
        k, na, th, rho, conv = plan.block_step(V, W, k, na, nb)
        assert conv == ores["converged"]
        worst["theta"] = max(worst["theta"], float(np.max(np.abs(th - ores["theta"]))))
        worst["rho"] = max(worst["rho"], float(np.max(np.abs(rho - ores["resnorm"]) / (1e-9 + 1e-6 * ores["resnorm"]))))
        if conv:
            break
        assert (k, na) == (st.k, st.na)
        G1, _ = plan.block_get_small(nb)
        if k > k_prev:      # no restart: the columns of G written by this step
            worst["G"] = max(worst["G"], float(np.max(np.abs(G1[:k_prev, k_prev - na_prev:k_prev] - st.G[:k_prev, k_prev - na_prev:k_prev]))))
        gap = np.min(np.abs(ores["theta"][:, None] - D[None, :]))
        if gap > 1e-3:      # A20: else the preconditioned vectors are legitimately ill-conditioned
            Vg = V[k - na:k, :n].cpu().numpy().T
            worst["v"] = max(worst["v"], float(np.max(np.abs(Vg - st.V[:, k - na:k]))))
    plan.close()
    return worst, conv


@pytest.mark.parametrize("name,nb,k_max,reorth", [("cfg1", 2, 16, 1), ("cfg1", 4, 9, 2), ("cfg2_m160", 3, 12, 1),
                                                  ("hub_exact_3_3", 2, 7, 1), ("cfg4_m243", 4, 16, 1)])
def test_block_lockstep(lib, name, nb, k_max, reorth):
    p = SMALL[name]()
    n = rec.Layout(p).n
    worst, _ = _lockstep_block(lib, p, nb, k_max, 20, _block(n, nb, 2101).copy(), reorth)
    assert worst["theta"] <= LAMBDA_ATOL and worst["rho"] <= 1.0 and worst["G"] <= 1e-10 and worst["v"] <= 1e-7, worst


def test_block_lockstep_full_config_cfg2(lib):
    p = full_config("cfg2")
    lay = rec.Layout(p)
    X0 = obd.start_lowest_diag(rec.diag_H(p, lay), 4).T.copy()
    worst, _ = _lockstep_block(lib, p, 4, 16, 12, X0)
    assert worst["theta"] <= LAMBDA_ATOL and worst["rho"] <= 1.0 and worst["G"] <= 1e-10 and worst["v"] <= 1e-7, worst


@pytest.mark.parametrize("name,nb", [("cfg1", 2), ("cfg1", 4), ("hub_exact_3_3", 3)])
def test_block_driver_vs_lapack(lib, name, nb):
    """Lowest nb eigenpairs of small exact problems against the dense eigendecomposition of the sector Hamiltonian."""
    import torch
    p = SMALL[name]()
    Hs, _ = kron.H_sector(p)
    w, U = np.linalg.eigh(Hs)
    n = Hs.shape[0]
    plan = lib.Plan(p, k_max=16, tol=1e-10, max_iter=4000, max_rhs=4)
    X0 = torch.zeros((nb, (n + 15) // 16 * 16), dtype=torch.float64, device="cuda"); X0[:, :n] = to_dev(_block(n, nb, 2301))
    rc, th, X, rho, iters, applies = plan.block_lowest_eigenpairs(X0)
    assert rc == lib.DMRG_OK and np.all(rho <= 1e-10) and applies >= nb * 2
    assert np.max(np.abs(th - w[:nb])) <= LAMBDA_ATOL
    Xh = X.cpu().numpy().T
    assert np.max(np.abs(Xh.T @ Xh - np.eye(nb))) <= 1e-9
    for i in range(nb):
        assert np.linalg.norm(Hs @ Xh[:, i] - th[i] * Xh[:, i]) <= 2e-10
    if w[nb] - w[nb - 1] > 1e-6:        # projector on the LAPACK eigenspace
        assert np.max(np.abs(U[:, :nb] @ (U[:, :nb].T @ Xh) - Xh)) <= OVERLAP_DEF
    plan.close()


@pytest.mark.parametrize("name", ["cfg2", "cfg4"])
def test_block_driver_full_config_vs_oracle(lib, name):
    """Full-size configs: the GPU block driver and the oracle's own block run reach the same lowest nb = 2 pairs."""
    import torch
    from dmrg_inputs import CONFIGS
    p = full_config(name)
    lay = rec.Layout(p)
    n = lay.n
    D = rec.diag_H(p, lay)
    k_max = CONFIGS[name]["k_max"]
    X0 = _block(n, 2, 2401)
    ores = obd.block_solve(oracle_apply(p, lay), D, X0.T.copy(), k_max, 1e-10, 3000)
    assert ores["converged"]
    plan = lib.Plan(p, k_max=k_max, tol=1e-10, max_iter=6000, max_rhs=2)
    X0d = torch.zeros((2, (n + 15) // 16 * 16), dtype=torch.float64, device="cuda"); X0d[:, :n] = to_dev(X0)
    rc, th, X, rho, iters, applies = plan.block_lowest_eigenpairs(X0d)
    assert rc == lib.DMRG_OK
    assert np.max(np.abs(th - ores["theta"])) <= LAMBDA_ATOL
    Xh = X.cpu().numpy().T
    if ores["theta"][1] - ores["theta"][0] > 1e-6:
        for i in range(2):
            assert abs(Xh[:, i] @ ores["X"][:, i]) >= 1 - OVERLAP_DEF
    plan.close()


def test_block_of_one_follows_single_vector_path(lib):
    """nb = 1: the block step computes what dmrg_davidson_step computes (other kernels, same mathematics)."""
    import torch
    p = SMALL["cfg2_m160"]()
    lay = rec.Layout(p)
    n = lay.n
    x0 = obd.start_lowest_diag(rec.diag_H(p, lay), 1)[:, 0]      # deterministic start (D): trajectories comparable (A20)
    plan = lib.Plan(p, k_max=8, tol=1e-12, max_rhs=2)
    Va, Wa = plan.new_basis(); Vb, Wb = plan.new_basis()
    plan.davidson_init(Va, Wa, x0=to_dev(x0))
    X0 = torch.zeros((1, Vb.stride(0)), dtype=torch.float64, device="cuda"); X0[0, :n] = to_dev(x0)
    kb, na = plan.block_init(Vb, Wb, X0)
    ka = 1
    for it in range(25):
        ka, lam, rho, ca = plan.davidson_step(Va, Wa, ka)
        kb, na, th, rb, cb = plan.block_step(Vb, Wb, kb, na, 1)
        assert ka == kb and ca == cb
        assert abs(lam - th[0]) <= LAMBDA_ATOL and abs(rho - rb[0]) <= 1e-9 + 1e-6 * rho
    plan.close()


def test_block_errors(lib):
    import torch
    p = SMALL["cfg1"]()
    plan1 = lib.Plan(p, k_max=8)
    V, W = plan1.new_basis()
    X0 = torch.zeros((2, V.stride(0)), dtype=torch.float64, device="cuda")
    with pytest.raises(lib.DmrgError) as e:       # no block workspaces without max_rhs >= 2
        plan1.block_init(V, W, X0)
    assert e.value.code == lib.DMRG_E_INVALID_ARG
    plan1.close()
    plan = lib.Plan(p, k_max=8, max_rhs=2)
    V, W = plan.new_basis()
    X0[0, :plan.n] = 1.0; X0[1, :plan.n] = 2.0    # dependent start vectors -> breakdown
    with pytest.raises(lib.DmrgError) as e:
        plan.block_init(V, W, X0)
        plan.block_step(V, W, 2, 2, 2)
    assert e.value.code == lib.DMRG_E_NUMERIC
    with pytest.raises(lib.DmrgError):
        lib.Plan(p, k_max=8, max_rhs=5)
    plan.close()
