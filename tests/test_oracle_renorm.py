"""Pins of oracle/renorm.py (O-REN: Alg. 1 lines 2, 5-7) against things other than itself: brute-force
ED energies and closed forms (no truncation -> exact), the dense definition rho = Psi Psi^T, the library SVD (Schmidt
weights), and the variational property under truncation."""
import math
import numpy as np
import pytest

from conftest import read_golden
from oracle import renorm, kron, rec


def _gold(N, Delta):
    for name in ("ed_energies.txt", "closed_forms.txt"):
        for model, n, params, sector, e0 in read_golden(name):
            if model == "heisenberg" and n == N and params.get("Delta") == Delta and params.get("J") == 1.0:
                return e0
    return None


@pytest.mark.parametrize("Delta", [1.0, 0.5, 0.0])
def test_untruncated_infinite_dmrg_is_exact(Delta):
    """m larger than every block: enlargement + superblock + (complete) rotation reproduce the open-chain ground-state
    energies N = 4 ... 12 of the golden files (ED / closed forms)."""
    recs = renorm.infinite_dmrg(12, 10 ** 6, 1.0, Delta)
    assert [r["n_sites"] for r in recs] == [4, 6, 8, 10, 12]
    checked = 0
    for r in recs:
        g = _gold(r["n_sites"], Delta)
        if Delta == 0.0:
            g = -sum(math.cos(k * math.pi / (r["n_sites"] + 1)) for k in range(1, r["n_sites"] // 2 + 1))   # XX chain, free fermions
        if g is not None:
            assert abs(r["energy"] - g) <= 1e-10, (r["n_sites"], r["energy"], g)
            checked += 1
        assert max(r["discarded"]) <= 1e-13
    assert checked >= 2
    assert recs[-1]["dim"] == (64, 64) and recs[-1]["n"] == 924


def _state(N_half=4, Delta=0.7):
    L = R = renorm.single_site_block()
    for _ in range(N_half - 1):
        L, R = renorm.enlarge(L, "left", 1.0, Delta), renorm.enlarge(R, "right", 1.0, Delta)
    p = renorm.superblock(L, R, 1.0, Delta, 0)
    Hs, _ = kron.H_sector(p)
    w, v = np.linalg.eigh(Hs)
    return p, rec.Layout(p), v[:, 0]


def test_density_matrix_is_the_partial_trace():
    """rho_L = Psi Psi^T, rho_R = Psi^T Psi with Psi the dense (dim_L x dim_R) wave function: block diagonal in the label,
    the sector blocks are what reduced_density_matrices returns; trace 1, positive semi-definite, same non-zero spectrum."""
    p, lay, x = _state()
    offL = np.concatenate([[0], np.cumsum(p.left.dims)]); offR = np.concatenate([[0], np.cumsum(p.right.dims)])
    Psi = np.zeros((offL[-1], offR[-1]))
    for (i, k) in lay.pairs:
        Psi[offL[i]:offL[i + 1], offR[k]:offR[k + 1]] = lay.seg(x, i, k)
    for side, full, off in (("left", Psi @ Psi.T, offL), ("right", Psi.T @ Psi, offR)):
        rho = renorm.reduced_density_matrices(p, lay, x, side)
        rebuilt = np.zeros_like(full)
        for s, r in enumerate(rho):
            rebuilt[off[s]:off[s + 1], off[s]:off[s + 1]] = r
        assert np.max(np.abs(rebuilt - full)) <= 1e-15
        assert abs(sum(np.trace(r) for r in rho) - 1.0) <= 1e-13
        assert min(np.linalg.eigvalsh(r).min() for r in rho if r.size) >= -1e-15
    sv = np.linalg.svd(Psi, compute_uv=False) ** 2
    for side in ("left", "right"):
        w = np.sort(np.concatenate([np.linalg.eigvalsh(r) for r in renorm.reduced_density_matrices(p, lay, x, side)]))[::-1]
        assert np.max(np.abs(w[:len(sv)] - np.sort(sv)[::-1])) <= 1e-14


@pytest.mark.parametrize("m", [1, 3, 7, 1000])
def test_truncation_keeps_the_largest_schmidt_weights(m):
    p, lay, x = _state()
    rho = renorm.reduced_density_matrices(p, lay, x, "left")
    U, kept, disc = renorm.truncation_basis(rho, m)
    offL = np.concatenate([[0], np.cumsum(p.left.dims)]); offR = np.concatenate([[0], np.cumsum(p.right.dims)])
    Psi = np.zeros((offL[-1], offR[-1]))
    for (i, k) in lay.pairs:
        Psi[offL[i]:offL[i + 1], offR[k]:offR[k + 1]] = lay.seg(x, i, k)
    sv = np.sort(np.linalg.svd(Psi, compute_uv=False) ** 2)[::-1]
    rank = int((sv > 1e-28).sum())
    nk = sum(u.shape[1] for u in U)
    assert nk == min(m, sum(int((np.linalg.eigvalsh(r) > 0).sum()) for r in rho))
    allk = np.sort(np.concatenate(kept))[::-1]
    assert np.max(np.abs(allk[:min(nk, rank)] - sv[:min(nk, rank)])) <= 1e-14       # the library SVD's largest weights
    assert abs(disc - (1.0 - allk.sum())) <= 1e-13
    for u, kw, r in zip(U, kept, rho):
        assert np.max(np.abs(u.T @ u - np.eye(u.shape[1]))) <= 1e-13 if u.shape[1] else True
        assert np.all(np.diff(kw) <= 1e-18)                                        # descending inside a sector
        if u.shape[1]:
            assert np.max(np.abs(r @ u - u * kw[None, :])) <= 1e-13


def test_truncated_run_is_variational_and_accurate():
    """XX chain (Delta = 0): closed form for every N.  With m = 24 kept states the N = 20 energy is an upper bound of the
    exact one (the renormalised basis spans a subspace) and close to it; a smaller m is worse, never better."""
    exact = lambda N: -sum(math.cos(k * math.pi / (N + 1)) for k in range(1, N // 2 + 1))
    r24 = renorm.infinite_dmrg(20, 24, 1.0, 0.0)
    r8 = renorm.infinite_dmrg(20, 8, 1.0, 0.0)
    for a, b in zip(r24, r8):
        e = exact(a["n_sites"])
        assert a["energy"] >= e - 1e-11 and b["energy"] >= a["energy"] - 1e-11
    assert r24[-1]["n_sites"] == 20 and abs(r24[-1]["energy"] - exact(20)) <= 1e-5
    assert r8[-1]["energy"] - exact(20) > 1e-5
    assert max(r24[-1]["dim"]) <= 2 * 24


def test_rotation_of_a_complete_basis_preserves_the_operator_algebra():
    """U complete (m = full): U^T O U has the spectrum of O for H, and [S+, S-] = 2 Sz survives on the boundary site."""
    L = renorm.single_site_block()
    for _ in range(3):
        L = renorm.enlarge(L, "left", 1.0, 0.3)
    rng = np.random.default_rng(2)
    U = [np.linalg.qr(rng.standard_normal((int(d), int(d))))[0] for d in L.sectors.dims]
    Lr = renorm.renormalise(L, U)
    H0, H1 = kron.dense_op(L.H, L.sectors), kron.dense_op(Lr.H, Lr.sectors)
    assert np.max(np.abs(np.linalg.eigvalsh(H0) - np.linalg.eigvalsh(H1))) <= 1e-13
    Sp, Sz = kron.dense_op(Lr.Sp, Lr.sectors), kron.dense_op(Lr.Sz, Lr.sectors)
    assert np.max(np.abs(Sp @ Sp.T - Sp.T @ Sp - 2.0 * Sz)) <= 1e-13
