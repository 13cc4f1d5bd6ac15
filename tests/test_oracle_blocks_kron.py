"""Pins for O-BLK / O-KRON: the LR split + sector blocking reproduces the site-level H entry-wise."""
import math
import numpy as np
import pytest
from conftest import read_golden
from oracle import ed, blocks, kron
from dmrg_inputs.problem import Sectors


def sorted_full_H(H, permL, permR):
    """Site-level H reordered to the composite (sorted left basis) x (sorted right basis) order."""
    mR = len(permR)
    comp = (permL[:, None] * mR + permR[None, :]).ravel()
    return H[np.ix_(comp, comp)]


@pytest.mark.parametrize("l,r,Delta", [(1, 1, 1.0), (2, 2, 0.5), (3, 2, 1.0), (4, 4, 0.5), (6, 6, 1.0)])
def test_heisenberg_lr_equals_site_level(l, r, Delta):
    N = l + r
    p = blocks.heisenberg_exact(l, r, 1.0, Delta, target_twice_sz=N % 2)  # odd N: 2Sz = +1
    H = ed.heisenberg_H_bond(N, 1.0, Delta)
    pl = blocks.block_basis_order(ed.heisenberg_twice_sz(l).reshape(-1, 1))
    pr = blocks.block_basis_order(ed.heisenberg_twice_sz(r).reshape(-1, 1))
    Hk = kron.H_full(p)
    assert np.abs(Hk - sorted_full_H(H, pl, pr)).max() < 1e-14
    Hs, leak = kron.H_sector(p)
    assert leak == 0.0
    assert Hs.shape[0] == math.comb(N, N // 2)   # n_up = ceil(N/2) of N spins
    assert np.array_equal(Hs, Hs.T)


def test_config1_sector_and_energy():
    p = blocks.heisenberg_exact(6, 6, 1.0, 1.0)
    assert list(p.left.dims) == [1, 6, 15, 20, 15, 6, 1]           # SURVEY 8(d) cfg 1
    assert list(p.left.labels.ravel()) == [-6, -4, -2, 0, 2, 4, 6]  # 2*Sz
    Hs, leak = kron.H_sector(p)
    assert Hs.shape == (924, 924) and leak == 0.0                    # C(12,6)
    w = np.linalg.eigvalsh(Hs)
    gold = {(r[0], r[1], r[2].get("Delta")): r[4] for r in read_golden("ed_energies.txt")}
    assert abs(w[0] - gold[("heisenberg", 12, 1.0)]) < 1e-11


@pytest.mark.slow
def test_config1_full_4096_exact_diagonalisation():
    # BASELINE.json config 1: "checked against full 4096x4096 exact diagonalisation":
    # the global ground state of the even AFM chain lies in Sz = 0.
    from scipy.linalg import eigh
    H = ed.heisenberg_H_bond(12, 1.0, 1.0)
    w = eigh(H, eigvals_only=True, subset_by_index=[0, 0])
    assert abs(w[0] - (-5.142090632841)) < 1e-10


@pytest.mark.parametrize("l,r,fold", [(1, 1, False), (2, 2, False), (2, 2, True), (3, 2, False), (2, 3, True)])
def test_hubbard_lr_equals_site_level(l, r, fold):
    t, U = 1.0, 4.0
    p = blocks.hubbard_exact(l, r, t, U, fold_U=fold)
    N = l + r
    H = ed.hubbard_H(N, t, U)
    nuL, ndL = ed.hubbard_counts(l)
    nuR, ndR = ed.hubbard_counts(r)
    pl = blocks.block_basis_order(np.stack([nuL, ndL], 1))
    pr = blocks.block_basis_order(np.stack([nuR, ndR], 1))
    assert np.abs(kron.H_full(p) - sorted_full_H(H, pl, pr)).max() == 0.0  # A6 sign rule: exact
    Hs, leak = kron.H_sector(p)
    assert leak == 0.0 and np.array_equal(Hs, Hs.T)


def test_hubbard_3plus3_energy_golden():
    gold = {(r[0], r[1], r[2].get("U")): r[4] for r in read_golden("ed_energies.txt")}
    p = blocks.hubbard_exact(3, 3, 1.0, 4.0)
    Hs, leak = kron.H_sector(p)
    assert leak == 0.0 and Hs.shape[0] == math.comb(6, 3) ** 2
    assert abs(np.linalg.eigvalsh(Hs)[0] - gold[("hubbard", 6, 4.0)]) < 1e-11
    # U = 0 free-fermion closed form at N = 6 (tests/golden/closed_forms.txt)
    p0 = blocks.hubbard_exact(3, 3, 1.0, 0.0)
    cf = -4 * sum(math.cos(k * math.pi / 7) for k in range(1, 4))
    assert abs(np.linalg.eigvalsh(kron.H_sector(p0)[0])[0] - cf) < 1e-11


@pytest.mark.parametrize("N,Delta", [(4, 1.0), (8, 0.5), (12, 1.0), (12, 0.5)])
def test_all_ones_closed_form(N, Delta):
    """RNG-free pin of the blocked apply layout: (H 1)_a = w(a)/2 + Delta*((N-1) - 2 w(a))/4 with
    w(a) the number of anti-parallel nearest-neighbour bonds of basis state a (Eq. 1)."""
    l = r = N // 2
    p = blocks.heisenberg_exact(l, r, 1.0, Delta)
    Hs, _ = kron.H_sector(p)
    y = Hs @ np.ones(Hs.shape[0])
    perm = blocks.block_basis_order(ed.heisenberg_twice_sz(l).reshape(-1, 1))
    idx = kron.target_index(p)
    m = 2 ** l
    expect = np.zeros(len(idx))
    for pos, comp in enumerate(idx):
        a, b = perm[comp // m], perm[comp % m]     # original l-bit basis indices
        bits = [(a >> (l - 1 - s)) & 1 for s in range(l)] + [(b >> (r - 1 - s)) & 1 for s in range(r)]
        w = sum(bits[s] != bits[s + 1] for s in range(N - 1))
        expect[pos] = w / 2 + Delta * ((N - 1) - 2 * w) / 4
    assert np.abs(y - expect).max() < 1e-13
    if N == 12:
        assert abs(y.sum() / len(y) - (3 - Delta / 4)) < 1e-12
