"""Pins of oracle/l11r.py (O-L11R: Alg. 2 and Eq. 12-13) against things other than itself: the Kronecker
definition (library `np.kron`), brute-force ED energies / closed forms, and the LR superblock of the same chain."""
import math
import numpy as np
import pytest

from conftest import read_golden
from oracle import l11r, renorm, kron


def test_algorithm_2_is_the_kronecker_product():
    rng = np.random.default_rng(4)
    for shapes in (((3, 4), (2, 2), (2, 2), (5, 3)), ((1, 1), (2, 3), (3, 2), (4, 4)), ((6, 2), (1, 2), (2, 1), (2, 7))):
        A, B, C, D = (rng.standard_normal(s) for s in shapes)
        x = rng.standard_normal(A.shape[1] * B.shape[1] * C.shape[1] * D.shape[1])
        want = np.kron(np.kron(np.kron(A, B), C), D) @ x
        assert np.max(np.abs(l11r.project_l11r(A, B, C, D, x) - want)) <= 1e-13 * np.max(np.abs(want))


def _blocks(n_sites, Delta):
    l = r = renorm.single_site_block()
    for _ in range(n_sites - 1):
        l, r = renorm.enlarge(l, "left", 1.0, Delta), renorm.enlarge(r, "right", 1.0, Delta)
    return l, r


def _dense(l, r, Delta, lay):
    H = np.zeros((lay.n, lay.n))
    for q in range(lay.n):
        e = np.zeros(lay.n); e[q] = 1.0
        H[:, q] = l11r.apply(l, r, 1.0, Delta, lay, e)
    return H


@pytest.mark.parametrize("n_block,Delta", [(1, 1.0), (2, 1.0), (3, 1.0), (4, 1.0), (1, 0.5), (3, 0.0), (5, 0.5)])
def test_ground_energy_and_lr_spectrum(n_block, Delta):
    """Blocks of n_block sites each + two sites = a chain of N = 2 n_block + 2 sites: the l-1-1-r operator on the S_z = 0 sector
    is symmetric, has dimension C(N, N/2), the ED / closed-form ground energy, the diagonal `diag` returns, and the spectrum
    of the LR superblock built from the ENLARGED blocks (two ways to express the same H_SB)."""
    N = 2 * n_block + 2
    l, r = _blocks(n_block, Delta)
    lay = l11r.Layout4(l, r, 0)
    assert lay.n == math.comb(N, N // 2)
    H = _dense(l, r, Delta, lay)
    assert np.max(np.abs(H - H.T)) <= 1e-13
    assert np.max(np.abs(np.diag(H) - l11r.diag(l, r, 1.0, Delta, lay))) <= 1e-14
    w = np.linalg.eigvalsh(H)
    gold = None
    for name in ("ed_energies.txt", "closed_forms.txt"):
        for model, n, params, sector, e0 in read_golden(name):
            if model == "heisenberg" and n == N and params.get("Delta") == Delta and params.get("J") == 1.0:
                gold = e0
    if Delta == 0.0:
        gold = -sum(math.cos(k * math.pi / (N + 1)) for k in range(1, N // 2 + 1))
    assert gold is not None and abs(w[0] - gold) <= 1e-10
    L, R = renorm.enlarge(l, "left", 1.0, Delta), renorm.enlarge(r, "right", 1.0, Delta)
    Hs, _ = kron.H_sector(renorm.superblock(L, R, 1.0, Delta, 0))
    assert np.max(np.abs(np.linalg.eigvalsh(Hs) - w)) <= 1e-11


def test_truncated_blocks_and_other_targets():
    """Renormalised (truncated) blocks, target 2 S_z = 2: the l-1-1-r operator still has the spectrum of the LR superblock."""
    l, r = _blocks(4, 0.7)
    p = renorm.superblock(renorm.enlarge(l, "left", 1.0, 0.7), renorm.enlarge(r, "right", 1.0, 0.7), 1.0, 0.7, 0)
    from oracle import rec
    lay2 = rec.Layout(p)
    Hs, _ = kron.H_sector(p)
    x = np.linalg.eigh(Hs)[1][:, 0]
    L, R = renorm.enlarge(l, "left", 1.0, 0.7), renorm.enlarge(r, "right", 1.0, 0.7)
    UL, _, _ = renorm.truncation_basis(renorm.reduced_density_matrices(p, lay2, x, "left"), 9)
    UR, _, _ = renorm.truncation_basis(renorm.reduced_density_matrices(p, lay2, x, "right"), 9)
    lt, rt = renorm.renormalise(L, UL), renorm.renormalise(R, UR)
    for target in (0, 2):
        lay = l11r.Layout4(lt, rt, target)
        H = _dense(lt, rt, 0.7, lay)
        assert np.max(np.abs(H - H.T)) <= 1e-13
        Hs2, _ = kron.H_sector(renorm.superblock(renorm.enlarge(lt, "left", 1.0, 0.7), renorm.enlarge(rt, "right", 1.0, 0.7), 1.0, 0.7, target))
        assert H.shape == Hs2.shape and np.max(np.abs(np.linalg.eigvalsh(H) - np.linalg.eigvalsh(Hs2))) <= 1e-11


def test_block_generator_shapes():
    """dmrg_inputs.heisenberg_block_synthetic (the l-1-1-r bench input): seeded, dims sum to m, H and Sz symmetric and
    block-diagonal, S+ raises the label by 2."""
    from dmrg_inputs import heisenberg_block_synthetic
    a, b = heisenberg_block_synthetic(64, 3, 5), heisenberg_block_synthetic(64, 3, 5)
    assert int(a.sectors.dims.sum()) == 64 and a.sectors.n_sectors == 7
    assert list(a.sectors.labels[:, 0]) == [-6, -4, -2, 0, 2, 4, 6]
    for op, op2 in ((a.H, b.H), (a.Sz, b.Sz), (a.Sp, b.Sp)):
        for x, y in zip(op.blocks, op2.blocks):
            assert np.array_equal(x, y)
    for op in (a.H, a.Sz):
        for s, d, blk in zip(op.src, op.dst, op.blocks):
            assert s == d and np.array_equal(blk, blk.T) and blk.shape == (a.sectors.dims[s],) * 2
    for s, d, blk in zip(a.Sp.src, a.Sp.dst, a.Sp.blocks):
        assert d == s + 1 and blk.shape == (a.sectors.dims[d], a.sectors.dims[s])
