"""Parity of the l-1-1-r strategy (Alg. 2, Eq. 12-13) with the CPU oracle O-L11R:
dmrg_plan_create_l11r + dmrg_apply_H against oracle.l11r.apply (1e-10 in the max norm, north_star), the flat layout, diag(H),
and the lowest eigenpair against brute-force ED values and the dense l-1-1-r operator of the oracle."""
import numpy as np
import pytest

from dmrg_inputs import random_vector
from dmrg_inputs.problem import Sectors, BlockOp
from oracle import l11r, renorm, rec, kron
from gpu_common import rel_maxnorm, to_dev, HPSI_RTOL, LAMBDA_ATOL, OVERLAP_DEF

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lib():
    import torch
    assert torch.cuda.is_available()
    import paper_1309_5571_b200 as lib
    lib.load_library()
    return lib


def _exact(n_block, Delta):
    l = r = renorm.single_site_block()
    for _ in range(n_block - 1):
        l, r = renorm.enlarge(l, "left", 1.0, Delta), renorm.enlarge(r, "right", 1.0, Delta)
    return l, r


def _truncated(n_block, Delta, m):
    l, r = _exact(n_block, Delta)
    L, R = renorm.enlarge(l, "left", 1.0, Delta), renorm.enlarge(r, "right", 1.0, Delta)
    p = renorm.superblock(L, R, 1.0, Delta, 0)
    lay = rec.Layout(p)
    Hs, _ = kron.H_sector(p)
    x = np.linalg.eigh(Hs)[1][:, 0]
    UL, _, _ = renorm.truncation_basis(renorm.reduced_density_matrices(p, lay, x, "left"), m)
    UR, _, _ = renorm.truncation_basis(renorm.reduced_density_matrices(p, lay, x, "right"), m)
    return renorm.renormalise(L, UL), renorm.renormalise(R, UR)


def _random_block(dims, seed):
    """A block with random symmetric H, Sz blocks and random S+ blocks on sectors of the given dims (labels 2 S_z = -k..k step 2):
    not a physical block, but every operator structure the l-1-1-r planner handles, with dims that span several tiles."""
    rng = np.random.default_rng(seed)
    ns = len(dims)
    labels = np.arange(ns) * 2 - (ns - 1)
    H, Sz, Sp = BlockOp(), BlockOp(), BlockOp()
    for s, d in enumerate(dims):
        if d == 0:
            continue
        g = rng.standard_normal((d, d)); H.add(s, s, g + g.T)
        g = rng.standard_normal((d, d)) / np.sqrt(max(d, 1)); Sz.add(s, s, g + g.T)
        if s + 1 < ns and dims[s + 1]:
            Sp.add(s, s + 1, rng.standard_normal((dims[s + 1], d)) / np.sqrt(max(d, 1)))
    return renorm.Block(Sectors(labels.reshape(-1, 1), np.array(dims)), H, Sz, Sp, 0)


def _synth(m, qmax, seed):
    """The generator bench.py's l-1-1-r probe uses (dmrg_inputs.heisenberg_block_synthetic), at a size the oracle finishes."""
    from dmrg_inputs import heisenberg_block_synthetic
    b = heisenberg_block_synthetic(m, qmax, seed)
    return renorm.Block(b.sectors, b.H, b.Sz, b.Sp, 0)


CASES = {
    "exact_1": lambda: (_exact(1, 1.0), 1.0, 0), "exact_2_d05": lambda: (_exact(2, 0.5), 0.5, 0), "exact_4": lambda: (_exact(4, 1.0), 1.0, 0),
    "exact_5_target2": lambda: (_exact(5, 0.7), 0.7, 2), "trunc_5_m12": lambda: (_truncated(5, 1.0, 12), 1.0, 0),
    "random_ragged": lambda: ((_random_block([3, 40, 70, 130, 66, 20, 1], 1), _random_block([2, 33, 65, 129, 64, 17, 1], 2)), 0.8, 0),
    "bench_generator_m160": lambda: ((_synth(160, 3, 71), _synth(160, 3, 72)), 1.0, 0),
    "random_uneven": lambda: ((_random_block([1, 0, 90, 7], 3), _random_block([5, 200, 31, 0, 2], 4)), 1.3, 1),
}


@pytest.mark.parametrize("name", list(CASES))
def test_l11r_apply_layout_diag(lib, name):
    import torch
    (l, r), Delta, target = CASES[name]()
    J = 0.9 if name.startswith("random") else 1.0
    lay = l11r.Layout4(l, r, target)
    plan = lib.Plan.from_l11r(l, r, J, Delta, target, k_max=4)
    assert plan.n == lay.n and list(plan.seg_offset) == lay.offset
    assert [(int(a), int(b)) for a, b in zip(plan.left_sector, plan.right_sector)] == lay.pairs
    for seed in (6001, 6002):
        x = random_vector(lay.n, seed)
        xd = to_dev(x)
        y = plan.apply_H(xd); y2 = plan.apply_H(xd)
        torch.cuda.synchronize()
        assert torch.equal(y, y2)
        assert rel_maxnorm(y.cpu().numpy(), l11r.apply(l, r, J, Delta, lay, x)) <= HPSI_RTOL
    Do = l11r.diag(l, r, J, Delta, lay)
    assert np.max(np.abs(plan.diag().cpu().numpy() - Do)) <= 1e-13 * max(1.0, np.max(np.abs(Do)))
    # Hermiticity through the kernels
    a, b = torch.randn(lay.n, dtype=torch.float64, device="cuda"), torch.randn(lay.n, dtype=torch.float64, device="cuda")
    assert abs(float(a @ plan.apply_H(b) - plan.apply_H(a) @ b)) <= 1e-11 * float(a.norm() * plan.apply_H(b).norm())
    plan.close()


def test_l11r_ground_state_is_the_ed_one(lib):
    """Blocks of 5 sites + 2 sites = the 12-site chain: the lowest eigenpair through the l-1-1-r plan is the ED ground state
    (tests/golden: -5.142090632841) and the one of the LR plan on the enlarged blocks (config 1)."""
    l, r = _exact(5, 1.0)
    plan = lib.Plan.from_l11r(l, r, 1.0, 1.0, 0, k_max=16, tol=1e-10, max_iter=2000)
    assert plan.n == 924
    rc, lam, x, rho, iters = plan.lowest_eigenpair(None, start_at_argmin_diag=True)
    assert rc == lib.DMRG_OK and abs(lam - (-5.142090632841)) <= LAMBDA_ATOL and rho <= 1e-10
    # eigenvector against the oracle's dense l-1-1-r operator
    lay = l11r.Layout4(l, r, 0)
    xg = x.cpu().numpy()
    assert np.linalg.norm(l11r.apply(l, r, 1.0, 1.0, lay, xg) - lam * xg) <= 1e-9
    plan.close()


def test_l11r_fewer_flops_than_lr(lib):
    """the l-1-1-r strategy works on the O(m^2) block operators instead of the O((2m)^2) enlarged ones: same
    superblock, same spectrum (oracle pins), fewer algorithmic FLOP per projection."""
    l, r = _truncated(5, 1.0, 20)
    p4 = lib.Plan.from_l11r(l, r, 1.0, 1.0, 0, k_max=4)
    pl = lib.Plan(renorm.superblock(renorm.enlarge(l, "left", 1.0, 1.0), renorm.enlarge(r, "right", 1.0, 1.0), 1.0, 1.0, 0), k_max=4)
    assert p4.n == pl.n
    assert p4.stats()["flop_per_apply"] < 0.75 * pl.stats()["flop_per_apply"]
    e4 = p4.lowest_eigenpair(None, start_at_argmin_diag=True)[1]; el = pl.lowest_eigenpair(None, start_at_argmin_diag=True)[1]
    assert abs(e4 - el) <= LAMBDA_ATOL
    p4.close(); pl.close()


def test_l11r_rejects_bad_operators(lib):
    l, r = _exact(2, 1.0)
    bad = renorm.Block(l.sectors, l.H, l.Sz, l.Sz, l.n_sites)        # "S+" that does not shift the label
    with pytest.raises(lib.DmrgError) as e:
        lib.Plan.from_l11r(bad, r, 1.0, 1.0, 0)
    assert e.value.code == lib.DMRG_E_SECTOR
