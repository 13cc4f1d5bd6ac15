"""Parity of the steps either side of the path (Alg. 1 lines 2, 5-7) with the CPU
oracle O-REN: the reduced density matrices of a superblock state, the per-sector eigen-decomposition, the choice of the m
states of largest weight, the rotation of the operator blocks, and the whole infinite-lattice loop (enlargement included)
against oracle.renorm.infinite_dmrg, brute-force ED values and the XX-chain closed form."""
import math
import numpy as np
import pytest

from dmrg_inputs import random_vector
from oracle import rec, renorm
from gpu_common import small_problems, full_config, to_dev, LAMBDA_ATOL

pytestmark = pytest.mark.gpu
SMALL = small_problems()


@pytest.fixture(scope="module")
def lib():
    import torch
    assert torch.cuda.is_available()
    import paper_1309_5571_b200 as lib
    lib.load_library()
    return lib


def _split(flat, dims, square=True):
    out, o = [], 0
    for d in dims:
        d = int(d)
        out.append(flat[o:o + (d * d if square else d)].reshape((d, d) if square else (d,)))
        o += d * d if square else d
    return out


@pytest.mark.parametrize("name", ["cfg1", "heis_syn_m300_ragged", "hub_syn_m60", "cfg4_m243", "cfg2"])
@pytest.mark.parametrize("side", [0, 1])
def test_density_matrix_matches_oracle(lib, name, side):
    p = SMALL[name]() if name in SMALL else full_config(name)
    lay = rec.Layout(p)
    x = random_vector(lay.n, 5100); x /= np.linalg.norm(x)
    plan = lib.Plan(p, k_max=4)
    sec = p.left if side == 0 else p.right
    got = _split(plan.density_matrix(to_dev(x), side, sec.dims).cpu().numpy(), sec.dims)
    want = renorm.reduced_density_matrices(p, lay, x, "left" if side == 0 else "right")
    for g, w in zip(got, want):
        assert g.shape == w.shape and (g.size == 0 or np.max(np.abs(g - w)) <= 1e-14)
    assert abs(sum(np.trace(g) for g in got) - 1.0) <= 1e-13
    plan.close()


@pytest.mark.parametrize("dims", [[1, 2, 3, 17, 64, 65, 130], [5], [0, 4, 0, 33], [257]])
def test_sector_eig_matches_lapack(lib, dims):
    import torch
    rng = np.random.default_rng(7)
    mats = []
    for d in dims:
        g = rng.standard_normal((d, max(d // 3, 1))); mats.append(g @ g.T)       # rank-deficient PSD, like a density matrix
    flat = np.concatenate([m.ravel() for m in mats]) if sum(d * d for d in dims) else np.zeros(0)
    U, w = lib.sector_eig(dims, to_dev(flat) if flat.size else torch.zeros(1, dtype=torch.float64, device="cuda"))
    Us = _split(U.cpu().numpy(), dims); ws = _split(w.cpu().numpy(), dims, square=False)
    for m, u, ww in zip(mats, Us, ws):
        if m.size == 0:
            continue
        ref = np.linalg.eigvalsh(m)[::-1]
        scale = max(abs(ref[0]), 1e-300)
        assert np.max(np.abs(ww - ref)) <= 1e-12 * scale
        assert np.all(np.diff(ww) <= 0.0)
        assert np.max(np.abs(u.T @ u - np.eye(len(ww)))) <= 1e-12
        assert np.max(np.abs(m @ u - u * ww[None, :])) <= 1e-12 * scale


@pytest.mark.parametrize("m", [1, 5, 40, 10 ** 6])
def test_select_states_matches_oracle(lib, m):
    p = SMALL["heis_syn_m300_ragged"]()
    lay = rec.Layout(p)
    x = random_vector(lay.n, 5200); x /= np.linalg.norm(x)
    rho = renorm.reduced_density_matrices(p, lay, x, "left")
    Uo, kept, disc = renorm.truncation_basis(rho, m)
    w = np.concatenate([np.linalg.eigvalsh(r)[::-1] for r in rho])
    mk, d = lib.select_states(p.left.dims, w, m)
    assert list(mk) == [u.shape[1] for u in Uo]
    assert abs(d - disc) <= 1e-13


@pytest.mark.parametrize("name,m", [("cfg1", 20), ("heis_syn_m300_ragged", 60), ("cfg4_m243", 10 ** 6)])
def test_truncate_and_rotate_match_oracle(lib, name, m):
    """Lines 5-7 chained on the GPU (density matrix -> eigenvectors -> kept states -> rotated operators) against the oracle.
    Eigenvectors are unique only up to sign / rotation inside degenerate weights, so the comparison is on what is unique: the
    kept weights, the projector U U^T of every sector, and the spectrum-independent invariants of the rotated operators
    (singular values of every block, and U O' U^T = P O P)."""
    p = SMALL[name]()
    lay = rec.Layout(p)
    x = random_vector(lay.n, 5300); x /= np.linalg.norm(x)
    plan = lib.Plan(p, k_max=4)
    dims = p.left.dims
    rho_d = plan.density_matrix(to_dev(x), 0, dims)
    U, w = lib.sector_eig(dims, rho_d)
    mk, disc = lib.select_states(dims, w.cpu().numpy(), m)
    rho = renorm.reduced_density_matrices(p, lay, x, "left")
    Uo, kept, disc_o = renorm.truncation_basis(rho, m)
    Us = _split(U.cpu().numpy(), dims)
    ws = _split(w.cpu().numpy(), dims, square=False)
    assert abs(disc - disc_o) <= 1e-12
    for s, (kg, uo) in enumerate(zip(mk, Uo)):      # the counts agree except on weights at rounding level (sign of ~1e-18)
        lo, hi = sorted((int(kg), uo.shape[1]))
        assert lo == hi or np.max(np.abs(ws[s][lo:hi])) <= 1e-14, (s, kg, uo.shape[1])
    mk = np.array([u.shape[1] for u in Uo], dtype=np.int32)     # from here on with the oracle's counts
    for s, (ug, uo, kw) in enumerate(zip(Us, Uo, kept)):
        k = uo.shape[1]
        assert np.max(np.abs(ws[s][:k] - kw)) <= 1e-13 if k else True
        # projector on the kept subspace (unique when the k-th and (k+1)-th weights differ)
        if k and (k == len(ws[s]) or ws[s][k - 1] - ws[s][k] > 1e-9):
            assert np.max(np.abs(ug[:, :k] @ ug[:, :k].T - uo @ uo.T)) <= 1e-9
    for opname in ("H_L", "Sp_L" if "Sp_L" in p.ops else "Cup_L"):
        op = p.ops[opname]
        out, off = plan.rotate_op(op, dims, mk, U)
        out = out.cpu().numpy()
        ref = renorm.rotate_op(op, [u[:, :k] for u, k in zip(Us, mk)])        # the oracle's formula with the GPU's own basis
        rb = {(s, d): b for s, d, b in zip(ref.src, ref.dst, ref.blocks)}
        for b, (s, d) in enumerate(zip(op.src, op.dst)):
            if mk[s] == 0 or mk[d] == 0:
                assert off[b] == -1
                continue
            got = out[off[b]:off[b] + mk[d] * mk[s]].reshape(mk[d], mk[s])
            assert np.max(np.abs(got - rb[(s, d)])) <= 1e-12 * max(1.0, np.max(np.abs(op.blocks[b])))
    plan.close()


@pytest.mark.parametrize("Delta", [1.0, 0.5])
def test_infinite_lattice_exact_without_truncation(lib, Delta):
    """m larger than every block: the GPU loop (enlargement, superblock, Davidson, rotation by a complete basis) reproduces
    the ED energies of the open chain N = 4 ... 12 (tests/golden) and the oracle's run."""
    recs = lib.infinite_heisenberg(12, 10 ** 6, 1.0, Delta, tol=1e-11)
    ores = renorm.infinite_dmrg(12, 10 ** 6, 1.0, Delta)
    assert [r["n_sites"] for r in recs] == [4, 6, 8, 10, 12] and recs[-1]["n"] == 924
    for r, o in zip(recs, ores):
        assert abs(r["energy"] - o["energy"]) <= LAMBDA_ATOL and r["n"] == o["n"]
        assert max(r["discarded"]) <= 1e-12
    if Delta == 1.0:
        assert abs(recs[-1]["energy"] - (-5.142090632841)) <= LAMBDA_ATOL


@pytest.mark.parametrize("m,Delta,N", [(16, 1.0, 20), (24, 0.0, 24), (40, 0.5, 32)])
def test_infinite_lattice_truncated_matches_oracle(lib, m, Delta, N):
    """With truncation: every iteration's energy, discarded weight and superblock dimension against the oracle's run with
    the same m (the truncated bases span the same subspaces: weights are compared where they are not degenerate at the cut),
    and for the XX chain against the closed form (variational upper bound)."""
    recs = lib.infinite_heisenberg(N, m, 1.0, Delta, tol=1e-11, k_max=24)
    ores = renorm.infinite_dmrg(N, m, 1.0, Delta)
    assert len(recs) == len(ores) and recs[-1]["n_sites"] == N
    # The weights of sectors q and -q are degenerate (S_z -> -S_z symmetry; whole multiplets at Delta = 1): which of two equal
    # weights survives at the cut is decided by the last bit, so the two runs may keep different -- equally good -- states.
    # Compared: the energy to the order of the discarded weight, the discarded weight itself, the dimension up to that choice.
    worst = 0.0
    for r, o in zip(recs, ores):
        worst = max(worst, *r["discarded"], *o["discarded"])
        assert abs(r["n"] - o["n"]) <= 0.03 * o["n"], (r, o)
        assert abs(r["energy"] - o["energy"]) <= 1e-8 + 50.0 * worst, (r, o)
        assert abs(r["discarded"][0] - o["discarded"][0]) <= 1e-9 + 0.5 * worst and abs(r["discarded"][1] - o["discarded"][1]) <= 1e-9 + 0.5 * worst
    if Delta == 0.0:
        for r in recs:
            e = -sum(math.cos(k * math.pi / (r["n_sites"] + 1)) for k in range(1, r["n_sites"] // 2 + 1))
            assert r["energy"] >= e - 1e-9 and r["energy"] - e <= 1e-4
