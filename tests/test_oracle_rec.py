"""Pins for O-REC (block-wise Eq. 11) and diag(H): equal to the Kronecker definition, special cases, invariants."""
import numpy as np
import pytest
from oracle import blocks, kron, rec
from dmrg_inputs import heisenberg_synthetic, hubbard_synthetic
from dmrg_inputs.problem import Problem, Sectors, BlockOp, HEISENBERG


def small_problems():
    return {
        "cfg1": blocks.heisenberg_exact(6, 6, 1.0, 1.0),
        "heis_syn_m40": heisenberg_synthetic(40, 4, "binomial", 1.0, seed=7),
        "heis_syn_m64_label": heisenberg_synthetic(64, 3, "gaussian", 0.5, seed=8, sz_mode="label"),
        "hub_exact_2_2": blocks.hubbard_exact(2, 2, 1.0, 4.0),
        "hub_exact_3_2_fold": blocks.hubbard_exact(3, 2, 1.0, 8.0, fold_U=True),
        "hub_syn_m30": hubbard_synthetic(30, 4.0, seed=9, ell=2),
        "hub_syn_m60": hubbard_synthetic(60, 8.0, seed=10, ell=3),
    }


PROBS = small_problems()


@pytest.mark.parametrize("name", list(PROBS))
def test_blockwise_equals_kron(name):
    p = PROBS[name]
    Hs, leak = kron.H_sector(p)
    assert leak == 0.0
    lay = rec.Layout(p)
    assert lay.n == Hs.shape[0] > 0
    rng = np.random.default_rng(5)
    x = rng.standard_normal(lay.n)
    y = rec.apply_blockwise(p, x, lay)
    yk = Hs @ x
    assert np.abs(y - yk).max() <= 1e-13 * max(1.0, np.abs(yk).max())
    # diag(H) for the preconditioner (A14)
    assert np.abs(rec.diag_H(p, lay) - np.diag(Hs)).max() <= 1e-14 * max(1.0, np.abs(np.diag(Hs)).max())
    # Hermiticity <a, H b> = <H a, b> and linearity
    a, b = rng.standard_normal(lay.n), rng.standard_normal(lay.n)
    Ha, Hb = rec.apply_blockwise(p, a, lay), rec.apply_blockwise(p, b, lay)
    assert abs(a @ Hb - Ha @ b) <= 1e-12 * (np.linalg.norm(a) * np.linalg.norm(Hb))
    assert np.abs(rec.apply_blockwise(p, 2 * a - 3 * b, lay) - (2 * Ha - 3 * Hb)).max() <= 1e-12 * np.abs(Ha).max() * 5


def test_layout_matches_kron_index():
    p = PROBS["hub_syn_m60"]
    lay = rec.Layout(p)
    idx = kron.target_index(p)
    assert lay.n == len(idx)
    # first element of every segment sits at composite index offL[i]*mR + offR[k]
    offL = np.concatenate([[0], np.cumsum(p.left.dims)])
    offR = np.concatenate([[0], np.cumsum(p.right.dims)])
    for (i, k), o in zip(lay.pairs, lay.offset):
        assert idx[o] == offL[i] * p.right.total_dim + offR[k]
        assert idx[o + 1 if p.right.dims[k] > 1 else o] - idx[o] in (0, 1)  # right index fastest


def test_single_sector_reduces_to_plain_matmul():
    # one sector per side -> Eq. 10 itself: X' = sum_a c_a A_a X B_a^T  (library matmul)
    rng = np.random.default_rng(3)
    dl, dr = 5, 7
    sym = lambda d: (lambda g: g + g.T)(rng.standard_normal((d, d)))
    HL, HR, SzL, SzR = sym(dl), sym(dr), sym(dl), sym(dr)
    ops = {n: BlockOp() for n in ("H_L", "H_R", "Sz_L", "Sz_R", "Sp_L", "Sp_R")}
    ops["H_L"].add(0, 0, HL); ops["H_R"].add(0, 0, HR); ops["Sz_L"].add(0, 0, SzL); ops["Sz_R"].add(0, 0, SzR)
    p = Problem(HEISENBERG, 1.7, 0.3, 0, 0, Sectors([[0]], [dl]), Sectors([[0]], [dr]), ops, [0])
    X = rng.standard_normal((dl, dr))
    y = rec.apply_blockwise(p, X.ravel()).reshape(dl, dr)
    assert np.abs(y - (HL @ X + X @ HR.T + 1.7 * 0.3 * SzL @ X @ SzR.T)).max() < 1e-13


def test_J0_reduces_to_sylvester_form():
    p = heisenberg_synthetic(48, 3, "binomial", 1.0, seed=11, J=0.0)
    lay = rec.Layout(p)
    x = np.random.default_rng(1).standard_normal(lay.n)
    y = rec.apply_blockwise(p, x, lay)
    exp = np.zeros_like(y)
    HL = {s: b for s, b in zip(p.ops["H_L"].src, p.ops["H_L"].blocks)}
    HR = {s: b for s, b in zip(p.ops["H_R"].src, p.ops["H_R"].blocks)}
    for (i, k) in lay.pairs:
        lay.seg(exp, i, k)[...] = HL[i] @ lay.seg(x, i, k) + lay.seg(x, i, k) @ HR[k].T
    assert np.abs(y - exp).max() < 1e-12


def mirror(p: Problem) -> Problem:
    sw = {"H_L": "H_R", "H_R": "H_L", "Sz_L": "Sz_R", "Sz_R": "Sz_L", "Sp_L": "Sp_R", "Sp_R": "Sp_L"}
    return Problem(p.model, p.J, p.Delta, p.t, p.U, p.right, p.left, {sw[k]: v for k, v in p.ops.items()}, p.target)


def test_mirror_heisenberg():
    # swapping L<->R and transposing every segment transposes the result
    p = heisenberg_synthetic(40, 4, "gaussian", 0.5, seed=12)
    q = mirror(p)
    lp, lq = rec.Layout(p), rec.Layout(q)
    x = np.random.default_rng(2).standard_normal(lp.n)
    xq = np.zeros(lq.n)
    for (i, k) in lp.pairs:
        lq.seg(xq, k, i)[...] = lp.seg(x, i, k).T
    y, yq = rec.apply_blockwise(p, x, lp), rec.apply_blockwise(q, xq, lq)
    for (i, k) in lp.pairs:
        assert np.abs(lq.seg(yq, k, i) - lp.seg(y, i, k).T).max() < 1e-12


def test_record_and_flop_counts_config1():
    p = PROBS["cfg1"]
    lay = rec.Layout(p)
    recs = rec.records(p, lay)
    assert len(lay.pairs) == 7 and len(recs) == 33
    gemms = sum((A is not None) + (B is not None) for _, A, B, _, _ in recs)
    assert gemms == 52
    # A24 by hand for dims 1,6,15,20,15,6,1 (pairs (q,-q)):
    d = [1, 6, 15, 20, 15, 6, 1]
    f_id = sum(2 * d[i] ** 2 * d[6 - i] + 2 * d[i] * d[6 - i] ** 2 for i in range(7))         # H_L(x)I, I(x)H_R: one GEMM each
    f_zz = sum(2 * d[i] ** 2 * d[6 - i] + 2 * d[i] * d[6 - i] ** 2 for i in range(7))         # Sz(x)Sz: two GEMMs, same shapes
    # S+(x)S- and S-(x)S+ move pair (i, 6-i) to (i+1, 5-i) and back; both association orders cost 2ab(a+b)
    f_pm = 2 * sum(2 * d[i] * d[i + 1] * (d[i] + d[i + 1]) for i in range(6))
    assert (f_id, f_zz, f_pm) == (60736, 60736, 99456)
    assert rec.flop_count(p, lay) == f_id + f_zz + f_pm == 220928


def test_empty_sector_and_no_pair():
    p = heisenberg_synthetic(20, 2, "binomial", 1.0, seed=13)
    p.target = np.array([99], dtype=np.int32)
    assert rec.Layout(p).n == 0
