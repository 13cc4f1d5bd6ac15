"""Pins for O-ED (oracle/ed.py): closed forms, brute-force goldens, algebraic invariants."""
import math
import numpy as np
import pytest
from conftest import read_golden
from oracle import ed


def sector_E0(model, N, params, sector):
    if model == "heisenberg":
        H = ed.heisenberg_H(N, params["J"], params["Delta"]) if N <= 8 else ed.heisenberg_H_bond(N, params["J"], params["Delta"])
        mask = ed.heisenberg_twice_sz(N) == sector["2Sz"]
    else:
        H = ed.hubbard_H(N, params["t"], params["U"])
        nu, nd = ed.hubbard_counts(N)
        mask = (nu == sector["Nup"]) & (nd == sector["Ndn"])
    w, _, _ = ed.lowest_in_sector(H, mask)
    return w[0]


def closed_form(model, N, params):
    if model == "heisenberg":
        if N == 2:
            return -params["J"] * (params["Delta"] / 4 + 0.5)
        if params["Delta"] == 0.0:
            return -params["J"] * sum(math.cos(k * math.pi / (N + 1)) for k in range(1, N // 2 + 1))
        if N == 4 and params["Delta"] == 1.0:
            return -(3 + 2 * math.sqrt(3)) / 4
    else:
        t, U = params["t"], params["U"]
        if U == 0.0:
            return -4 * t * sum(math.cos(k * math.pi / (N + 1)) for k in range(1, N // 2 + 1))
        if N == 2:
            return U / 2 - math.sqrt(U * U / 4 + 4 * t * t)
    raise AssertionError("no closed form")


@pytest.mark.parametrize("row", [r for r in read_golden("closed_forms.txt") if not (r[0] == "hubbard" and r[1] == 6)],
                         ids=lambda r: f"{r[0]}-N{r[1]}-{r[2]}")
def test_closed_forms(row):
    model, N, params, sector, E0 = row
    cf = closed_form(model, N, params)
    assert abs(cf - E0) < 1e-11          # the stored decimal is the formula
    assert abs(sector_E0(model, N, params, sector) - cf) < 1e-11


@pytest.mark.parametrize("row", [r for r in read_golden("ed_energies.txt") if not (r[0] == "hubbard" and r[1] == 6)],
                         ids=lambda r: f"{r[0]}-N{r[1]}-{r[2]}")
def test_bruteforce_goldens(row):
    model, N, params, sector, E0 = row
    assert abs(sector_E0(model, N, params, sector) - E0) < 2e-12 * max(1, abs(E0)) + 1e-11


def test_bond_builder_equals_literal_eq1():
    for N in (2, 3, 5, 8):
        assert np.array_equal(ed.heisenberg_H(N, 1.3, 0.7), ed.heisenberg_H_bond(N, 1.3, 0.7)) or \
            np.abs(ed.heisenberg_H(N, 1.3, 0.7) - ed.heisenberg_H_bond(N, 1.3, 0.7)).max() < 1e-15


def test_spin_algebra_and_embedding():
    # [S+, S-] = 2 Sz ; S- = (S+)^T ; Eq. 2 embedding puts the operator on tensor factor j
    assert np.array_equal(ed.S_PLUS @ ed.S_MINUS - ed.S_MINUS @ ed.S_PLUS, 2 * ed.S_Z)
    N = 4
    for j in range(1, N + 1):
        O = ed.embed(ed.S_Z, j, N)
        for a in range(2 ** N):
            bit = (a >> (N - j)) & 1  # factor j is the j-th most significant bit; 0 = up
            assert O[a, a] == (0.5 if bit == 0 else -0.5)
    # operators on different sites commute (bosonic, L84)
    assert np.array_equal(ed.embed(ed.S_PLUS, 1, 3) @ ed.embed(ed.S_MINUS, 3, 3), ed.embed(ed.S_MINUS, 3, 3) @ ed.embed(ed.S_PLUS, 1, 3))


def test_heisenberg_symmetric_and_conserves_sz():
    for N, D in ((4, 1.0), (6, 0.5)):
        H = ed.heisenberg_H(N, 1.0, D)
        assert np.array_equal(H, H.T)
        q = ed.heisenberg_twice_sz(N)
        assert np.all(H[q[:, None] != q[None, :]] == 0.0)  # block-diagonal in Sz (L96)
    assert np.count_nonzero(ed.heisenberg_twice_sz(12) == 0) == 924  # C(12,6), Fig. 1 (L94)


def test_fermion_anticommutation():
    # {c_p, c_q^+} = delta_pq, {c_p, c_q} = 0 for all modes: pins the Phi strings of Eq. 5-7
    N = 2
    modes = [(j, s) for j in range(1, N + 1) for s in (0, 1)]
    c = {m: ed.hubbard_mode_op(ed.C_ANN, m[0], m[1], N) for m in modes}
    cd = {m: ed.hubbard_mode_op(ed.C_DAG, m[0], m[1], N) for m in modes}
    I = np.eye(4 ** N)
    for p in modes:
        assert np.array_equal(cd[p], c[p].T)
        for q in modes:
            assert np.array_equal(c[p] @ cd[q] + cd[q] @ c[p], I if p == q else 0 * I)
            assert np.array_equal(c[p] @ c[q] + c[q] @ c[p], 0 * I)


def test_hubbard_symmetric_conserves_and_t0_limit():
    N = 3
    H = ed.hubbard_H(N, 1.0, 4.0)
    assert np.array_equal(H, H.T)
    nu, nd = ed.hubbard_counts(N)
    off = (nu[:, None] != nu[None, :]) | (nd[:, None] != nd[None, :])
    assert np.all(H[off] == 0.0)
    # t = 0: diagonal, entries U * (number of doubly occupied sites)
    H0 = ed.hubbard_H(N, 0.0, 3.0)
    assert np.array_equal(H0, np.diag(np.diag(H0)))
    dbl = np.zeros(4 ** N)
    for a in range(4 ** N):
        bits = [(a >> (2 * N - 1 - p)) & 1 for p in range(2 * N)]
        dbl[a] = sum(bits[2 * j] & bits[2 * j + 1] for j in range(N))
    assert np.array_equal(np.diag(H0), 3.0 * dbl)
    assert np.array_equal(np.diag(ed.hubbard_double_occupancy(N)), dbl)
    # mode order: site-major, sigma=-1/2 (s=0, "dn") before +1/2 (s=1, "up")
    up = np.array([sum(((a >> (2 * N - 1 - (2 * j + 1))) & 1) for j in range(N)) for a in range(4 ** N)])
    assert np.array_equal(nu, up)
