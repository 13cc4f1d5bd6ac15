"""Seeded synthetic DMRG-shaped inputs.

The paper measures on its own DMRG runs with truncated blocks that cannot be
reproduced without a full DMRG code; these generators stand in for them with
the *shapes* of the paper's workload (Table 5: sector
counts, skewed sector sizes, max matrix size, target-sector dimension).

Only random draws and bookkeeping live here -- no arithmetic of the method.
Generator: numpy ``default_rng(seed)`` (PCG64).  Draw order: sizes(L), sizes(R);
then the left block operators in the order of the ``dmrg_problem`` struct,
sectors ascending; then the right block operators; vectors come from a
separate stream.
"""
from __future__ import annotations
import math
import numpy as np
from .problem import Sectors, BlockOp, Problem, HEISENBERG, HUBBARD


def sector_profile(weights: np.ndarray, m: int, rng: np.random.Generator, jitter: float = 0.1) -> np.ndarray:
    """Sector sizes: weights x seeded jitter (1 + jitter*U(-1,1)), largest-remainder
    rounding to sum exactly ``m``, every listed sector >= 1 (reading A11)."""
    w = np.asarray(weights, dtype=np.float64).ravel()
    ns = w.size
    if m < ns:
        raise ValueError("m smaller than the number of sectors")
    w = w * (1.0 + jitter * rng.uniform(-1.0, 1.0, size=ns))
    w = w / w.sum()
    # one state reserved for every sector, the rest apportioned by largest remainder
    quota = w * (m - ns)
    base = np.floor(quota).astype(np.int64)
    rem = quota - base
    short = int((m - ns) - base.sum())
    order = np.argsort(-rem, kind="stable")
    base[order[:short]] += 1
    dims = base + 1
    assert dims.sum() == m and dims.min() >= 1
    return dims.astype(np.int32)


def _sym_block(rng: np.random.Generator, d: int, std: float) -> np.ndarray:
    """Symmetric d x d block: upper triangle incl. diagonal i.i.d. N(0,std^2), mirrored (A10)."""
    g = rng.standard_normal((d, d)) * std
    u = np.triu(g)
    return u + np.triu(g, 1).T


def _heis_side(rng, dims, labels, m, sz_mode):
    ns = len(dims)
    H, Sz, Sp = BlockOp(), BlockOp(), BlockOp()
    std = 1.0 / math.sqrt(m)
    for s in range(ns):
        H.add(s, s, _sym_block(rng, int(dims[s]), 1.0))
    for s in range(ns):
        if sz_mode == "dense":
            Sz.add(s, s, _sym_block(rng, int(dims[s]), std))
        else:  # literal reading of "Sz diagonal in sector label": q * identity (stress input, A8)
            Sz.add(s, s, float(labels[s]) * np.eye(int(dims[s])))
    lab = [int(x) for x in labels]
    for s in range(ns):
        if lab[s] + 1 in lab:
            d = lab.index(lab[s] + 1)
            Sp.add(s, d, rng.standard_normal((int(dims[d]), int(dims[s]))) * std)
    return H, Sz, Sp


def heisenberg_synthetic(m: int, qmax: int, profile: str, Delta: float, seed: int,
                         J: float = 1.0, sigma: float = 1.6, sz_mode: str = "dense") -> Problem:
    """Configs 2-3 of BASELINE.json: Sz sectors -qmax..+qmax, seeded binomial- or
    Gaussian-shaped sizes summing to m; H symmetric block-diagonal N(0,1); Sz
    block-diagonal (dense symmetric N(0,1/m), reading A8); S+ maps q -> q+1 with
    N(0,1/m) entries; target Sz_total = 0."""
    rng = np.random.default_rng(seed)
    q = np.arange(-qmax, qmax + 1)
    if profile == "binomial":
        w = np.array([math.comb(2 * qmax, int(x) + qmax) for x in q], dtype=np.float64)
    elif profile == "gaussian":
        w = np.exp(-(q.astype(np.float64) ** 2) / (2.0 * sigma * sigma))
    else:
        raise ValueError(profile)
    dl = sector_profile(w, m, rng)
    dr = sector_profile(w, m, rng)
    HL, SzL, SpL = _heis_side(rng, dl, q, m, sz_mode)
    HR, SzR, SpR = _heis_side(rng, dr, q, m, sz_mode)
    return Problem(HEISENBERG, J, Delta, 0.0, 0.0,
                   Sectors(q.reshape(-1, 1), dl), Sectors(q.reshape(-1, 1), dr),
                   {"H_L": HL, "H_R": HR, "Sz_L": SzL, "Sp_L": SpL, "Sz_R": SzR, "Sp_R": SpR},
                   np.array([0]))


def _hub_side(rng, dims, labels, m, ell):
    ns = len(dims)
    std = 1.0 / math.sqrt(m)
    H, Cup, Cdn, D = BlockOp(), BlockOp(), BlockOp(), BlockOp()
    lab = [tuple(int(v) for v in x) for x in labels]
    for s in range(ns):
        H.add(s, s, _sym_block(rng, int(dims[s]), 1.0))
    for shift, op in (((1, 0), Cup), ((0, 1), Cdn)):
        for s in range(ns):
            tgt = (lab[s][0] + shift[0], lab[s][1] + shift[1])
            if tgt in lab:
                d = lab.index(tgt)
                op.add(s, d, rng.standard_normal((int(dims[d]), int(dims[s]))) * std)
    for s in range(ns):
        nu, nd = lab[s]
        lo, hi = max(0, nu + nd - ell), min(nu, nd)
        D.add(s, s, np.diag(rng.integers(lo, hi + 1, size=int(dims[s])).astype(np.float64)))
    return H, Cup, Cdn, D


def hubbard_synthetic(m: int, U: float, seed: int, t: float = 1.0, ell: int = 8, sigma: float = 1.2) -> Problem:
    """Configs 4-5 of BASELINE.json: two U(1) labels (N_up, N_dn) in [0,ell]^2, sizes from a
    seeded 2-D Gaussian about (ell/2, ell/2); H symmetric block-diagonal N(0,1); c^dagger_up,
    c^dagger_dn sector-shifting with N(0,1/m) entries; D = diag(seeded double-occupancy counts);
    target N_up = N_dn = ell (half filling of the 2*ell-site superblock)."""
    rng = np.random.default_rng(seed)
    labs = np.array([(a, b) for a in range(ell + 1) for b in range(ell + 1)], dtype=np.int32)
    c = ell / 2.0
    w = np.exp(-((labs[:, 0] - c) ** 2 + (labs[:, 1] - c) ** 2) / (2.0 * sigma * sigma))
    dl = sector_profile(w, m, rng)
    dr = sector_profile(w, m, rng)
    HL, CuL, CdL, DL = _hub_side(rng, dl, labs, m, ell)
    HR, CuR, CdR, DR = _hub_side(rng, dr, labs, m, ell)
    return Problem(HUBBARD, 0.0, 0.0, t, U, Sectors(labs, dl), Sectors(labs, dr),
                   {"H_L": HL, "H_R": HR, "Cup_L": CuL, "Cdn_L": CdL, "Cup_R": CuR, "Cdn_R": CdR,
                    "D_L": DL, "D_R": DR}, np.array([ell, ell]))


class SimpleBlock:
    """An un-enlarged block for the l-1-1-r strategy: sectors (labels = 2 S_z) and the sector-blocked
    operators H (block-diagonal), Sz, Sp (label + 2) of its boundary site.  Container only."""

    def __init__(self, sectors, H, Sz, Sp):
        self.sectors, self.H, self.Sz, self.Sp = sectors, H, Sz, Sp


def heisenberg_block_synthetic(m: int, qmax: int, seed: int, sigma: float = 1.6) -> SimpleBlock:
    """Synthetic un-enlarged block with the shape of a truncated DMRG block (same recipe as `heisenberg_synthetic`, A8-A11):
    sectors 2 S_z = -2 qmax .. 2 qmax in steps of 2 with a seeded Gaussian size profile summing to m, H symmetric N(0,1)
    blocks, Sz dense symmetric N(0,1/m) blocks, S+ blocks N(0,1/m) from label q to q + 2."""
    rng = np.random.default_rng(seed)
    q = np.arange(-qmax, qmax + 1)
    dims = sector_profile(np.exp(-q.astype(np.float64) ** 2 / (2.0 * sigma * sigma)), m, rng)
    H, Sz, Sp = BlockOp(), BlockOp(), BlockOp()
    std = 1.0 / np.sqrt(m)
    for s, d in enumerate(dims):
        d = int(d)
        g = rng.standard_normal((d, d)); H.add(s, s, np.triu(g) + np.triu(g, 1).T)
        g = rng.standard_normal((d, d)) * std; Sz.add(s, s, np.triu(g) + np.triu(g, 1).T)
    for s in range(len(dims) - 1):
        Sp.add(s, s + 1, rng.standard_normal((int(dims[s + 1]), int(dims[s]))) * std)
    return SimpleBlock(Sectors((2 * q).reshape(-1, 1), dims), H, Sz, Sp)


def random_vector(n: int, seed: int) -> np.ndarray:
    """Seeded N(0,1) vector on the n target-sector entries (A19 start (R); H*psi test vectors)."""
    return np.random.default_rng(seed).standard_normal(n)


# BASELINE.json configs (config 1 uses exact blocks, built by oracle.blocks / tests).
CONFIGS = {
    "cfg2": dict(kind="heisenberg", m=512, qmax=8, profile="binomial", Delta=1.0, k_max=16, iters=50),
    "cfg3": dict(kind="heisenberg", m=2048, qmax=16, profile="gaussian", Delta=0.5, k_max=24, iters=100),
    "cfg4": dict(kind="hubbard", m=1024, U=4.0, k_max=16, iters=50),
    "cfg5a": dict(kind="hubbard", m=4096, U=8.0, k_max=32, iters=100),
    "cfg5b": dict(kind="hubbard", m=16384, U=8.0, k_max=32, iters=100),
    # headline-curve sweep (same Heisenberg generator, sigma = 1.6)
    "heis4096": dict(kind="heisenberg", m=4096, qmax=16, profile="gaussian", Delta=0.5, k_max=24, iters=100),
    "heis8192": dict(kind="heisenberg", m=8192, qmax=16, profile="gaussian", Delta=0.5, k_max=24, iters=100),
}
_SEED_INDEX = {"cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5a": 5, "cfg5b": 6, "heis4096": 7, "heis8192": 8}


def make_config(name: str, scale_m: int | None = None) -> Problem:
    """Problem for a named config; operators seeded 1000+c.  ``scale_m`` shrinks the per-side
    dimension (same recipe) for tests the oracle must finish in seconds."""
    c = dict(CONFIGS[name])
    seed = 1000 + _SEED_INDEX[name]
    m = scale_m if scale_m is not None else c["m"]
    if c["kind"] == "heisenberg":
        return heisenberg_synthetic(m, c["qmax"], c["profile"], c["Delta"], seed)
    return hubbard_synthetic(m, c["U"], seed)


def vector_seed(name: str, purpose: str) -> int:
    base = {"start": 2000, "hpsi": 3000}[purpose]
    return base + _SEED_INDEX[name]
