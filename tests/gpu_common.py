"""Helpers shared by the -m gpu parity tests: problems, oracle calls, tolerances (north_star)."""
import functools
import numpy as np
from dmrg_inputs import make_config, heisenberg_synthetic, hubbard_synthetic
from oracle import blocks, rec, davidson as odav

HPSI_RTOL = 1e-10      # north_star: max-norm relative error of H*psi
LAMBDA_ATOL = 1e-9     # north_star: lowest eigenvalue, absolute
OVERLAP_DEF = 1e-6     # north_star: |<v_gpu|v_oracle>| >= 1 - 1e-6


def small_problems():
    """Small cases that still span several 64x64 tiles, ragged tails, odd dims and every term type."""
    return {
        "cfg1": lambda: blocks.heisenberg_exact(6, 6, 1.0, 1.0),
        "heis_exact_3_4_d0.5": lambda: blocks.heisenberg_exact(3, 4, 1.0, 0.5, target_twice_sz=1),
        "heis_syn_m40": lambda: heisenberg_synthetic(40, 4, "binomial", 1.0, seed=7),
        "heis_syn_m64_label": lambda: heisenberg_synthetic(64, 3, "gaussian", 0.5, seed=8, sz_mode="label"),
        "heis_syn_m300_ragged": lambda: heisenberg_synthetic(300, 3, "gaussian", 0.5, seed=11, sigma=1.3),
        "heis_syn_m517": lambda: heisenberg_synthetic(517, 5, "gaussian", 1.0, seed=12, J=0.7),
        "hub_exact_2_2": lambda: blocks.hubbard_exact(2, 2, 1.0, 4.0),
        "hub_exact_3_2_fold": lambda: blocks.hubbard_exact(3, 2, 1.0, 8.0, fold_U=True),
        "hub_exact_3_3": lambda: blocks.hubbard_exact(3, 3, 1.0, 4.0),
        "hub_syn_m30": lambda: hubbard_synthetic(30, 4.0, seed=9, ell=2),
        "hub_syn_m60": lambda: hubbard_synthetic(60, 8.0, seed=10, ell=3),
        "hub_syn_m400": lambda: hubbard_synthetic(400, 4.0, seed=13, ell=3),
        "cfg2_m160": lambda: make_config("cfg2", 160),
        "cfg4_m243": lambda: make_config("cfg4", 243),
    }


def fuzz_problem(seed, m_max=700):
    """Seeded random problem shapes beyond the named configs: per-side dimension, sector count, profile width,
    couplings and model all drawn from the seed (generators of dmrg_inputs, no arithmetic of the method here)."""
    rng = np.random.default_rng(90000 + seed)
    m = int(rng.integers(20, m_max))
    if seed % 2 == 0:
        qmax = int(rng.integers(1, 7))
        return heisenberg_synthetic(m, qmax, ["gaussian", "binomial"][int(rng.integers(0, 2))], float(rng.uniform(-1.5, 1.5)),
                                    seed=int(rng.integers(1, 1 << 30)), J=float(rng.uniform(0.2, 2.0)),
                                    sigma=float(rng.uniform(0.6, 2.5)), sz_mode=["dense", "label"][int(rng.integers(0, 2))])
    ell = int(rng.integers(1, 5))
    return hubbard_synthetic(max(m, (ell + 1) ** 2), float(rng.uniform(0.0, 10.0)), seed=int(rng.integers(1, 1 << 30)),
                             t=float(rng.uniform(0.3, 2.0)), ell=ell, sigma=float(rng.uniform(0.7, 2.0)))


@functools.lru_cache(maxsize=4)
def full_config(name):
    return make_config(name)


def oracle_apply(p, lay=None):
    lay = lay or rec.Layout(p)
    recs = rec.records(p, lay)
    return lambda v: rec.apply_blockwise(p, v, lay, recs)


def rel_maxnorm(a, b):
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).cuda()


def basis_to_numpy(T, n, k):
    """(k_max, ldv) device tensor -> n x k Fortran-order numpy (columns = basis vectors)."""
    return np.asfortranarray(T[:k, :n].cpu().numpy().T)
