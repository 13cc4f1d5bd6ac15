"""Parity of dmrg_apply_H (C ABI -> grouped DMMA kernels) with the CPU oracle O-REC / the closed form.

Bar (north_star): max|y_gpu - y_oracle| / max|y_oracle| <= 1e-10 on the same seeded inputs; the GPU
result is bitwise reproducible run to run (no atomics, fixed reduction order)."""
import ctypes as C
import numpy as np
import pytest

from dmrg_inputs import random_vector, heisenberg_synthetic
from dmrg_inputs.problem import Problem, Sectors, BlockOp, HEISENBERG
from dmrg_inputs.synthetic import vector_seed
from oracle import blocks, rec, ed
from gpu_common import small_problems, full_config, fuzz_problem, oracle_apply, rel_maxnorm, to_dev, HPSI_RTOL

pytestmark = pytest.mark.gpu
SMALL = small_problems()


@pytest.fixture(scope="module")
def lib():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_1309_5571_b200 as lib
    lib.load_library()
    return lib


@pytest.mark.parametrize("name", list(SMALL))
def test_apply_matches_oracle_small(lib, name):
    import torch
    p = SMALL[name]()
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=8)
    assert plan.n == lay.n and list(plan.seg_offset) == lay.offset
    assert [(int(a), int(b)) for a, b in zip(plan.left_sector, plan.right_sector)] == lay.pairs
    st = plan.stats()
    assert st["n_pairs"] == len(lay.pairs)
    apply_o = oracle_apply(p, lay)
    for seed in (3001, 3002):
        x = random_vector(lay.n, seed)
        y = plan.apply_H(to_dev(x))
        torch.cuda.synchronize()
        assert rel_maxnorm(y.cpu().numpy(), apply_o(x)) <= HPSI_RTOL
    # diag(H) of the preconditioner (A14)
    Do = rec.diag_H(p, lay)
    assert np.max(np.abs(plan.diag().cpu().numpy() - Do)) <= 1e-13 * max(1.0, np.max(np.abs(Do)))
    # A24 FLOP convention: the library's count never exceeds the oracle's (which also counts D records)
    assert 0 < st["flop_per_apply"] <= rec.flop_count(p, lay)
    plan.close()


def test_cfg1_all_ones_closed_form(lib):
    """RNG-free pin: H applied to the all-ones vector on the S_z = 0 sector of the open 12-site chain is
    w(a)/2 + Delta((N-1) - 2 w(a))/4 with w(a) = number of anti-parallel nearest-neighbour bonds."""
    N, Delta = 12, 1.0
    p = blocks.heisenberg_exact(6, 6, 1.0, Delta)
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=8)
    y = plan.apply_H(to_dev(np.ones(lay.n))).cpu().numpy()
    # basis states of every segment entry: block basis index (sorted by label, stable) -> bit strings
    permL = blocks.block_basis_order(ed.heisenberg_twice_sz(6).reshape(-1, 1))
    permR = blocks.block_basis_order(ed.heisenberg_twice_sz(6).reshape(-1, 1))
    offL = np.concatenate([[0], np.cumsum(p.left.dims)])
    offR = np.concatenate([[0], np.cumsum(p.right.dims)])
    expect = np.zeros(lay.n)
    for (i, k), o in zip(lay.pairs, lay.offset):
        for a in range(p.left.dims[i]):
            for b in range(p.right.dims[k]):
                la, rb = int(permL[offL[i] + a]), int(permR[offR[k] + b])
                bits = [(la >> (5 - s)) & 1 for s in range(6)] + [(rb >> (5 - s)) & 1 for s in range(6)]
                w = sum(1 for s in range(N - 1) if bits[s] != bits[s + 1])
                expect[o + a * p.right.dims[k] + b] = w / 2 + Delta * ((N - 1) - 2 * w) / 4
    assert np.max(np.abs(y - expect)) <= 1e-12
    assert abs(y.sum() / lay.n - (3 - Delta / 4)) <= 1e-12


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5a", "cfg5b", "heis4096", "heis8192"])
def test_apply_matches_oracle_full_config(lib, name):
    """BASELINE.json configs 2-5 (5a literal and 5b paper scale, reading A12) and the two Heisenberg sweep points of
    the headline curve at full size, WHOLE vector against O-REC, in the launch configuration bench.py times.
    (cfg5b / heis8192: ~3e11 FLOP of host BLAS each, a few seconds.)"""
    import torch
    p = full_config(name)
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=4)
    x = random_vector(lay.n, vector_seed(name, "hpsi"))
    xd = to_dev(x)
    y = plan.apply_H(xd)
    y2 = plan.apply_H(xd)
    torch.cuda.synchronize()
    assert torch.equal(y, y2), "apply_H is not bitwise reproducible"
    assert rel_maxnorm(y.cpu().numpy(), oracle_apply(p, lay)(x)) <= HPSI_RTOL
    # Hermiticity at full size: <a, H b> = <H a, b>
    a, b = torch.randn(lay.n, dtype=torch.float64, device="cuda"), torch.randn(lay.n, dtype=torch.float64, device="cuda")
    Ha, Hb = plan.apply_H(a), plan.apply_H(b)
    assert abs(float(a @ Hb - Ha @ b)) <= 1e-11 * float(a.norm() * Hb.norm())
    plan.close()


def _sampled_output_parity(lib, name, picks):
    """Output segments of sampled pairs, each computed one by one from its own records (Eq. 11)."""
    p = full_config(name)
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=2)
    x = random_vector(lay.n, vector_seed(name, "hpsi"))
    y = plan.apply_H(to_dev(x)).cpu().numpy()
    recs = rec.records(p, lay)
    sizes = np.array([int(lay.dl[i]) * int(lay.dr[k]) for i, k in lay.pairs])
    order = np.argsort(-sizes, kind="stable")
    sample = [lay.pairs[order[q]] for q in picks]
    scale = np.max(np.abs(y))
    for out in sample:
        acc = np.zeros((int(lay.dl[out[0]]), int(lay.dr[out[1]])))
        for c, A, B, (i, k), jl in recs:
            if jl != out:
                continue
            T = lay.seg(x, i, k)
            T = T if A is None else A @ T
            T = T if B is None else T @ B.T
            acc += c * T
        got = lay.seg(y, *out)
        assert np.max(np.abs(got - acc)) <= HPSI_RTOL * scale, (name, out)
    st = plan.stats()
    plan.close()
    return st


@pytest.mark.slow
def test_apply_cfg5b_sampled_segments_and_memory(lib):
    """Paper-scale config 5b: besides the whole-vector comparison above, sampled output segments recomputed one by one
    from their own records (an independent path through the oracle's record list), and the peak-memory bound."""
    st = _sampled_output_parity(lib, "cfg5b", [0, 7, 40, -1])
    assert st["device_bytes"] < 40e9


def test_unaligned_vectors_and_bitwise_determinism(lib):
    import torch
    p = SMALL["heis_syn_m300_ragged"]()
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=4)
    x = random_vector(lay.n, 5)
    yo = oracle_apply(p, lay)(x)
    buf_x = torch.zeros(lay.n + 3, dtype=torch.float64, device="cuda")
    buf_y = torch.zeros(lay.n + 3, dtype=torch.float64, device="cuda")
    for ox, oy in ((1, 0), (0, 1), (1, 1), (3, 2)):
        xv = buf_x[ox:ox + lay.n]; xv.copy_(to_dev(x))
        yv = buf_y[oy:oy + lay.n]
        plan.apply_H(xv, yv)
        assert rel_maxnorm(yv.cpu().numpy(), yo) <= HPSI_RTOL
    ys = [plan.apply_H(to_dev(x)).clone() for _ in range(5)]
    assert all(torch.equal(ys[0], t) for t in ys[1:])
    plan.close()


def _tiny(dl, dr, lab_l, lab_r, target):
    """Heisenberg-type problem with random blocks on given sectors (labels 1-D)."""
    rng = np.random.default_rng(77)
    def side(dims, labs):
        H, Sz, Sp = BlockOp(), BlockOp(), BlockOp()
        for s, d in enumerate(dims):
            g = rng.standard_normal((d, d)); H.add(s, s, g + g.T)
            g = rng.standard_normal((d, d)); Sz.add(s, s, g + g.T)
        for s, q in enumerate(labs):
            if q + 1 in labs:
                t = labs.index(q + 1)
                Sp.add(s, t, rng.standard_normal((dims[t], dims[s])))
        return H, Sz, Sp
    HL, SzL, SpL = side(dl, lab_l); HR, SzR, SpR = side(dr, lab_r)
    return Problem(HEISENBERG, 1.0, 0.7, 0.0, 0.0, Sectors(np.array(lab_l).reshape(-1, 1), np.array(dl)),
                   Sectors(np.array(lab_r).reshape(-1, 1), np.array(dr)),
                   {"H_L": HL, "H_R": HR, "Sz_L": SzL, "Sp_L": SpL, "Sz_R": SzR, "Sp_R": SpR}, np.array([target]))


def test_edge_cases(lib):
    import torch
    # empty sectors are skipped (A26); a 1x1 world; one pair only
    for dl, dr, ll, lr, tgt in (([3, 0, 5], [4, 2, 0], [-1, 0, 1], [-1, 0, 1], 0),
                                ([1], [1], [0], [0], 0),
                                ([65, 1], [1, 129], [0, 1], [-1, 0], 0),
                                ([2, 3], [3, 2], [0, 1], [0, 1], 2)):
        p = _tiny(dl, dr, ll, lr, tgt)
        lay = rec.Layout(p)
        plan = lib.Plan(p, k_max=2)
        assert plan.n == lay.n
        x = random_vector(lay.n, 9)
        y = plan.apply_H(to_dev(x)).cpu().numpy()
        assert rel_maxnorm(y, oracle_apply(p, lay)(x)) <= HPSI_RTOL
        plan.close()
    # no admissible pair -> SECTOR error; overlapping x/y -> INVALID_ARG
    with pytest.raises(lib.DmrgError) as e:
        lib.Plan(_tiny([2], [2], [0], [0], 5))
    assert e.value.code == lib.DMRG_E_SECTOR
    p = _tiny([4, 4], [4, 4], [0, 1], [-1, 0], 0)
    plan = lib.Plan(p, k_max=2)
    buf = torch.zeros(2 * plan.n, dtype=torch.float64, device="cuda")
    with pytest.raises(lib.DmrgError) as e:
        plan.apply_H(buf[:plan.n], buf[1:plan.n + 1])
    assert e.value.code == lib.DMRG_E_INVALID_ARG
    plan.close()
    # an operator whose blocks disagree on the label shift (A4)
    bad = _tiny([2, 2, 2], [2, 2, 2], [-1, 0, 1], [-1, 0, 1], 0)
    bad.ops["Sp_L"].add(0, 2, np.ones((2, 2)))
    with pytest.raises(lib.DmrgError) as e:
        lib.Plan(bad)
    assert e.value.code == lib.DMRG_E_SECTOR
    # bad options
    with pytest.raises(lib.DmrgError) as e:
        lib.Plan(p, k_max=40)
    assert e.value.code == lib.DMRG_E_INVALID_ARG


def test_zero_couplings_reduce_to_sylvester_form(lib):
    """J = 0 -> y = H_L X + X H_R^T segment by segment (special case with a library routine)."""
    p = heisenberg_synthetic(120, 3, "gaussian", 0.5, seed=31, J=0.0)
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=2)
    x = random_vector(lay.n, 1)
    y = plan.apply_H(to_dev(x)).cpu().numpy()
    HL = {s: b for s, b in zip(p.ops["H_L"].src, p.ops["H_L"].blocks)}
    HR = {s: b for s, b in zip(p.ops["H_R"].src, p.ops["H_R"].blocks)}
    for (i, k) in lay.pairs:
        X = lay.seg(x, i, k)
        assert np.max(np.abs(lay.seg(y, i, k) - (HL[i] @ X + X @ HR[k].T))) <= 1e-11
    plan.close()


@pytest.mark.parametrize("seed", range(16))
def test_apply_matches_oracle_fuzz(lib, seed, monkeypatch):
    """Random shapes x two planner granularities: the default, and 200 work units per SM, which splits the K range of
    every output tile as finely as the planner allows (split-K partials, last-arriver reduction and the stage-1 ->
    stage-2 counters all exercised on small problems).  Same bar as everywhere: 1e-10 in the max norm, bitwise
    reproducible, and both plans agree to rounding."""
    import torch
    p = fuzz_problem(seed)
    lay = rec.Layout(p)
    x = random_vector(lay.n, 100 + seed)
    want = oracle_apply(p, lay)(x)
    xd = to_dev(x)
    for ups in (None, "200"):
        if ups is None:
            monkeypatch.delenv("DMRG_UNITS_PER_SM", raising=False)
        else:
            monkeypatch.setenv("DMRG_UNITS_PER_SM", ups)
        plan = lib.Plan(p, k_max=2)
        assert plan.n == lay.n
        y = plan.apply_H(xd)
        y2 = plan.apply_H(xd)
        torch.cuda.synchronize()
        assert torch.equal(y, y2)
        assert rel_maxnorm(y.cpu().numpy(), want) <= HPSI_RTOL, (seed, ups)
        plan.close()


def test_two_streams_on_one_plan_are_ordered(lib):
    """include/dmrg_b200.h: a plan serves one call at a time; calls that name different streams are ordered by the library
    (plan-owned event).  Applies of ONE plan issued alternately on two streams, without any synchronisation by the
    caller, must give the bits of the single-stream results (interleaved tickets would give garbage or hang)."""
    import torch
    p = full_config("cfg2")
    lay = rec.Layout(p)
    plan = lib.Plan(p, k_max=4)
    xs = [to_dev(random_vector(lay.n, 700 + i)) for i in range(6)]
    ref = [plan.apply_H(x).clone() for x in xs]
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = [torch.empty_like(x) for x in xs]
    for rep in range(5):
        for i, x in enumerate(xs):
            plan.apply_H(x, outs[i], stream=(s1 if i % 2 == 0 else s2))
    torch.cuda.synchronize()
    for o, r in zip(outs, ref):
        assert torch.equal(o, r)
    plan.close()


def test_reserved_basis_driver_allocates_nothing(lib):
    """options.reserve_basis: the driver's V, W exist after plan creation (no allocation in the hot calls)."""
    import torch
    p = SMALL["cfg2_m160"]()
    plan = lib.Plan(p, k_max=12, tol=1e-9, reserve_basis=True)
    b0 = plan.stats()["device_bytes"]
    assert b0 >= 2 * 8 * plan.n * 12
    rc, lam, x, rho, iters = plan.lowest_eigenpair(None, start_at_argmin_diag=True)
    assert rc == lib.DMRG_OK and plan.stats()["device_bytes"] == b0
    plan.close()


def test_soak_shapes_multi_rhs_and_streamed_input(lib, monkeypatch):
    """40 further random shapes (seeds 1000-1039, per-side dimension up to 900) with the planner's unit size varied from 3 to 200
    units per SM: dmrg_apply_H, dmrg_apply_H_multi with three right-hand sides, and the projected vector that
    dmrg_davidson_step_host returns for a PINNED input (streamed in by loader CTAs) against the oracle -- the ring with stages of
    up to three k-tiles, partial stages, one-k-tile items and the per-segment ready counters all get exercised."""
    import torch
    for seed in range(1000, 1040):
        p = fuzz_problem(seed, m_max=900)
        lay = rec.Layout(p)
        if lay.n == 0:
            continue
        ups = [None, 3, 40, 200][seed % 4]
        if ups:
            monkeypatch.setenv("DMRG_UNITS_PER_SM", str(ups))
        else:
            monkeypatch.delenv("DMRG_UNITS_PER_SM", raising=False)
        plan = lib.Plan(p, k_max=6, max_rhs=3)
        ap = oracle_apply(p, lay)
        x = random_vector(lay.n, 7000 + seed)
        assert rel_maxnorm(plan.apply_H(to_dev(x)).cpu().numpy(), ap(x)) <= HPSI_RTOL, seed
        ld = (lay.n + 15) // 16 * 16
        X = torch.zeros((3, ld), dtype=torch.float64, device="cuda"); Y = torch.empty_like(X)
        xs = [random_vector(lay.n, 8000 + 3 * seed + r) for r in range(3)]
        for r in range(3):
            X[r, :lay.n] = to_dev(xs[r])
        plan.apply_H_multi(X, Y)
        for r in range(3):
            assert rel_maxnorm(Y[r, :lay.n].cpu().numpy(), ap(xs[r])) <= HPSI_RTOL, (seed, r)
        V, W = plan.new_basis()
        plan.davidson_init(V, W, start_at_argmin_diag=True)
        hx = V[0, :lay.n].cpu().pin_memory(); hw = torch.empty(lay.n, dtype=torch.float64).pin_memory()
        plan.davidson_step_host(V, W, 1, hx, hw)
        yo = ap(hx.numpy())
        if np.max(np.abs(yo)) > 0:
            assert rel_maxnorm(hw.numpy(), yo) <= HPSI_RTOL, seed
        assert torch.equal(V[0, :lay.n].cpu(), hx)
        plan.close()


def test_plan_create_destroy_cycle_leaks_nothing(lib):
    """A plan is created per superblock (Alg. 1): every device buffer of a plan is a slice of one allocation, freed by
    dmrg_plan_destroy.  Forty create / apply / destroy cycles over different shapes (both models, with and without a reserved
    basis, one to three right-hand sides) are run twice: the first pass absorbs what the driver reserves once per process (kernel
    images, local-memory pool), across the second the free-memory figure must not move; a plan created afterwards still gives
    the bits of the first one."""
    import torch
    p0 = SMALL["cfg2_m160"]()
    lay0 = rec.Layout(p0)
    x0 = to_dev(random_vector(lay0.n, 4242))
    plan = lib.Plan(p0, k_max=8)
    y_first = plan.apply_H(x0).clone()
    plan.close()
    probs = [fuzz_problem(3000 + it, m_max=400) for it in range(40)]

    def cycle():
        for it, p in enumerate(probs):
            lay = rec.Layout(p)
            if lay.n == 0:
                continue
            plan = lib.Plan(p, k_max=6, max_rhs=1 + it % 3, reserve_basis=bool(it % 2))
            y = plan.apply_H(to_dev(random_vector(lay.n, 5000 + it)))
            assert bool(torch.isfinite(y).all())
            del y
            plan.close()
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        return torch.cuda.mem_get_info()[0]

    free0 = cycle()
    free1 = cycle()
    assert abs(free1 - free0) <= (2 << 20), (free0, free1)
    plan = lib.Plan(p0, k_max=8)
    assert torch.equal(plan.apply_H(x0), y_first)
    plan.close()
