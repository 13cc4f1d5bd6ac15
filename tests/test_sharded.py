"""Output sharding: the LPT owner table (host logic of the C library, no GPU needed), the
all-reduce plumbing on CPU with gloo and world_size 2 (each rank applies the records of the outputs it owns -- here through
the oracle -- and the sum must be the whole projection), and on one GPU the sharded plans of R = 2, 3 emulated ranks."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_outputs_is_lpt():
    import paper_1309_5571_b200 as lib
    rng = np.random.default_rng(1)
    cost = rng.integers(1, 10 ** 9, size=81)
    for R in (1, 2, 3, 8):
        own = lib.binding.partition_outputs(cost, R)
        assert own.min() >= 0 and own.max() < R
        load = np.array([cost[own == r].sum() for r in range(R)])
        # LPT guarantee: max load <= mean + largest item; and the table is the textbook greedy one
        assert load.max() <= cost.sum() / R + cost.max()
        ref_load = np.zeros(R, dtype=np.int64); ref = np.zeros(81, dtype=np.int32)
        for q in sorted(range(81), key=lambda q: (-int(cost[q]), q)):
            r = int(np.argmin(ref_load)); ref[q] = r; ref_load[r] += cost[q]
        assert np.array_equal(own, ref)
    assert np.array_equal(lib.binding.partition_outputs([5, 5, 5, 5], 2), [0, 1, 0, 1])     # ties: lower index first, lower rank first


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import paper_1309_5571_b200 as lib
from paper_1309_5571_b200.sharded import sharded_apply
from dmrg_inputs import make_config, random_vector
from oracle import rec
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
p = make_config("cfg4", 120); lay = rec.Layout(p); recs = rec.records(p, lay)
pair_index = {{pr: q for q, pr in enumerate(lay.pairs)}}
cost = np.zeros(len(lay.pairs), dtype=np.int64)
for c, A, B, (i, k), jl in recs:
    di, dk, dj, dl = int(lay.dl[i]), int(lay.dr[k]), int(lay.dl[jl[0]]), int(lay.dr[jl[1]])
    cost[pair_index[jl]] += 2 * dj * di * dk if B is None else (2 * di * dk * dl if A is None else min(2*di*dk*dl + 2*dj*di*dl, 2*dj*di*dk + 2*dj*dk*dl))
own = lib.binding.partition_outputs(cost, world)
mine = [r for r in recs if own[pair_index[r[4]]] == rank]
def apply_local(x, y):
    y += torch.from_numpy(rec.apply_blockwise(p, x.numpy(), lay, mine))
x = torch.from_numpy(random_vector(lay.n, 3100)); y = torch.empty_like(x)
sharded_apply(apply_local, x, y, dist)
full = rec.apply_blockwise(p, x.numpy(), lay, recs)
print(json.dumps({{"rank": rank, "err": float(np.max(np.abs(y.numpy() - full))), "owned": int((own == rank).sum()), "n_out": len(own),
                  "sum": float(y.sum())}}), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    import socket
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as s:
        s.bind(("127.0.0.1", 0))
        return str(s.getsockname()[1])


def test_sharded_apply_gloo_world_size_2(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(WORKER.format(root=ROOT))
    outs = None
    for attempt in range(3):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=_free_port(), OMP_NUM_THREADS="1", WORLD_SIZE="2")
        procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)), stdout=subprocess.PIPE,
                                  stderr=subprocess.PIPE, text=True) for r in range(2)]
        res = [p.communicate(timeout=300) for p in procs]
        if all(p.returncode == 0 for p in procs):
            outs = [json.loads([l for l in o.splitlines() if l.startswith("{")][-1]) for o, _ in res]
            break
    assert outs is not None, res
    assert sum(o["owned"] for o in outs) == outs[0]["n_out"] and min(o["owned"] for o in outs) > 0
    for o in outs:
        assert o["err"] <= 1e-12
    assert outs[0]["sum"] == outs[1]["sum"]          # every rank holds the same bits after the all-reduce


@pytest.mark.gpu
@pytest.mark.parametrize("name,R", [("cfg2_m160", 2), ("cfg4_m243", 3), ("heis_syn_m517", 2)])
def test_sharded_plans_on_one_gpu(name, R):
    """R emulated ranks on one GPU, one after the other (no kernel waits on another): every output segment is written by
    exactly its owner, the sum over ranks is the whole projection (oracle, 1e-10), and Alg. 3 with the sharded line 2
    (dmrg_davidson_step_given_w) follows the unsharded run."""
    import torch
    import paper_1309_5571_b200 as lib
    from paper_1309_5571_b200.sharded import sharded_apply
    from dmrg_inputs import random_vector
    from oracle import rec
    from gpu_common import small_problems, oracle_apply, rel_maxnorm, to_dev, HPSI_RTOL, LAMBDA_ATOL
    p = small_problems()[name]()
    lay = rec.Layout(p)
    plans = [lib.Plan(p, k_max=8, tol=1e-10, shard_rank=r, shard_count=R) for r in range(R)]
    ref = lib.Plan(p, k_max=8, tol=1e-10)
    own = plans[0].shard_owner()
    assert all(np.array_equal(own, q.shard_owner()) for q in plans) and set(own) == set(range(R))
    x = to_dev(random_vector(lay.n, 3200))
    ys = [sharded_apply(lambda a, b, q=q: q.apply_H(a, b), x, torch.empty_like(x)) for q in plans]
    for q, (i, k) in enumerate(lay.pairs):
        sl = slice(lay.offset[q], lay.offset[q] + int(lay.dl[i]) * int(lay.dr[k]))
        for r in range(R):
            if r != own[q]:
                assert float(ys[r][sl].abs().max()) == 0.0
    total = sum(ys)
    assert rel_maxnorm(total.cpu().numpy(), oracle_apply(p, lay)(x.cpu().numpy())) <= HPSI_RTOL
    assert float((total - ref.apply_H(x)).abs().max()) <= 1e-12 * float(total.abs().max())
    # Davidson: line 2 sharded (sum over the emulated ranks stands in for the all-reduce), lines 3-14 on rank 0's plan
    V, W = plans[0].new_basis(); Vr, Wr = ref.new_basis()
    plans[0].davidson_init(V, W, start_at_argmin_diag=True); ref.davidson_init(Vr, Wr, start_at_argmin_diag=True)
    k = kr = 1
    n = lay.n
    for it in range(30):
        W[k - 1, :n] = sum(sharded_apply(lambda a, b, q=q: q.apply_H(a, b), V[k - 1, :n], torch.empty(n, dtype=torch.float64, device="cuda")) for q in plans)
        k, lam, rho, conv = plans[0].davidson_step_given_w(V, W, k)
        kr, lam_r, rho_r, conv_r = ref.davidson_step(Vr, Wr, kr)
        assert k == kr and conv == conv_r and abs(lam - lam_r) <= LAMBDA_ATOL and abs(rho - rho_r) <= 1e-9 + 1e-6 * rho_r
    for q in plans + [ref]:
        q.close()
