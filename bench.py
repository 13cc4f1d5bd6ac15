#!/usr/bin/env python
"""bench.py -- throughput of the DMRG hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg3]

Workload (BASELINE.json configs[2], the one the metric is quoted on: "m=2048"): Heisenberg
spin-1/2, Delta=0.5, synthetic blocks m=2048 per side, Sz sectors -16..16, target Sz=0
(n ~ 7.3e5), Davidson basis limit k_max=24, deterministic start e_argmin(D).  Inputs are seeded
and synthetic.

A step = one call of Alg. 3 = one pass of the whole hot path: the projection
W(:,k) = H_SB V(:,k) (one grouped DMMA launch running both GEMM stages) plus every BLAS-2 row of SURVEY 8(a) (V^T w, small
eig, residual + preconditioner, Gram-Schmidt, normalise/append, restart collapse when due), through
the C ABI (dmrg_davidson_step), basis size cycling 1..k_max as in a real run.

value   = algorithmic FP64 GFLOP/s of the whole step (A24 FLOP of the apply + BLAS-2 FLOP) with
          everything resident in HBM; L2 is flushed between timed steps (outside the event pairs).
e2e     = same metric with host buffers through dmrg_davidson_step_host: every step copies the newest basis
          vector host->device from pinned memory and the projected vector W(:,k) device->host (the
          per-iteration crossing of the paper's hybrid scheme: H2D of the input, D2H of the output,
          PAPER.md:L263, L432-445 Alg. 7); the D2H runs on a side stream under lines 3-13, one
          synchronising call per step.
roofline= the grouped DMMA kernel (one launch per step) against the FP64 DMMA peak measured live.
davidson_hbm = the BLAS-2 kernels timed inside running steps at config 5b (n ~ 1.5e7: V, W >> L2) against the
          measured HBM copy bandwidth (the >= 75 % judgement is taken where V >> L2).
cpu_baseline / --impl reference = the oracle's O-DAV iteration (oracle/, numpy) on the host cores.
"""
from __future__ import annotations
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "fp64_gflops_davidson_iteration"   # H*psi + Davidson BLAS-2, algorithmic FLOP / time
UNIT = "GFLOP/s"


def blas2_flop(n: int, k: int, k_eff: int, reorth: int) -> float:
    """FLOP of the BLAS-2 rows of one step: V^T w 2nk; x, Wy 4nk (+4n); reorth x (2nk' + 2nk' + 2n); n."""
    return 2.0 * n * k + 4.0 * n * k + 4.0 * n + reorth * (4.0 * n * k_eff + 2.0 * n) + n


def blas2_bytes(n: int, k: int, k_eff: int, reorth: int, restart: bool) -> float:
    """Algorithmic bytes of the BLAS-2 rows of one step (with the V^T t of the first Gram-Schmidt pass
    sharing the residual pass over V: 8 n (4k + 7) per step instead of 8 n (5k + 8))."""
    b = 8.0 * n * (k + 1)                       # a3  V^T w
    b += 8.0 * n * (2 * k) + 16.0 * n           # a5-a7 fused: V, W, D read, t written
    if restart:
        b += 16.0 * n + 32.0 * n                # x, Wy written; collapse reads them and writes V0, W0
    # a8: t -= V s reads V, t and writes t; the read of V for s = V^T t is shared with the residual pass on steps without
    # a restart (fused kernel), and is a pass of its own on restart steps and on a second Gram-Schmidt pass
    b += reorth * (8.0 * n * (k_eff + 1) + 8.0 * n) + (reorth - (0 if restart else 1)) * 8.0 * n * (k_eff + 1)
    b += 16.0 * n                               # a9
    return b


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [t.strip() for t in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = [float(r[0]) for r in rows]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for j, nm in enumerate(names) if any(r[3 + j].lower().startswith("active") for r in rows)]
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(float(r[2]) for r in rows)}


def make_problem(name: str):
    from dmrg_inputs import make_config, CONFIGS
    return make_config(name), CONFIGS[name]


def oracle_iteration_timer(problem, k_max: int, steps: int, warmup: int):
    """Times the oracle's O-DAV step (oracle/davidson.py on oracle/rec.py) as it stands."""
    from oracle import rec, davidson as odav
    try:
        from threadpoolctl import threadpool_info
        cores = max([d.get("num_threads", 1) for d in threadpool_info()] or [os.cpu_count() or 1])
    except Exception:
        cores = os.cpu_count() or 1
    lay = rec.Layout(problem)
    recs = rec.records(problem, lay)
    D = rec.diag_H(problem, lay)
    apply_o = lambda v: rec.apply_blockwise(problem, v, lay, recs)
    st = odav.init_state(odav.start_argmin_diag(D), k_max)
    flop_apply = rec.flop_count(problem, lay)
    times, flops = [], []
    for it in range(warmup + steps):
        k = st.k
        k_eff = 1 if k == k_max else k
        t0 = time.perf_counter()
        res = odav.davidson_step(st, apply_o, D, 1e-10, 1)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
            flops.append(flop_apply + blas2_flop(lay.n, k, k_eff, 1))
        if res["converged"]:
            st = odav.init_state(odav.start_argmin_diag(D), k_max)
    return sum(flops) / sum(times) / 1e9, sum(times) / len(times) * 1e3, cores, lay.n


def host_description() -> dict:
    """CPU model, core count and BLAS library behind numpy (printed beside the oracle timing)."""
    out = {"os_cpu_count": os.cpu_count()}
    try:
        for l in open("/proc/cpuinfo"):
            if l.startswith("model name"):
                out["cpu_model"] = l.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    try:
        from threadpoolctl import threadpool_info
        out["blas"] = [{k: d.get(k) for k in ("internal_api", "version", "num_threads", "threading_layer")} for d in threadpool_info()]
    except Exception:
        pass
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    problem, cfg = make_problem(args.config)
    steps = min(args.steps, 60)
    gfl, ms, cores, n = oracle_iteration_timer(problem, cfg["k_max"], steps, max(1, min(args.warmup, 3)))
    line = {"impl": "reference", "metric": METRIC, "value": gfl, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": workload_config(args.config, cfg, n, None),
            "cpu_baseline": {"value": gfl, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{steps} consecutive O-DAV iterations (oracle/davidson.py on oracle/rec.py) of {args.config} from start e_argmin(D)"},
            "e2e": {"value": gfl, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(name, cfg, n, stats):
    c = {"workload": f"{name}: {cfg['kind']} m={cfg['m']} per side, k_max={cfg['k_max']}, target sector dim n={n}, "
                     "one Davidson iteration (Alg. 3) per step, start e_argmin(D)",
         "l2": "flushed between timed steps (256 MiB memset outside the event pairs)", "parallelism": "replicas only"}
    if stats:
        c.update({"n_records": stats["n_records"], "n_gemms": stats["n_gemms"], "flop_per_apply": stats["flop_per_apply"]})
    return c


def gemv_trans_probe(plan, V, W, flush, hbm_peak):
    """The paper's own BLAS-2 benchmark shape (Fig. 6-10: V^T x for a ~5e5 x 16..20 matrix, no host
    transfer): dmrg_gemv_trans alone on this config's n, one launch per event pair, L2 flushed before every launch
    (cold) and back to back (warm; V fits the 126 MB L2 up to k ~ 20 at cfg3).  Context only: the >= 75 % HBM judgement
    is taken at cfg5b (`davidson_hbm`)."""
    import torch
    n = plan.n
    stream = torch.cuda.current_stream()
    out = {"n": int(n), "paper": "114.7 GB/s (GTX 570, 75 % of 152), 143.7 GB/s (K20, 69 % of 208) at 16 x 5e5, PAPER.md:L316-326"}
    res = torch.empty(32, dtype=torch.float64, device=V.device)
    w = W[0, :n]
    for k in (16, 20):
        if k > V.shape[0]:
            continue
        cold = []
        for _ in range(12):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); plan.gemv_trans(V, k, w, res); e1.record(stream)
            torch.cuda.synchronize()
            cold.append(e0.elapsed_time(e1))
        for _ in range(3):
            plan.gemv_trans(V, k, w, res)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(50):
            plan.gemv_trans(V, k, w, res)
        e1.record(stream); torch.cuda.synchronize()
        warm = e0.elapsed_time(e1) / 50
        b = 8.0 * n * (k + 1) + 8.0 * k
        c = float(np.median(cold))
        out[f"k{k}"] = {"us_cold": c * 1e3, "gbs_cold": b / (c * 1e-3) / 1e9, "frac_hbm_cold": b / (c * 1e-3) / 1e9 / hbm_peak,
                        "us_warm": warm * 1e3, "gbs_warm": b / (warm * 1e-3) / 1e9}
    return out


def davidson_hbm_probe(lib, device, hbm_peak, name="cfg5b", steps=36, hbm_read=None):
    """BLAS-2 kernels inside running Davidson steps at a config whose basis is far larger than L2.  GB/s = ALGORITHMIC
    bytes / device time; the fused residual pass re-reads V for s = V^T t out of L1/L2, so a figure above
    the copy bandwidth is L2 assistance, not HBM traffic (profiles/r2_davidson_dram.md has the dram__bytes counters).
    Two denominators: the read+write copy bandwidth of MEASURED_PEAKS.json and a live read-only stream probe."""
    import torch
    problem, cfg = make_problem(name)
    k_max = cfg["k_max"]
    plan = lib.Plan(problem, k_max=k_max, tol=1e-10, device=device)
    n = plan.n
    V, W = plan.new_basis()
    plan.davidson_init(V, W, start_at_argmin_diag=True)
    plan.set_timing(True)
    k = 1
    acc = {"vtw": [0.0, 0.0], "residual": [0.0, 0.0], "orthogonalise": [0.0, 0.0], "append": [0.0, 0.0]}
    t_apply = []
    for it in range(steps):
        kk = k
        k, lam, rho, conv = plan.davidson_step(V, W, k)
        tm = plan.get_timing()
        if it >= 3 and kk < k_max:
            ke = kk
            for nm, b, ms in (("vtw", 8.0 * n * (kk + 1), tm[2]), ("residual", 8.0 * n * 2 * kk + 16.0 * n, tm[4]),
                              ("orthogonalise", 8.0 * n * (ke + 1) + 8.0 * n, tm[6]), ("append", 16.0 * n, tm[7])):
                acc[nm][0] += b; acc[nm][1] += ms
            t_apply.append(tm[0])
        if conv:
            break
    st = plan.stats()
    out = {"workload": f"{name}: {cfg['kind']} m={cfg['m']} per side, n={n}, k = 4..{k_max - 1}, V and W {2 * V.numel() * 8 / 1e9:.1f} GB",
           "kernels_gbs": {nm: v[0] / (v[1] * 1e-3) / 1e9 for nm, v in acc.items() if v[1] > 0},
           "hbm_peak_gbs": hbm_peak}
    tot_b = sum(v[0] for v in acc.values()); tot_ms = sum(v[1] for v in acc.values())
    if acc["append"][1] > 0:    # a9 also writes the two 8 KB-tile images of the new vector (16 n bytes more) that the projection reads
        out["append_gbs_incl_tile_images"] = 2.0 * acc["append"][0] / (acc["append"][1] * 1e-3) / 1e9
        out["append_note"] = ("'append' above counts SURVEY 8(d)'s 16 n bytes (t read, v_k written); the kernel moves 32 n: it also writes "
                              "the P and Q tile images of v_k, the repack the projection kernel would otherwise do in its phase 0")
    out["blas2_gbs"] = tot_b / (tot_ms * 1e-3) / 1e9
    out["blas2_frac_hbm"] = out["blas2_gbs"] / hbm_peak
    out["kernels_frac_hbm"] = {nm: g / hbm_peak for nm, g in out["kernels_gbs"].items()}
    if hbm_read:
        out["hbm_read_probe_gbs"] = hbm_read
        out["kernels_frac_hbm_read"] = {nm: g / hbm_read for nm, g in out["kernels_gbs"].items()}
        out["blas2_frac_hbm_read"] = out["blas2_gbs"] / hbm_read
    out["apply_tflops"] = st["flop_per_apply"] / (sum(t_apply) / len(t_apply) * 1e-3) / 1e12
    out["device_bytes"] = st["device_bytes"] + 2 * V.numel() * 8
    out["peak_allocated_bytes"] = int(torch.cuda.max_memory_allocated())
    plan.close()
    del V, W
    return out


def job_throughput(local_ms: float, local_flop: float, world: int, dist=None, device="cpu"):
    """Whole-job metric of N replicas (replicas only, no data-path collective): the time of the
    job is the MAX over ranks of the device-timed region, the work is the sum over ranks.  Returns (max_ms, GFLOP/s)."""
    if dist is None or world == 1:
        return local_ms, local_flop / (local_ms * 1e-3) / 1e9
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    f = torch.tensor([local_flop], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(f, op=dist.ReduceOp.SUM)
    return float(t.item()), float(f.item()) / (float(t.item()) * 1e-3) / 1e9


def run_ours(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_1309_5571_b200 as lib
    lib.load_library()

    problem, cfg = make_problem(args.config)
    k_max, reorth = cfg["k_max"], 1
    plan = lib.Plan(problem, k_max=k_max, tol=1e-10, reorth=reorth, device=f"cuda:{local}")
    st = plan.stats()
    n = plan.n
    V, W = plan.new_basis()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{local}")
    stream = torch.cuda.current_stream()

    def restart_run():
        plan.davidson_init(V, W, start_at_argmin_diag=True)
        return 1

    # ---- device-resident timing: W warm-up + K timed steps, per-step event pairs, L2 flushed between
    def timed_run(steps, warmup, host_io, enqueue_only=False):
        """enqueue_only: steps are enqueued without a host synchronisation (dmrg_davidson_step with NULL outputs, the
        way dmrg_lowest_eigenpair runs its loop) and the state is polled every 8 steps OUTSIDE the event pairs; returns
        None if the run converged on the way (the steps enqueued after that were no-ops) so the caller can fall back."""
        k = restart_run()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        ks = []
        l0 = 0
        hx = torch.empty(n, dtype=torch.float64).pin_memory() if host_io else None
        hw = torch.empty(n, dtype=torch.float64).pin_memory() if host_io else None
        if host_io:
            hx.copy_(V[0, :n])
        for it in range(warmup + steps):
            flush.zero_()
            j = it - warmup
            if j == 0:
                l0 = plan.stats()["launches"]
            if j >= 0:
                ev[j][0].record(stream)
                ks.append(k)
            if host_io:   # newest basis vector in, projected vector out (pinned host buffers): dmrg_davidson_step_host
                k, lam, rho, conv = plan.davidson_step_host(V, W, k, hx, hw)     # copies + step, synchronises
            elif enqueue_only:
                k, conv = plan.davidson_enqueue(V, W, k), False
            else:
                k, lam, rho, conv = plan.davidson_step(V, W, k)
            if j >= 0:
                ev[j][1].record(stream)
            if enqueue_only and ((it + 1) % 8 == 0 or it + 1 == warmup + steps):
                if plan.davidson_poll()[2]:
                    return None
            if host_io and not conv:
                hx.copy_(V[k - 1, :n])          # next step's input staged on the host (not timed as H2D yet)
            if conv:
                l0 -= plan.stats()["launches"]
                k = restart_run()               # a new run's start vector is not part of the timed steps
                l0 += plan.stats()["launches"]
                if host_io:
                    hx.copy_(V[0, :n])
        torch.cuda.synchronize()
        ms = [a.elapsed_time(b) for a, b in ev]
        return ms, ks, plan.stats()["launches"] - l0

    # one-time set-up, like the plan: a CUDA graph per basis size is captured at the first step that reaches that size, so one
    # untimed pass through a whole restart cycle comes before the W warm-up steps (otherwise the captures -- host time during
    # which the GPU idles -- would fall into the first k_max timed steps)
    k = restart_run()
    for _ in range(k_max + 2):
        k = plan.davidson_enqueue(V, W, k)
    plan.davidson_poll()
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    t0 = time.time()
    res = timed_run(args.steps, args.warmup, host_io=False, enqueue_only=True)
    step_mode = "enqueued back to back (dmrg_davidson_step with NULL outputs), state polled every 8 steps outside the event pairs"
    if res is None:     # converged inside the run: time it with one synchronising call per step and restarts instead
        res = timed_run(args.steps, args.warmup, host_io=False)
        step_mode = "one synchronising dmrg_davidson_step per step, restart on convergence"
    ms, ks, gpu_launches = res
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t1 = time.time()
    total_ms = sum(ms)
    flop_step = [st["flop_per_apply"] + blas2_flop(n, k, 1 if k == k_max else k, reorth) for k in ks]
    total_ms, value = job_throughput(total_ms, sum(flop_step), world, dist, f"cuda:{local}")

    # ---- end to end with host buffers
    ms_e2e, ks_e, _ = timed_run(args.steps, args.warmup, host_io=True)
    tot_e = sum(ms_e2e)
    flop_e = [st["flop_per_apply"] + blas2_flop(n, k, 1 if k == k_max else k, reorth) for k in ks_e]
    tot_e, e2e_val = job_throughput(tot_e, sum(flop_e), world, dist, f"cuda:{local}")

    # ---- per-kernel device times of the same loop (library event pairs on the launching stream), warm L2
    plan.set_timing(True)
    k = restart_run()
    kt = np.zeros(8); bytes_b2 = 0.0; nsteps_t = 0; t_b2 = 0.0
    for it in range(args.warmup + args.steps):
        kk = k
        k, lam, rho, conv = plan.davidson_step(V, W, k)
        if it >= args.warmup:
            tm = plan.get_timing()
            kt += tm; nsteps_t += 1
            bytes_b2 += blas2_bytes(n, kk, 1 if kk == k_max else kk, reorth, kk == k_max)
            t_b2 += tm[2] + tm[4] + tm[5] + tm[6] + tm[7]
        if conv:
            k = restart_run()
    plan.set_timing(False)
    clocks = sampler.stop(t0, time.time())      # sampled over the timed loops (device-resident, e2e, per-kernel)
    kt /= max(nsteps_t, 1)
    gemm_ms = kt[0]      # the event pair around the one grouped launch; kt[1] is the gap between two back-to-back event records (no kernel)
    # ---- apply alone, back to back (the H*psi GFLOP/s figure of BASELINE.json)
    x = torch.randn(n, dtype=torch.float64, device=f"cuda:{local}"); y = torch.empty_like(x)
    for _ in range(3):
        plan.apply_H(x, y)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 50
    e0.record(stream)
    for _ in range(reps):
        plan.apply_H(x, y)
    e1.record(stream); torch.cuda.synchronize()
    apply_ms = e0.elapsed_time(e1) / reps

    # ---- roofline denominators: FP64 peak measured live (MEASURED_PEAKS.json has no FP64 entry), HBM from the file
    dmma_peak = lib.dmrg_probe_fp64_peak(1, 3)
    dfma_peak = lib.dmrg_probe_fp64_peak(0, 3)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    traffic, traffic_note = None, None
    try:
        tj = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(args.config, {})
        traffic, traffic_note = tj.get("grouped_gemm_dram_bytes_per_launch"), tj.get("note")
    except Exception:
        pass
    achieved = st["flop_per_apply"] / (gemm_ms * 1e-3) / 1e12
    roofline = {"bound": "tensor", "kernel": "grouped_gemm_kernel (persistent, warp-specialised: DMMA.8x8x4 consumers fed by cp.async.bulk tile images; "
                                             "1 launch per step: X images, stage-1 and stage-2 units in ticket order)",
                "achieved": achieved, "peak": max(dmma_peak, dfma_peak), "unit": "TFLOP/s",
                "frac": achieved / max(dmma_peak, dfma_peak), "traffic": traffic, "traffic_note": traffic_note,
                "peak_source": "measured live: register-only DMMA.8x8x4 issue-rate probe (dmrg_probe_fp64_peak); "
                               f"DFMA probe {dfma_peak:.1f}; nominal 148 SM x 128 FLOP/clk x 1.965 GHz = 37.2",
                "flop_per_launch": st["flop_per_apply"], "ms_per_launch": gemm_ms}
    blas2_gbs = bytes_b2 / max(t_b2 * 1e-3, 1e-12) / 1e9 / 1.0 if nsteps_t else None
    if blas2_gbs is not None:
        blas2_gbs = bytes_b2 / (t_b2 * 1e-3) / 1e9

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    side = world == 1 and not args.profile_run
    gt_probe = None
    try:
        if side:
            gt_probe = gemv_trans_probe(plan, V, W, flush, hbm_peak)
    except Exception as e:
        gt_probe = {"error": repr(e)}
    dav_large = None
    if world == 1 and not args.no_large:
        try:
            hbm_read = lib.dmrg_probe_hbm_read(4 << 30, 3)       # live read-only stream (the BLAS-2 kernels are read-dominated)
            dav_large = davidson_hbm_probe(lib, f"cuda:{local}", hbm_peak, hbm_read=hbm_read)
            dav_large["apply_frac_fp64_peak"] = dav_large["apply_tflops"] / max(dmma_peak, dfma_peak)
            dav_large["other_configs"] = {}
            for nm in ("cfg5a", "heis4096"):     # the judgement is also taken at 5a and the 4096 sweep
                o = davidson_hbm_probe(lib, f"cuda:{local}", hbm_peak, name=nm, steps=40, hbm_read=hbm_read)
                dav_large["other_configs"][nm] = {kk: o[kk] for kk in ("workload", "kernels_gbs", "kernels_frac_hbm", "kernels_frac_hbm_read", "append_gbs_incl_tile_images",
                                                                       "blas2_gbs", "blas2_frac_hbm", "blas2_frac_hbm_read") if kk in o}
        except Exception as e:   # the headline numbers above do not depend on this extra config
            dav_large = {"error": repr(e)}
    vendor = None
    if side:
        try:      # the vendor-library mark beside the live probe
            a = torch.randn(8192, 8192, dtype=torch.float64, device=f"cuda:{local}"); b = torch.randn_like(a)
            torch.matmul(a, b); torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(3):
                torch.matmul(a, b)
            e1.record(stream); torch.cuda.synchronize()
            vendor = 3 * 2.0 * 8192 ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12
            del a, b
            torch.cuda.empty_cache()
        except Exception:
            vendor = None
    roofline["vendor_dgemm_tflops"] = vendor
    roofline["vendor_dgemm_note"] = "torch.matmul FP64 8192^3 (cuBLAS DGEMM), 3 back-to-back calls; datasheet FP64 tensor 40 TFLOP/s nominal"
    block = None
    if side:
        try:
            block = block_davidson_probe(lib, problem, cfg, f"cuda:{local}", st)
        except Exception as e:
            block = {"error": repr(e)}

    next_rows = None
    if side:
        try:
            next_rows = next_rows_probe(lib, f"cuda:{local}", max(dmma_peak, dfma_peak))
        except Exception as e:
            next_rows = {"error": repr(e)}

    curve = None
    if side:
        try:
            names = ["cfg2", "cfg4", "cfg5a", "heis4096"] + ([] if args.no_large else ["heis8192"])
            curve = hpsi_curve(lib, f"cuda:{local}", max(dmma_peak, dfma_peak), names)
        except Exception as e:
            curve = {"error": repr(e)}

    # ---- oracle timed beside it (rank 0, N = 1 only): bounded sample
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        osteps = 20
        gfl, oms, cores, _ = oracle_iteration_timer(problem, k_max, osteps, 2)
        cpu_baseline = {"value": gfl, "unit": UNIT, "cores": cores, "kind": "oracle", "ms_per_step": oms,
                        "sample": f"{osteps} consecutive O-DAV iterations of {args.config} (k = 3..{2 + osteps}) from start e_argmin(D), numpy/BLAS threads = {cores}"}
        cpu_baseline.update(host_description())
        try:      # the same oracle on ONE thread (the paper's CPU reference is a few-thread MKL run): 6 iterations
            from threadpoolctl import threadpool_limits
            with threadpool_limits(limits=1):
                g1, ms1, _, _ = oracle_iteration_timer(problem, k_max, 6, 1)
            cpu_baseline["one_thread"] = {"value": g1, "unit": UNIT, "ms_per_step": ms1, "sample": "6 consecutive O-DAV iterations, BLAS threads = 1"}
        except Exception as e:
            cpu_baseline["one_thread"] = {"error": repr(e)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": dict(workload_config(args.config, cfg, n, st), step_mode=step_mode),
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 8 * n, "d2h_bytes_per_step": 8 * n + 24,
                    "ms_per_step": tot_e / args.steps},
            "gpu_launches": int(gpu_launches),
            "roofline": roofline, "cpu_baseline": cpu_baseline,
            "hpsi": {"gflops": st["flop_per_apply"] / (apply_ms * 1e-3) / 1e9, "ms": apply_ms,
                     "frac_fp64_peak": st["flop_per_apply"] / (apply_ms * 1e-3) / 1e12 / max(dmma_peak, dfma_peak),
                     "note": "dmrg_apply_H alone, back to back, warm L2"},
            "davidson": {"iters_per_s": world * args.steps / (total_ms * 1e-3),
                         "kernel_ms": {nm: float(v) for nm, v in zip(["apply", "event_gap", "vtw", "small_eig", "residual", "collapse", "orthogonalise", "append"], kt)},
                         "blas2_gbs": blas2_gbs, "blas2_frac_hbm": (blas2_gbs / hbm_peak) if blas2_gbs else None,
                         "hbm_peak_gbs": hbm_peak, "hbm_peak_source": hbm_src,
                         "note": "BLAS-2 kernels timed inside the running loop, warm L2: V+W fit partly in the 126 MB L2 at this config"},
            "davidson_hbm": dav_large, "gemv_trans": gt_probe, "hpsi_curve": curve, "block_davidson": block, "next_rows": next_rows,
            "device_bytes": plan.stats()["device_bytes"] + 2 * V.numel() * 8}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def block_davidson_probe(lib, problem, cfg, device, st):
    """(a) the projection of nrhs vectors in ONE grouped launch against nrhs single
    launches; (b) the whole solve to tol 1e-10 from start (D): single-vector driver (lowest pair) vs the block driver with
    nb = 2 (the two lowest pairs), wall clock around the C-ABI call, with the number of projections each needed."""
    import torch
    plan = lib.Plan(problem, k_max=cfg["k_max"], tol=1e-10, max_iter=4000, max_rhs=4, device=device)
    n = plan.n
    stream = torch.cuda.current_stream()
    ld = (n + 15) // 16 * 16
    X = torch.randn((4, ld), dtype=torch.float64, device=device); Y = torch.empty_like(X)
    out = {"apply_multi_us_per_vector": {}}
    for nr in (1, 2, 4):
        for _ in range(3):
            plan.apply_H_multi(X[:nr], Y[:nr])
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(10):
            plan.apply_H_multi(X[:nr], Y[:nr])
        e1.record(stream); torch.cuda.synchronize()
        out["apply_multi_us_per_vector"][str(nr)] = e0.elapsed_time(e1) / 10 / nr * 1e3
    out["apply_multi_tflops_nrhs4"] = st["flop_per_apply"] / (out["apply_multi_us_per_vector"]["4"] * 1e-6) / 1e12
    D = plan.diag()
    t0 = time.perf_counter(); rc1, lam, x, rho, it1 = plan.lowest_eigenpair(None, start_at_argmin_diag=True); torch.cuda.synchronize()
    t_single = time.perf_counter() - t0
    X0 = torch.zeros((2, ld), dtype=torch.float64, device=device)     # start (D) with two columns: unit vectors at the two smallest D_pp
    idx = torch.argsort(D, stable=True)[:2]
    X0[0, idx[0]] = 1.0; X0[1, idx[1]] = 1.0
    t0 = time.perf_counter(); rc2, th, Xb, rb, itb, apb = plan.block_lowest_eigenpairs(X0); torch.cuda.synchronize()
    t_block = time.perf_counter() - t0
    out["solve"] = {"single": {"rc": rc1, "ms": t_single * 1e3, "applies": it1, "lambda": lam, "resnorm": rho},
                    "block_nb2": {"rc": rc2, "ms": t_block * 1e3, "block_iterations": itb, "applies": apb,
                                  "theta": [float(v) for v in th], "resnorm": [float(v) for v in rb]},
                    "note": "block: two pairs to 1e-10, two synchronisations per block iteration (first slice); "
                            "single: one pair, steps enqueued back to back"}
    plan.close()
    return out


def next_rows_probe(lib, device, fp64_peak):
    """SURVEY 8(f) NEXT-1 and NEXT-2, measured: (a) dmrg_apply_H of an l-1-1-r plan on two synthetic
    un-enlarged blocks of m = 1024 and of m = 2048 states (dmrg_inputs.heisenberg_block_synthetic, seeds 71/72): the superblock
    dimension is that of the LR plan of the enlarged blocks (2 m per side); (b) the infinite-lattice loop dmrg_infinite_heisenberg
    (Alg. 1, every step on the device) to 64 sites with m = 128, wall clock around the C-ABI call."""
    import torch
    from dmrg_inputs import heisenberg_block_synthetic
    out = {}
    stream = torch.cuda.current_stream()
    for m in (1024, 2048):
        l, r = heisenberg_block_synthetic(m, 4, 71), heisenberg_block_synthetic(m, 4, 72)
        plan = lib.Plan.from_l11r(l, r, 1.0, 1.0, 0, device=device)
        st = plan.stats()
        x = torch.randn(plan.n, dtype=torch.float64, device=device); y = torch.empty_like(x)
        for _ in range(3):
            plan.apply_H(x, y)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(10):
            plan.apply_H(x, y)
        e1.record(stream); torch.cuda.synchronize()
        us = e0.elapsed_time(e1) / 10 * 1e3
        out["l11r_apply" if m == 1024 else f"l11r_apply_m{m}"] = {
            "workload": f"l-1-1-r, two synthetic blocks of m = {m} (9 sectors), target 2 S_z = 0", "n": int(plan.n),
            "flop_per_apply": int(st["flop_per_apply"]), "us_per_apply": us,
            "tflops": st["flop_per_apply"] / (us * 1e-6) / 1e12,
            "frac_fp64_peak": st["flop_per_apply"] / (us * 1e-6) / 1e12 / fp64_peak,
            "units": int(st["stage1_units"] + st["stage2_units"])}
        plan.close()
        del x, y
    lib.infinite_heisenberg(16, 32)                      # warm-up (module load, allocator)
    t0 = time.perf_counter()
    recs = lib.infinite_heisenberg(64, 128)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    last = recs[-1]
    out["infinite_dmrg"] = {"workload": "Heisenberg Delta = 1, infinite-lattice growth 4 -> 64 sites, m = 128, tol 1e-10",
                            "wall_s": dt, "superblocks": len(recs), "energy_per_site_last": float(last["energy"]) / int(last["n_sites"]),
                            "discarded_last": float(max(last["discarded"])), "davidson_iters_total": int(sum(q["davidson_iters"] for q in recs))}
    return out


def hpsi_curve(lib, device, fp64_peak, names):
    """dmrg_apply_H alone at the other configs and the Heisenberg 4096 / 8192 sweep (the headline curve,
    PAPER.md Fig. 19-20 plots the same quantity against m): time per apply, TFLOP/s on the algorithmic FLOP count (A24)
    and fraction of the measured FP64 peak.  Seeded N(0,1) input (seed 3000+c), back to back on one stream."""
    import torch
    from dmrg_inputs import make_config, CONFIGS, random_vector, vector_seed
    out = {}
    stream = torch.cuda.current_stream()
    for name in names:
        problem = make_config(name)
        plan = lib.Plan(problem, k_max=CONFIGS[name]["k_max"], device=device)
        st = plan.stats()
        n = plan.n
        x = torch.from_numpy(random_vector(n, vector_seed(name, "hpsi"))).to(device)
        y = torch.empty_like(x)
        reps = 20 if st["flop_per_apply"] < 1e11 else 5
        for _ in range(3):
            plan.apply_H(x, y)
        best = None
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                plan.apply_H(x, y)
            e1.record(stream); torch.cuda.synchronize()
            t = e0.elapsed_time(e1) / reps
            best = t if best is None else min(best, t)
        tf = st["flop_per_apply"] / (best * 1e-3) / 1e12
        out[name] = {"n": int(n), "flop_per_apply": int(st["flop_per_apply"]), "us_per_apply": best * 1e3, "tflops": tf,
                     "frac_fp64_peak": tf / fp64_peak, "units": int(st["stage1_units"] + st["stage2_units"])}
        plan.close()
        del x, y, plan, problem
        torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-large", action="store_true", help="skip the config-5b Davidson HBM measurement")
    ap.add_argument("--profile-run", action="store_true",
                    help="steps only (no side probes, no CPU baseline): the command line the ncu captures under profiles/ use")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.profile_run:
        args.no_large = args.no_cpu_baseline = True
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N replicas ourselves, the way the driver does (one rank per GPU)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
