#!/usr/bin/env python
"""bench.py -- the headline measurement of the sigma = H psi hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg5] [--impl reference]

A step is one Davidson iteration: one H psi (dmrg_sigma: stage-1 and stage-2 grouped GEMMs) plus the
device-side Davidson vector work of that iteration (subspace dots, Ritz vector, residual,
preconditioner, orthogonalisation); the per-bond H diagonal is computed once at the start of the timed
region.  value = EXECUTED FP64 TFLOP/s over the whole timed region: the flops of the GEMMs the plan runs (the
paper's cost measure 2MNK per GEMM, after the planner's de-duplication of X = psi R^T products;
unpadded), ms_per_step = ms per H psi.  The canonical count (one GEMM pair per term and symmetry-block
combination, no de-duplication) and the rate on it are printed beside it (`canonical_flops_per_hpsi`,
`canonical_tflops`) so that a smarter plan cannot inflate the rate.
Inputs are seeded synthetic (dmrg_workload), resident in HBM before the timed region starts.
With N > 1 (torchrun) every rank runs an independent replica of the same bond ("replicas only":
BASELINE.json fixes the path to one GPU with no sharding and no collectives).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64_tflops_per_hpsi"
# dram__bytes_read.sum + dram__bytes_write.sum of all GEMM launches of one H psi, from a committed ncu launch list
# (NOT measured by this run): config -> (bytes, source)
NCU_DRAM_BYTES_PER_HPSI = {"cfg5": (2.006e12, "profiles/r2_cfg5_launches.csv (round 2, final kernel; 42 GEMM launches of the second dmrg_sigma call)"),
                           "cfg4": (2.294e11, "profiles/r2_cfg4_split_small_launches.csv (round 2, final kernel; 12 GEMM launches of the second dmrg_sigma call)"),
                           "cfg3": (1.641e11, "profiles/r2_cfg3_launches.csv (round 2, final kernel; 4 GEMM launches of the second dmrg_sigma call)"),
                           "cfg2": (9.88e9, "profiles/r2_cfg2_launches.csv (round 2, final kernel; 2 GEMM launches of the second dmrg_sigma call)")}
UNIT = "TFLOP/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg5", help="cfg1..cfg5 of BASELINE.json (default: the headline K=73 D=3000); so2 / so3: the spin-orbit "
                                                     "variants (complex FP64, N only; SURVEY section 8(f) NEXT-4) of cfg2 / cfg3, --sigma-only only")
    ap.add_argument("--bond-dim", type=int, default=0, metavar="D",
                    help="override the bond dimension of a direct-fill config (cfg3-5; footprint experiments, e.g. the largest D that "
                         "fits one GPU: DESIGN.md section 5); the workload name says so")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workspace-gib", type=float, default=0.0, help="X workspace (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="dmrg_plan_options field (copy_mode, split_waves, min_split_stages, max_merged_cols, "
                         "cost_order_only, split_small, release_r_store, tile_run_stages); repeatable")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "shard"],
                    help="N > 1: replicas (default; BASELINE.json fixes the path to one GPU: N independent copies, weak scaling) or "
                         "shard (operator parallelism, PAPER.md:81,162: the terms are partitioned over the ranks and every H psi ends "
                         "with one NCCL all-reduce of sigma inside dmrg_sigma; strong scaling)")
    ap.add_argument("--sigma-only", type=int, default=0, metavar="N",
                    help="profiling mode: no Davidson, no oracle; N plain dmrg_sigma calls (after one warm-up call) and a short "
                         "JSON line with the per-stage device times -- the command the ncu captures under profiles/ wrap")
    ap.add_argument("--operators", default="default", choices=["default", "renorm"],
                    help="default: the config's generator (CPU blocking for cfg1-2, direct fill for cfg3-5); renorm: both blocks "
                         "grown ON THE DEVICE by chained dmrg_renormalize calls with seeded random site tensors (physical operators; "
                         "the oracle legs are skipped: oracle inputs must not come from the CUDA path)")
    ap.add_argument("--davidson-to", type=float, default=0.0, metavar="TOL",
                    help="after the timed steps, run the Davidson from the reading-12 guess (unit vector at argmin Hd + 1e-3 noise) "
                         "to this residual and report iterations and wall time (BASELINE.json configs[2])")
    return ap.parse_args()


def plan_options(args):
    out = {}
    for kv in args.opt:
        k, v = kv.split("=", 1)
        out[k] = float(v) if k == "split_waves" else int(v)
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except Exception:
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7), ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def pick_sample_blocks(pr, layout, budget_flops):
    """Output blocks for the bounded oracle sample: cheapest-first would be unrepresentative, so take
    blocks in a fixed pseudo-random order until their summed contraction cost reaches the budget.
    The cost of an output block is estimated from its share of psi (uniform terms) -- a sizing heuristic only."""
    rng = np.random.Generator(np.random.Philox(1234))
    order = rng.permutation(len(layout))
    sizes = layout[:, 4] * layout[:, 5]
    return order, sizes


def oracle_sample(pr, psi, total_flops, seconds):
    """The oracle (all terms) on a bounded sample of sigma blocks, for the parity check of the timed configuration:
    the LARGEST sigma block (the 436 x 436 class at cfg 5: 7 x 7 tiles, the most split-K parts) whenever the oracle can
    do it in about half a minute, plus seeded random blocks up to the budget."""
    import oracle
    ncores = oracle.num_threads()
    layout = np.asarray(pr.layout)
    order, sizes = pick_sample_blocks(pr, layout, 0)
    share = sizes / sizes.sum()
    target_rate = 1.5e9 * ncores   # first guess, FLOP/s
    budget = target_rate * seconds
    chosen, acc = [], 0.0
    big = int(np.argmax(sizes))
    if share[big] * total_flops <= 30.0 * 3.5e9 * ncores:
        chosen.append(big)
    for b in order:
        if len(chosen) >= 5 and acc >= budget:
            break
        if int(b) in chosen or (chosen and acc + share[b] * total_flops > 4 * budget):
            continue   # keep a second outsized block out of a small sample
        chosen.append(int(b))
        acc += share[b] * total_flops
    t0 = time.perf_counter()
    sig, st = oracle.opair_sigma(pr, psi, only_out=chosen, return_stats=True)
    dt = time.perf_counter() - t0
    dims = [(int(layout[b][4]), int(layout[b][5])) for b in chosen]
    return {"value": st["flops"] / dt * 1e-12, "unit": UNIT, "cores": ncores, "kind": "oracle",
            "sample": f"{len(chosen)} of {len(layout)} sigma blocks ({st['flops']:.3e} of {total_flops:.3e} FLOP, "
                      f"{int(st['tasks'])} tasks) in {dt:.1f} s incl. term expansion and intermediates",
            "seconds": dt, "flops": st["flops"], "blocks": chosen, "block_dims": dims, "sigma": sig}


def oracle_term_sample(pr, psi, total_flops, seconds, k=0):
    """Time the oracle (as it stands) on a bounded sample of the workload: every stride-th operator-pair term on
    all sigma blocks (no fixed term-expansion / intermediates overhead beyond what the sampled terms need)."""
    import oracle
    from dmrg_workload.problem import term_subset_problem
    nterms = len(pr.term_coef)
    rate_guess = 3.5e9 * oracle.num_threads()               # FLOP/s, sizing only (measured ~3.8e9 per core)
    stride = int(max(1, min(nterms, round(total_flops / max(rate_guess * seconds, 1.0)))))
    ids = np.arange(k % stride, nterms, stride)
    sub = term_subset_problem(pr, ids)
    t0 = time.perf_counter()
    _, st = oracle.opair_sigma(sub, psi, return_stats=True)
    dt = time.perf_counter() - t0
    return {"value": st["flops"] / dt * 1e-12, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"every {stride}-th of {nterms} terms on all {len(pr.layout)} sigma blocks ({st['flops']:.3e} of "
                      f"{total_flops:.3e} FLOP, {int(st['tasks'])} tasks) in {dt:.1f} s",
            "seconds": dt, "flops": st["flops"], "tasks": int(st["tasks"])}


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0")))


def run_reference(args):
    """--impl reference: for this tier the reference arm is the CPU oracle, timed as it stands.  It stands on
    oracle/ and dmrg_workload/ alone: the product package is never imported here."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    from dmrg_workload.problem import make_config, random_psi
    import oracle
    pr = make_config(args.config)
    psi = random_psi(pr.psi_size, 5)
    total = oracle.opair_count(pr)["flops"]   # the oracle's own cost counter (pinned: tests/test_oracle_flopcount.py)
    assert "paper_2311_02854_b200" not in sys.modules
    # Each step = the oracle, as it stands, on a bounded SAMPLE of the workload: every stride-th operator-pair term
    # (all sigma blocks), sized so that the whole run takes a few minutes.  (Sampling sigma blocks instead would
    # make every step pay the oracle's full term expansion and its 8 GB of intermediates, ~80 s at cfg 5.)
    per_step = max(2.0, min(30.0, 150.0 / max(1, args.steps + args.warmup)))
    for k in range(args.warmup):
        oracle_term_sample(pr, psi, total, per_step, k)
    t0 = time.perf_counter()
    fl, ntask, last = 0.0, 0, None
    for k in range(args.steps):
        last = oracle_term_sample(pr, psi, total, per_step, args.warmup + k)
        fl += last["flops"]; ntask += last["tasks"]
    res = {"unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": "per step: " + last["sample"]}
    dt = time.perf_counter() - t0
    val = fl / dt * 1e-12
    res["value"] = val
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / max(1, args.steps) * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, pr), "note": "each step = the CPU oracle on a bounded sample of the operator-pair terms"},
            "cpu_baseline": res, "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_name(cfg, pr):
    m = pr.meta
    return (f"{cfg}: K={m['K']} N={pr.N_tot} 2Sz={pr.twoSz_tot} D={m['D']} two-dot {m['nL']}-1-1-{m['nR']} "
            f"({m['mode']} operators{', banded integrals' if m.get('banded') else ''}), one H psi per Davidson iteration")


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import paper_2311_02854_b200 as g
    from dmrg_workload.problem import make_config, random_psi

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path)")
    torch.cuda.set_device(local)
    from paper_2311_02854_b200 import replicas
    replicas.init("nccl", torch.device("cuda", local))
    stream = torch.cuda.current_stream()

    t0 = time.perf_counter()
    renorm_info = None
    if args.operators == "renorm":
        from dmrg_workload.integrals import make_integrals
        from dmrg_workload.problem import CONFIGS
        from paper_2311_02854_b200 import bondgen
        c = CONFIGS[args.config]
        ints = make_integrals(c["K"], c["seed"], banded=c.get("banded", False))
        pr = bondgen.build_bond(g, c["K"], c["nL"], c["N_tot"], 0, c["D"], ints, c["seed"], stream=stream,
                                log=(lambda m: print(m, file=sys.stderr)) if rank == 0 else None)
        pr.meta["banded"] = c.get("banded", False)
        ops = pr.ops
        t_gen, t_load = pr.seconds["total"], 0.0
        rs = pr.renorm_stats
        big = [r for r in rs if r["dim"] >= 0.9 * max(x["dim"] for x in rs)]
        renorm_info = {"steps": len(rs), "flops": sum(r["flops"] for r in rs), "device_ms": sum(r["device_ms"] for r in rs),
                       "tflops_full_size_steps": sum(r["flops"] for r in big) / max(1e-9, sum(r["device_ms"] for r in big)) * 1e-9,
                       "seconds_total": pr.seconds["total"], "seconds_chains": pr.seconds["chains"]}
    else:
        pr = make_config(args.config, D=args.bond_dim) if args.bond_dim > 0 else make_config(args.config)
        t_gen = time.perf_counter() - t0
        t0 = time.perf_counter()
        ops = g.OpsStore(pr.secL, pr.secR, pr.ops, pr.blocks, pr.values, pr.lin_ptr, pr.lin_op, pr.lin_coef)
        t_load = time.perf_counter() - t0
    free1, _ = torch.cuda.mem_get_info()
    ws = int(args.workspace_gib * 2 ** 30) if args.workspace_gib > 0 else int(min(24 * 2 ** 30, 0.25 * free1))
    t0 = time.perf_counter()
    popts = plan_options(args)
    sharded = args.parallelism == "shard" and world > 1
    comm = None
    if sharded:
        popts.update(shard_rank=rank, shard_count=world)
    plan = g.Plan(ops, pr.term_coef, pr.term_idx, pr.site_ops, pr.site_parity, pr.N_tot, pr.twoSz_tot, ws, **popts)
    if sharded:
        comm = g.Comm.from_torch_distributed(torch.device("cuda", local))
        plan.set_comm(comm)
    t_plan = time.perf_counter() - t0
    st = plan.stats()
    n = plan.psi_size
    is_z = np.dtype(getattr(pr, "dtype", np.float64)).kind == "c"
    if is_z:
        from dmrg_workload.problem import random_psi_z
        if args.sigma_only <= 0:
            raise SystemExit("bench.py: the spin-orbit configs are measured with --sigma-only N (the headline metric is BASELINE.json's real cfg5)")
        psi_h = random_psi_z(n // 2, 5)   # psi_size counts doubles
    else:
        psi_h = random_psi(n, 5)
    x = torch.from_numpy(psi_h).cuda()
    sig = torch.empty_like(x)

    if args.sigma_only > 0:
        plan.sigma(x, sig, stream)
        torch.cuda.synchronize()
        plan.set_timing(True)
        rows = []
        for _ in range(args.sigma_only):
            plan.sigma(x, sig, stream)
            rows.append(plan.stage_ms())
        med = [float(np.median([r[i] for r in rows])) for i in range(3)]
        fl = st["s1_flops"] + st["s2_flops"]
        zpar = None
        if is_z and not args.no_cpu_baseline:
            # parity of this launch configuration against the complex oracle on sampled sigma blocks (largest one first)
            from oracle import zsigma
            lay = np.asarray(pr.layout)
            sizes = lay[:, 4] * lay[:, 5]
            blocks = [int(np.argmax(sizes)), int(np.argmin(sizes))] + [int(b) for b in np.random.Generator(np.random.Philox(1234)).permutation(len(lay))[:3]]
            t0 = time.perf_counter()
            ref = zsigma.zopair_sigma(pr, psi_h, only_out=blocks)
            got = sig.cpu().numpy()
            err = max(float(np.abs(got[int(lay[b][6]):int(lay[b][6] + sizes[b])] - ref[int(lay[b][6]):int(lay[b][6] + sizes[b])]).max()) for b in blocks)
            zpar = {"max_abs_err_over_norm": err / float(np.linalg.norm(got)), "blocks_checked": len(blocks), "largest_block": [int(lay[blocks[0]][4]), int(lay[blocks[0]][5])],
                    "tolerance": 1e-11, "oracle": "oracle/zsigma.py", "oracle_seconds": time.perf_counter() - t0}
        print(json.dumps({"mode": "sigma-only", "dtype": "c128 (as real FP64 GEMMs, 8 MNK flops per complex GEMM)" if is_z else "f64", "parity_sampled": zpar, "config": workload_name(args.config, pr), "calls": args.sigma_only, "plan_options": popts,
                          "stage1_ms": med[0], "stage2_ms": med[1], "hpsi_ms": med[2], "executed_tflops": fl / med[2] * 1e-9,
                          "s1_tflops": st["s1_flops"] / med[0] * 1e-9, "s2_tflops": st["s2_flops"] / med[1] * 1e-9,
                          "launches_per_hpsi": int(st["launches"]), "chunks": int(st["chunks"]),
                          "stats": {k: st[k] for k in ("s1_flops", "s2_flops", "padded_flops", "stage_flops", "warp_flops", "canon_flops", "s1_tiles", "s2_tiles",
                                                       "s1_fill", "s2_fill", "s1_stages", "s2_stages")}}))
        plan.destroy()
        ops.free()
        return
    # FP64 pipe peak, measured live under the same conditions (roofline denominator)
    peak_dmma = g.fp64_peak_tflops(1, 300.0, stream)
    peak_dfma = g.fp64_peak_tflops(0, 300.0, stream)

    def barrier():
        replicas.barrier(torch.cuda.synchronize)

    # ---- warm-up: W Davidson iterations (allocates the Davidson workspace) ---------------------
    W, K = max(args.warmup, 3), args.steps
    plan.davidson(x.clone(), max_iter=W, max_space=max(W, K), tol=0.0, stream=stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    xk = x.clone()
    try:
        uuid = str(torch.cuda.get_device_properties(local).uuid)
        gpu_id = uuid if uuid.startswith("GPU-") else "GPU-" + uuid
    except Exception:
        gpu_id = str(local)
    clocks = ClockSampler(gpu_id)
    clocks.start()
    barrier()
    e0.record(stream)
    res = plan.davidson(xk, max_iter=K, max_space=K, tol=0.0, stream=stream)   # EXACTLY K steps (tol 0 never stops early)
    e1.record(stream)
    barrier()
    clk = clocks.stop()
    ms_total = e0.elapsed_time(e1)
    assert res["iters"] == K
    flops_canon = st["canon_flops"]
    flops = st["s1_flops"] + st["s2_flops"]       # executed: what the GEMM launches of one H psi compute (unpadded)
    if sharded:
        # one bond shared by all ranks: the job's work is the SUM of the shards' executed flops, its time the slowest rank's
        import torch.distributed as dist
        tot = torch.tensor([flops, flops_canon], dtype=torch.float64, device="cuda")
        dist.all_reduce(tot)
        job_flops, job_canon = float(tot[0]), float(tot[1])
        ms_step = replicas.max_over_ranks(ms_total / K, "cuda")
        value = job_flops / (ms_step * 1e-3) * 1e-12
    else:
        thr, ms_step = replicas.job_throughput(flops, ms_total / K, world, "cuda")   # max over ranks
        value = thr * 1e-12

    # ---- kernel-only H psi (no Davidson vector work) and the roofline of the GEMM kernel --------
    ts = []
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); plan.sigma(x, sig, stream); b.record(stream); torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    ms_sigma = float(np.median(ts))
    # dmrg_sigma enqueues its launches back to back on the caller's stream (per chunk: stage 1, stage 2, split-K
    # reduce); "launch duration" of the roofline is the device time of the whole call, which is > 99 % GEMM launches
    # (profiles/).  A second call with the library's per-group events gives the per-stage split.
    plan.set_timing(True)
    plan.sigma(x, sig, stream)
    s1_ms, s2_ms, _ = plan.stage_ms()
    plan.set_timing(False)
    gemm_ms = ms_sigma
    achieved = flops / (gemm_ms * 1e-3) * 1e-12
    # DRAM bytes of all GEMM launches of one H psi, from the ncu pass committed as profiles/r1_cfg5_launches.csv
    # (dram__bytes_read.sum + dram__bytes_write.sum); only meaningful for the configuration that was profiled
    traffic, traffic_src = NCU_DRAM_BYTES_PER_HPSI.get(args.config, (None, None))
    roofline = {"bound": "tensor", "achieved": achieved, "peak": peak_dmma, "unit": "TFLOP/s", "frac": achieved / peak_dmma,
                "flops": "executed (s1_flops + s2_flops of the plan, unpadded)",
                "traffic": traffic, "traffic_unit": "bytes per H psi (ncu, all GEMM launches)",
                "traffic_source": f"NOT this run: {traffic_src}" if traffic else None,
                "kernel": "grouped_gemm_kernel (DMMA.8x8x4, all launches of one H psi)",
                "peak_source": "builder probe, measured live in this process: dmrg_fp64_peak_tflops(DMMA) (csrc/fp64_peak.cu); MEASURED_PEAKS.json "
                               "has no FP64 entry; nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                "canonical_tflops": flops_canon / (gemm_ms * 1e-3) * 1e-12, "canonical_frac": flops_canon / (gemm_ms * 1e-3) * 1e-12 / peak_dmma,
                "peak_dfma_measured": peak_dfma, "stage1_ms_serialised": s1_ms, "stage2_ms_serialised": s2_ms, "hpsi_ms": ms_sigma, "launches_per_hpsi": int(st["launches"]),
                "executed_flops_per_hpsi": flops, "padded_flops_per_hpsi": st["padded_flops"],
                "canonical_flops_per_hpsi": flops_canon, "algorithmic_bytes_per_hpsi": st["alg_bytes"],
                "hbm_gbs_if_streamed": st["alg_bytes"] / (gemm_ms * 1e-3) * 1e-9}

    # ---- end to end through the C ABI with host buffers ---------------------------------------------
    e2e = None
    if not args.no_e2e:
        pin_in = torch.from_numpy(psi_h).pin_memory()          # pinned host buffers, as the contract asks
        pin_out = torch.empty_like(pin_in).pin_memory()
        psi_pin, out_h = pin_in.numpy(), pin_out.numpy()
        plan.sigma_host(psi_pin, out_h, stream)
        barrier()
        t0 = time.perf_counter()
        ne = max(2, min(K, 4))
        for _ in range(ne):
            plan.sigma_host(psi_pin, out_h, stream)
        barrier()
        dt = (time.perf_counter() - t0) / ne
        e2e = {"value": world * flops / dt * 1e-12, "unit": UNIT, "h2d_bytes_per_step": int(8 * n), "d2h_bytes_per_step": int(8 * n),
               "ms_per_step": dt * 1e3, "call": "dmrg_sigma_host (H2D psi from pinned host memory, H psi, D2H sigma)"}

    # ---- CPU oracle beside it (rank 0, N = 1 only) ---------------------------------------------------
    cpu = None
    parity = None
    dav_to = None
    if args.davidson_to > 0:
        hd = torch.empty_like(x)
        plan.hdiag(hd, stream)
        torch.cuda.synchronize()
        guess = torch.from_numpy(1e-3 * random_psi(n, 7)).cuda()
        guess[int(torch.argmin(hd))] += 1.0
        t0 = time.perf_counter()
        r2 = plan.davidson(guess, max_iter=300, max_space=30, tol=args.davidson_to, stream=stream)
        torch.cuda.synchronize()
        dav_to = {"tol": args.davidson_to, "iters": r2["iters"], "converged": r2["converged"], "seconds": time.perf_counter() - t0,
                  "energy": r2["energy"], "resid": r2["resid"], "guess": "unit vector at argmin Hd + 1e-3 seeded noise (DESIGN.md reading 12)",
                  "max_space": 30}
    if rank == 0 and world == 1 and not args.no_cpu_baseline and args.operators != "renorm":
        cpu = oracle_term_sample(pr, psi_h, flops_canon, args.cpu_seconds)
        # parity on sampled sigma blocks (all terms), in the launch configuration that was timed; the oracle's
        # fixed cost (full term expansion, all intermediates) dominates this call, so it is not the cpu_baseline
        chk = oracle_sample(pr, psi_h, flops_canon, 1.0)
        blocks, refs = chk["blocks"], chk["sigma"]
        got = sig.cpu().numpy()
        nrm = float(np.linalg.norm(got))
        lay = np.asarray(pr.layout)
        err = 0.0
        for b in blocks:
            o, cnt = int(lay[b][6]), int(lay[b][4] * lay[b][5])
            err = max(err, float(np.abs(got[o:o + cnt] - refs[o:o + cnt]).max()))
        parity = {"max_abs_err_over_norm": err / nrm, "blocks_checked": len(blocks), "largest_block": max(chk["block_dims"], key=lambda d: d[0] * d[1]),
                  "tolerance": 1e-11, "oracle_seconds": chk["seconds"]}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic", "config": {"workload": workload_name(args.config, pr), "l2": "inputs larger than L2 (operator store + X workspace stream through every step)",
                                                "parallelism": ("operator-parallel shards + one NCCL all-reduce of sigma per H psi" if sharded else "replicas only") if world > 1 else "single GPU",
                                                "psi_size": int(n), "psi_blocks": int(len(pr.layout)), "terms": int(len(pr.term_coef)),
                                                "tasks": int(st["tasks"]), "chunks": int(st["chunks"])},
                "clocks": clk, "e2e": e2e, "gpu_launches": int(K * (st["launches"] + 15) + 4),   # GEMM / reduce launches + 15 Davidson vector kernels per step, + hdiag, start-up
                "roofline": roofline, "cpu_baseline": cpu,
                "ms_per_hpsi_kernel_only": ms_sigma, "frac_of_fp64_peak_whole_step": value / world / peak_dmma,
                "canonical_flops_per_hpsi": job_canon if sharded else flops_canon,
                "canonical_tflops": (job_canon if sharded else world * flops_canon) / (ms_step * 1e-3) * 1e-12,
                "plan_options": popts,
                "parity_sampled": parity,
                "footprint_gb": {"operator_store": ops.device_bytes / 1e9, "plan_and_workspace": st["plan_device_bytes"] / 1e9,
                                 "davidson_vectors": (2 * max(W, K) + 3) * 8 * n / 1e9},
                "setup_s": {"generate": t_gen, "ops_load": t_load, "plan": t_plan},
                "davidson": {"iters": res["iters"], "theta_last": res["energy"], "resid_last": res["resid"]},
                "davidson_to_tol": dav_to, "renormalization": renorm_info,
                "context": "paper: ~13-15 TFLOP/s FP64-TC per A100 for the GEMM step at large D (PAPER.md:231); D=14000 on 48 A100-80GB (PAPER.md:17)"}
        print(json.dumps(line))
    plan.destroy()
    if comm is not None:
        comm.destroy()
    ops.free()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
