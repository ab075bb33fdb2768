"""HBM footprint of one bond as a function of the bond dimension D, from structure-only planning (no GPU needed):

    python -m paper_2311_02854_b200.footprint [--K 73 --nL 35 --N 114] [--D 3000 4000 5000 ...] [--workspace-gib 24]

For every D: the sector tables of the d_max(D) model (dmrg_workload/sectors.py; Eq. 25), the operator store
dmrg_ops_load would hold, and the plan dmrg_plan_create would build (packed R copy, X workspace, padded psi, descriptors,
tensor maps), with and without release_r_store, plus the Davidson vectors of a 30-vector space.  The paper's memory
wall is D = 3000 on 4 x A100-40GB; this prints where it sits on one 180 GB B200.
"""
import argparse
import json
import time

import paper_2311_02854_b200 as g
from dmrg_workload.problem import make_direct_problem

HBM_BYTES = 183359 * 2 ** 20      # nvidia-smi total of a B200 (B200_PROFILING.md)
RESERVE = 2 * 2 ** 30             # CUDA context, allocator slack


def footprint(K, nL, N, D, ws_gib, max_space=30, banded=True):
    pr = make_direct_problem(K, nL, N, 0, D=D, seed=1, banded=banded, structure_only=True)
    ops, plan = g.load_problem(pr, workspace_bytes=int(ws_gib * 2 ** 30), structure_only=True)
    st = plan.stats()
    is_r = pr.ops[:, 0] == 1
    # bytes of the R-side allocation = padded stored R blocks + R lincombs: everything the store holds minus the L side
    secL, secR = pr.secL, pr.secR
    def side_bytes(side):
        sec = secL if side == 0 else secR
        tot = 0
        for op in pr.ops[pr.ops[:, 0] == side]:
            dn, ds = int(op[4]), int(op[5])
            idx = {(int(s[0]), int(s[1])): int(s[2]) for s in sec}
            for (n, sz), dcol in idx.items():
                drow = idx.get((n + dn, sz + ds))
                if drow is not None:
                    tot += 8 * drow * ((dcol + 1) & ~1)
        return tot
    r_bytes = side_bytes(1)
    out = {"D": D, "dmax": int(max(pr.secL[:, 2].max(), pr.secR[:, 2].max())), "psi_size": int(plan.psi_size), "tasks": int(st["tasks"]),
           "exec_tflop": (st["s1_flops"] + st["s2_flops"]) * 1e-12, "store_gb": ops.device_bytes / 1e9, "store_r_side_gb_upper": r_bytes / 1e9,
           "plan_gb": st["plan_device_bytes"] / 1e9, "x_workspace_gb": 8 * st["xws_elems"] / 1e9, "chunks": int(st["chunks"]),
           "davidson_gb": (2 * max_space + 3) * 8 * plan.psi_size / 1e9}
    out["total_gb"] = out["store_gb"] + out["plan_gb"] + out["davidson_gb"]
    # release_r_store: the steady state drops the R-side originals.  Where the originals and the plan's packed copy do not
    # fit side by side while the plan is created, dmrg_plan_create parks the R side in host memory first (needs that
    # much host RAM; measured: D = 4500 runs that way), so the steady state is what has to fit.
    out["total_release_r_gb"] = out["total_gb"] - min(out["store_r_side_gb_upper"], out["store_gb"])
    out["host_parking_gb"] = min(out["store_r_side_gb_upper"], out["store_gb"]) if out["store_gb"] + out["plan_gb"] > (HBM_BYTES - RESERVE) / 1e9 else 0.0
    plan.destroy()
    ops.free()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--K", type=int, default=73)
    ap.add_argument("--nL", type=int, default=35)
    ap.add_argument("--N", type=int, default=114)
    ap.add_argument("--D", type=int, nargs="+", default=[1000, 2000, 3000, 3500, 4000, 4500])
    ap.add_argument("--workspace-gib", type=float, default=12.0)
    a = ap.parse_args()
    cap = (HBM_BYTES - RESERVE) / 1e9
    best = {"keep": None, "release": None}
    for D in a.D:
        t0 = time.perf_counter()
        r = footprint(a.K, a.nL, a.N, D, a.workspace_gib)
        r["plan_seconds"] = time.perf_counter() - t0
        r["fits"] = r["total_gb"] <= cap
        r["fits_release_r"] = r["total_release_r_gb"] <= cap
        if r["fits"]:
            best["keep"] = D
        if r["fits_release_r"]:
            best["release"] = D
        print(json.dumps(r), flush=True)
    print(json.dumps({"capacity_gb": cap, "largest_D_fitting": best}))


if __name__ == "__main__":
    main()
