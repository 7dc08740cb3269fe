"""Roofline sweeps of ax_e, gs, ax and the CG iteration (BASELINE.json configs[3]).

    python -m paper_2606_12650_b200.sweep [--which e|n|both|big|paper|coop] [--reps 50] [--out sweep.csv]

4a (e): brick meshes with E = 2^10 .. 2^17 at N = 7;  4b (n): N = 3 .. 15 at E = 4096 (16^3); perturbed
geometry (amplitude 0.05), u uniform[-1,1) per LOCAL point (seed 1004), `reps` back-to-back
applications timed with CUDA events after 3 untimed ones, best and median of 5 repeats.
big: N = 7 .. 11 at E = 2^15 (32^3, working sets 1.2 - 4.1 GB, far beyond L2): the three operators plus
the CG iteration (20 iterations per call), for the ">= 70 % at N = 7-11" target of BASELINE.json.
Reported per point: us per application, model GB/s (ax_e 64 B/pt; gs 20 B per listed copy + 4 B per
row; ax = both; CG iteration: the canonical unfused 168 B/pt + gs), model GFLOP/s, fraction of the measured
copy peak (MEASURED_PEAKS.json, else the guide's fallback) and of the nominal 8 TB/s, and whether the working
set fits in L2 ("L2-resident": effective GB/s can then exceed the HBM peak; the >= 70 % claim is made
on the other points only).
paper: the paper's own sweep: N in {4, 6, 8}, E = 2^1 .. 2^14, CG 100 iterations, GDOFS.
coop: the CG iteration on small meshes, graph replay against the cooperative whole-solve launch.

This tool only times.  Parity of every point against the oracle is `python tests/sweep_parity.py`, which
calls the generators below and appends its columns (the product never imports the oracle).
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_BYTES = 126e6
BIG_SWEEP = [dict(brick=(32, 32, 32), N=N) for N in range(7, 12)]


def _peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


def _time(fn, reps, repeats=5):
    import torch
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    out = []
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        out.append(e0.elapsed_time(e1) / reps * 1e3)          # us per application
    return min(out), float(np.median(out))


def run_point(mesh, reps, with_cg=False):
    import torch
    from paper_2606_12650_b200 import Nekbone
    from workloads import sweep_field, rhs_unique
    from workloads.configs import SWEEP_SEED
    nk = Nekbone.from_mesh(mesh)
    u = torch.from_numpy(sweep_field(mesh)).cuda()
    w = nk.empty()
    v = u.clone()
    s = nk.gs_sizes()
    L, N = mesh.L, mesh.N
    b_ax_e = 64.0 * L
    b_gs = 20.0 * s["n_listed"] + 4.0 * s["n_rows"]
    fl = (12.0 * (N + 1) + 15.0) * L
    rows = []
    jobs = [("ax_e", lambda: nk.ax_e(u, w), b_ax_e, fl, reps),
            ("gs", lambda: nk.gs(v), b_gs, 0.0, reps),
            ("ax", lambda: nk.ax(u, w), b_ax_e + b_gs, fl, reps)]
    if with_cg:
        f = torch.from_numpy(rhs_unique(mesh, SWEEP_SEED)).cuda()
        x = nk.empty()
        hist = torch.empty(21, dtype=torch.float64, device="cuda")
        gs_adds = float(L - nk.sizes()["n_unique"])
        # one call = cg_init + 20 iterations; per iteration: the canonical unfused model
        jobs.append(("cg_iteration", lambda: nk.cg(f, 20, x=x, res_hist=hist), 20 * (168.0 * L + b_gs),
                     20 * ((12.0 * (N + 1) + 27.0) * L + gs_adds), max(1, reps // 10)))
    for name, fn, nbytes, flops, r in jobs:
        if name == "gs":
            v.copy_(u)                                         # 50 in-place gs scale shared entries by <= 8^50: finite
        best, med = _time(fn, r)
        per = 20.0 if name == "cg_iteration" else 1.0
        rows.append(dict(kernel=name, E=mesh.E, N=N, L=L, us_best=best / per, us_median=med / per,
                         gbs=nbytes / best / 1e3, gflops=flops / best / 1e3,
                         working_set_mb=(72.0 * L) / 1e6, l2_resident=bool(72.0 * L <= L2_BYTES)))
    nk.close()
    del u, w, v
    torch.cuda.empty_cache()
    return rows


def config4_points(which, reps=None):
    """(csv header, generator of (csv rows of one point, its mesh))."""
    from workloads import E_SWEEP, N_SWEEP, SWEEP_REPEATS, sweep_mesh
    reps = reps or SWEEP_REPEATS
    peak, kind = _peak()
    points = []
    if which in ("e", "both"):
        points += [("4a", p) for p in E_SWEEP]
    if which in ("n", "both"):
        points += [("4b", p) for p in N_SWEEP]
    if which == "big":
        points += [("big", p) for p in BIG_SWEEP]
    header = ("sweep,kernel,E,N,L,us_best,us_median,model_GBs,frac_of_%s_copy_peak,frac_of_8TBs,model_GFLOPs,"
              "working_set_MB,l2_resident" % kind)

    def gen():
        for tag, p in points:
            mesh = sweep_mesh(p)
            rows = [f"{tag},{r['kernel']},{r['E']},{r['N']},{r['L']},{r['us_best']:.2f},{r['us_median']:.2f},"
                    f"{r['gbs']:.1f},{r['gbs'] / peak:.4f},{r['gbs'] / 8000.0:.4f},{r['gflops']:.1f},"
                    f"{r['working_set_mb']:.1f},{int(r['l2_resident'])}" for r in run_point(mesh, reps, tag == "big")]
            yield rows, mesh
    return header, gen()


PAPER_HEADER = "N,E,n_local,dofs_E_N3,ms_per_100_iterations_mean_of_5,GDOFS,final_residual,solve_path"


def paper_points():
    """The paper's own sweep (S 8(f) f-2, Figs 7-12): N in {4, 6, 8}, E = 2^1 .. 2^14,
    100 warm-up + 100 timed CG iterations, mean of 5 runs, GDOFS = E N^3 100 / (t 1e9) (Eq. 1) and the
    final residual.  Meshes and RHS are this repo's seeded bricks (amplitude 0.05, seed 1004): the
    paper's own generator is not available, so only the SHAPE of its curves is comparable.
    Yields (csv row, mesh, f, residual history as numpy)."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    from workloads import brick_mesh, rhs_unique, sweep_brick
    from workloads.configs import SWEEP_AMPLITUDE, SWEEP_SEED
    for N in (4, 6, 8):
        for k in range(1, 15):
            mesh = brick_mesh(*sweep_brick(k), N, SWEEP_AMPLITUDE)
            nk = Nekbone.from_mesh(mesh)
            f_np = rhs_unique(mesh, SWEEP_SEED)
            f = torch.from_numpy(f_np).cuda()
            x = nk.empty()
            hist = torch.empty(101, dtype=torch.float64, device="cuda")
            nk.cg(f, 100, x=x, res_hist=hist)                       # 100 warm-up iterations
            torch.cuda.synchronize()
            ts = []
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                nk.cg(f, 100, x=x, res_hist=hist)
                e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            t = float(np.mean(ts))
            dofs = mesh.E * N ** 3
            h = hist.cpu().numpy()
            row = (f"{N},{mesh.E},{mesh.L},{dofs},{t:.4f},{dofs * 100 / (t * 1e-3) / 1e9:.4f},"
                   f"{float(h[-1]):.6e},{nk.solve_path()}")
            nk.close()
            yield row, mesh, f_np, h


def coop_points():
    """nk_cg per iteration on small meshes: CUDA graph replay ("coop" = 0) against the cooperative whole-solve launch
    ("coop" = 1); the measurement behind NK_COOP_AUTO_MAX_L.  N in {3, 4, 6, 7, 8, 9, 11}, E = 2^1 .. 2^14 up to 2^22
    points; mean of 5 timed solves of 100 iterations after a warm-up solve."""
    import torch
    from paper_2606_12650_b200 import Nekbone
    from workloads import brick_mesh, rhs_unique, sweep_brick
    from workloads.configs import SWEEP_AMPLITUDE, SWEEP_SEED

    def timed(nk, f, x, h):
        nk.cg(f, 100, x=x, res_hist=h)
        torch.cuda.synchronize()
        ts = []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            nk.cg(f, 100, x=x, res_hist=h)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.mean(ts))

    yield "N,E,n_local,graph_us_per_iteration,cooperative_us_per_iteration,graph_over_cooperative,default_path"
    for N in (3, 4, 6, 7, 8, 9, 11):
        for k in range(1, 15):
            mesh = brick_mesh(*sweep_brick(k), N, SWEEP_AMPLITUDE)
            if mesh.L > (1 << 22):
                break
            nk = Nekbone.from_mesh(mesh)
            default_path = nk.solve_path()
            f = torch.from_numpy(rhs_unique(mesh, SWEEP_SEED)).cuda()
            x, h = nk.empty(), torch.empty(101, dtype=torch.float64, device="cuda")
            nk.set_option("coop", 0)
            tg = timed(nk, f, x, h)
            nk.set_option("coop", 1)
            tc = timed(nk, f, x, h)
            nk.close()
            yield f"{N},{mesh.E},{mesh.L},{tg * 10:.2f},{tc * 10:.2f},{tg / tc:.3f},{default_path}"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--which", default="both", choices=["e", "n", "both", "big", "paper", "coop"])
    ap.add_argument("--reps", type=int, default=None)
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    lines = []
    if args.which == "coop":
        for row in coop_points():
            lines.append(row)
            print(row, flush=True)
    elif args.which == "paper":
        lines.append(PAPER_HEADER)
        for row, _, _, _ in paper_points():
            lines.append(row)
            print(row, flush=True)
    else:
        header, points = config4_points(args.which, args.reps)
        lines.append(header)
        for rows, _ in points:
            for row in rows:
                lines.append(row)
                print(row, flush=True)
    if args.out:
        with open(args.out, "w") as fh:
            fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
