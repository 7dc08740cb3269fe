#!/usr/bin/env python
"""The sweeps of `python -m paper_2606_12650_b200.sweep` with the oracle beside every point.

    python tests/sweep_parity.py --which paper|e|n|both [--out file.csv]

The product's sweep tool only times (the product never imports the oracle); this script lives under tests/
because it does: for every point it sets the oracle up on the same seeded mesh and appends parity columns
to the timing rows, so that no number of the sweep rests on an unchecked code path.

* --which paper: N in {4, 6, 8}, E = 2^1 .. 2^14, 100 CG iterations.
  The paper's own correctness criterion is that the residual after the 100 iterations agrees between
  implementations for every (N, E) (section VIII-B, section VIII-C): columns
  oracle_final_residual, rel_diff_final, max_rel_diff_history (over the part of the history where the oracle's
  own rounding band is <= 1e-11), kstar, parity (pass = DESIGN.md R15 protocol, tests/parity.history_parity).
* --which e|n|both (BASELINE.json configs[3]): one application of ax_e, gs, ax on the sweep's input against
  the oracle over the whole vector; column parity_err = the largest R14-scaled error of the three, parity =
  pass at 1e-12.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
for p in (ROOT, HERE):
    if p not in sys.path:
        sys.path.insert(0, p)

from parity import elem_err, scaled_err, gs_scale, history_parity, oracle_variants   # noqa: E402


def paper_point_parity(mesh, f, hist_gpu):
    """Oracle CG (both builds) on the point's mesh; returns the parity columns."""
    from oracle.nko import Oracle
    niter = len(hist_gpu) - 1
    orc = Oracle.from_mesh(mesh)
    _, ho = orc.cg(f, niter)
    orc.close()
    rel_final = abs(hist_gpu[-1] - ho[-1]) / ho[-1] if ho[-1] > 0 else abs(hist_gpu[-1])
    if np.all(np.abs(hist_gpu - ho) <= 1e-10 * ho):
        return dict(oracle_final=ho[-1], rel_final=rel_final, worst=float(np.abs(hist_gpu / ho - 1).max()),
                    kstar=niter, ok=True)
    # flat 1e-10 failed somewhere: the band protocol decides
    ok, worst, kstar = history_parity(hist_gpu, ho, [h for _, h in oracle_variants(mesh, f, niter)])
    return dict(oracle_final=ho[-1], rel_final=rel_final, worst=worst, kstar=kstar, ok=ok)


def operator_point_parity(mesh, u):
    """max R14-scaled error of one application of ax_e, gs, ax on the GPU against the oracle."""
    import torch
    from oracle.nko import Oracle
    from paper_2606_12650_b200 import Nekbone
    P = mesh.n ** 3
    orc, gpu = Oracle.from_mesh(mesh), Nekbone.from_mesh(mesh)
    ud = torch.from_numpy(u).cuda()
    errs = [elem_err(gpu.ax_e(ud).cpu().numpy(), orc.ax_e(u), P),
            scaled_err(gpu.gs(ud.clone()).cpu().numpy(), orc.gs(u), gs_scale(u, mesh.glo_num)),
            elem_err(gpu.ax(ud).cpu().numpy(), orc.ax(u), P)]
    orc.close()
    gpu.close()
    return max(errs)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--which", default="paper", choices=["paper", "e", "n", "both"])
    ap.add_argument("--reps", type=int, default=None)
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    from paper_2606_12650_b200 import sweep
    lines = []
    if args.which == "paper":
        lines.append(sweep.PAPER_HEADER + ",oracle_final_residual,rel_diff_final,max_rel_diff_history,kstar,parity")
        for row, mesh, f, hist in sweep.paper_points():
            q = paper_point_parity(mesh, f, hist)
            lines.append(f"{row},{q['oracle_final']:.6e},{q['rel_final']:.2e},{q['worst']:.2e},{q['kstar']},"
                         f"{'pass' if q['ok'] else 'FAIL'}")
            print(lines[-1], flush=True)
    else:
        from workloads import sweep_field
        header, points = sweep.config4_points(args.which, args.reps)
        lines.append(header + ",parity_err,parity")
        for rows, mesh in points:
            err = operator_point_parity(mesh, sweep_field(mesh))
            for row in rows:
                lines.append(f"{row},{err:.2e},{'pass' if err <= 1e-12 else 'FAIL'}")
                print(lines[-1], flush=True)
    if args.out:
        with open(args.out, "w") as fh:
            fh.write("\n".join(lines) + "\n")
    if any(l.endswith("FAIL") for l in lines):
        raise SystemExit("sweep_parity: at least one point failed parity")


if __name__ == "__main__":
    main()
