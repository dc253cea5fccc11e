"""Compute a steady ship-wave pattern: the paper's whole method (PAPER.md sections 3-4) from the command line.

    python -m paper_1403_5044_b200.solve --N 361 --M 121 --h 0.15 --x1 -14 --froude 0.7 --eps 1.0 \\
        [--bandwidth 31] [--continuation 0.5,1.0] [--jv fd|analytic] [--forcing] [--out surface.npz]

Builds the block-banded linear-Jacobian preconditioner (section 4.2, App. B/C), runs the damped inexact
Newton-GMRES iteration (section 4.1) from the flat surface (L227) - through the given source strengths in turn
when --continuation is used (L229) - and writes the free surface zeta(x, y), the potential phi(x, y) and the
unknown vector u (eq. (18)) to an .npz file.  Everything numerical runs in libsws / libsws_jfnk on the GPU; this
file only parses arguments, reads the nodal planes zeta, phi back from the library (sws_get_fields_host) and
prints the Newton log.  There is no CPU fallback.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--N", type=int, default=91)
    ap.add_argument("--M", type=int, default=31)
    ap.add_argument("--h", type=float, default=0.3, help="dx = dy")
    ap.add_argument("--x1", type=float, default=-9.0)
    ap.add_argument("--froude", type=float, default=0.7)
    ap.add_argument("--eps", type=float, default=1.0)
    ap.add_argument("--n-rad", type=float, default=0.05)
    ap.add_argument("--bandwidth", type=int, default=0, help="odd block bandwidth of the preconditioner (0: all of D)")
    ap.add_argument("--continuation", default="", help="comma-separated source strengths to pass through, ending at --eps")
    ap.add_argument("--jv", choices=["fd", "analytic"], default="fd")
    ap.add_argument("--forcing", action="store_true", help="Eisenstat-Walker inner tolerances")
    ap.add_argument("--ftol", type=float, default=1e-9)
    ap.add_argument("--eta", type=float, default=1e-3)
    ap.add_argument("--restart", type=int, default=60)
    ap.add_argument("--device", type=int, default=0)
    ap.add_argument("--f64-panels", action="store_true", help="keep the preconditioner's factor panels in FP64 (default FP32)")
    ap.add_argument("--out", default="")
    a = ap.parse_args(argv)

    import torch

    import paper_1403_5044_b200 as sws
    import paper_1403_5044_b200.jfnk as jf
    if not torch.cuda.is_available():
        raise SystemExit("paper_1403_5044_b200.solve: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(a.device)
    p = dict(N=a.N, M=a.M, x1=a.x1, y1=0.0, dx=a.h, dy=a.h, froude=a.froude, eps=a.eps, n_rad=a.n_rad, dy_scheme=0)
    stages = [float(v) for v in a.continuation.split(",") if v.strip()]
    if not stages or stages[-1] != a.eps:
        stages.append(a.eps)
    # flat surface, uniform stream (L227): phi_1 = x_1, phi_x = 1, zeta_1 = 0, zeta_x = 0
    u0 = np.zeros(2 * (a.N + 1) * a.M)
    blk = u0[:(a.N + 1) * a.M].reshape(a.M, a.N + 1)
    blk[:, 0] = a.x1
    blk[:, 1:] = 1.0
    kw = dict(ftol=a.ftol, eta=a.eta, restart=a.restart, gmres_maxit=4 * a.restart, jv_mode=2 if a.jv == "fd" else 0,
              forcing=int(a.forcing), eta_max=0.5)
    t0 = time.perf_counter()
    with sws.Context(p, max_batch=1, device=a.device) as ctx, \
            jf.Preconditioner(p, bandwidth=a.bandwidth, device=a.device, f32_panels=not a.f64_panels) as pc, jf.Solver(ctx, pc, a.restart) as s:
        t1 = time.perf_counter()
        u, stats, done = s.continuation(torch.from_numpy(u0).cuda(a.device), stages, **kw)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        F = ctx.residual(u)
        res = float(F.abs().max())
        zeta, phi, _, _ = ctx.fields_host()      # the nodal planes of the state sws_residual just evaluated
    u = u.cpu().numpy()
    report = {"mesh": f"{a.N}x{a.M}", "h": a.h, "froude": a.froude, "eps_reached": stages[done - 1] if done else None,
              "converged": done == len(stages), "stages": [dict(eps=e, steps=st["steps"], jv_products=st["jv_products"],
                                                                residual_evals=st["residual_evals"],
                                                                converged=st["converged"])
                                                           for e, st in zip(stages, stats)],
              "residual_inf": res, "setup_s": t1 - t0, "solve_s": t2 - t1,
              "zeta_min": float(zeta.min()), "zeta_max": float(zeta.max())}
    print(json.dumps(report))
    if a.out:
        np.savez(a.out, u=u, zeta=zeta, phi=phi, x=a.x1 + a.h * np.arange(a.N), y=a.h * np.arange(a.M), report=json.dumps(report))
    return 0 if report["converged"] else 1


if __name__ == "__main__":
    raise SystemExit(main())
