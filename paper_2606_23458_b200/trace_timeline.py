"""Phase timeline of the persistent kernels (explicit step, CG iteration) from the instrumentation build.

    python -m paper_2606_23458_b200.trace_timeline [--n 1001] [--precision f64|f32] [--iteration 3] [--run-steps]

Builds libpff_trace.so if needed (the product sources with -DPFF_TRACE), steps config 5 of side n a few times, then
records one explicit step and one CG iteration: thread 0 of every CTA stamps clock64 / %globaltimer when, chunk by chunk,
its data has arrived, the node prologue, the element pass and the gather are done, and at the grid-wide phases of the
tail.  Prints per-chunk phase durations (SM cycles, mean over CTAs) and the tail as nanoseconds since the first CTA
started.  Measurement tooling only: no arithmetic of the method lives here.

Buffer layout (pff_trace_set): 256 int64 per CTA, [0,128) SM cycles, [128,256) nanoseconds; slot 0 = start, slots
1 + 4k .. 4 + 4k = chunk k (arrived, prologue, elements, gather), 100 = chunk phase over, 101 = after the first grid
barrier, 102 = interface nodes done, 103 = block partials written, 104 = after the second grid barrier, 105 = scalars
advanced.  The CG kernel's rows start at word 0, the step kernel's at word 256 * 1024.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def section(a, base, name, out):
    t = a[base:base + 1024 * 256].reshape(1024, 256)
    clk, gt = t[:, :128], t[:, 128:]
    act = clk[:, 0] != 0
    clk, gt = clk[act], gt[act]
    out.append(f"== {name}: {int(act.sum())} CTAs")
    if not act.any():
        return
    g0 = gt[:, 0].min()
    out.append(" chunk  CTAs    wait  prologue  elements   gather    total   (SM cycles, mean over CTAs)")
    rows = []
    for k in range(24):
        have = clk[:, 4 + 4 * k] != 0
        if not have.any():
            break
        c, prev = clk[have], (clk[:, 0] if k == 0 else clk[:, 4 * k])[have]
        d = [c[:, 1 + 4 * k] - prev, c[:, 2 + 4 * k] - c[:, 1 + 4 * k], c[:, 3 + 4 * k] - c[:, 2 + 4 * k],
             c[:, 4 + 4 * k] - c[:, 3 + 4 * k]]
        rows.append([x.mean() for x in d] + [sum(d).mean()])
        out.append(" %4d %6d %7.0f %9.0f %9.0f %8.0f %8.0f" % (k, have.sum(), *rows[-1]))
    out.append("  mean        %7.0f %9.0f %9.0f %8.0f %8.0f" % tuple(np.mean(rows, axis=0)))
    out.append(" phase (ns since the first CTA started)      min      mean       max")
    for label, i in (("start", 0), ("chunk phase over", 100), ("after grid barrier 1", 101), ("interface nodes done", 102),
                     ("block partials written", 103), ("after grid barrier 2", 104), ("scalars advanced", 105)):
        ok = gt[:, i] != 0
        if ok.any():
            v = gt[ok, i] - g0
            out.append(" %-40s %8d %9.0f %9d" % (label, v.min(), v.mean(), v.max()))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=1001)
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--iteration", type=int, default=3)
    ap.add_argument("--run-steps", action="store_true", help="record the step kernel pff_run_steps launches (deferred interface "
                    "update where the mesh allows it) instead of the one-call kernel of pff_explicit_step")
    args = ap.parse_args()
    sys.path.insert(0, ROOT)
    from paper_2606_23458_b200 import build
    os.environ["PFF_LIBRARY"] = build.build(trace=True)
    import torch
    import paper_2606_23458_b200 as pff
    from pff_inputs import config
    cfg = config(5, n=args.n)
    mesh = pff.Mesh(cfg["xy"], cfg["tri"], cfg["material"], precision=pff.PFF_F32 if args.precision == "f32" else pff.PFF_F64)
    st = mesh.new_state(u=cfg["u0"], d=cfg["d0"])
    dt, bc = 0.5 * mesh.dt_crit, mesh.bc()
    mesh.pff_init_accel(st, bc)
    for _ in range(5):
        mesh.pff_explicit_step(st, bc, dt)
        mesh.pff_damage_solve(st, rel_tol=1e-8, allow_noconv=True)
    buf = torch.zeros(2 * 256 * 1024, dtype=torch.int64, device=mesh.device)
    pff._check(mesh.L.pff_trace_set(mesh.h, buf.data_ptr(), args.iteration))
    if args.run_steps:  # three steps: every launch stamps the same rows, the last one stays
        mesh.pff_set_graph_mode(False)
        mesh.pff_run_steps(st, bc, dt, 3, damage_every=1, rel_tol=1e-8, allow_noconv=True)
    else:
        mesh.pff_explicit_step(st, bc, dt)
        mesh.pff_damage_solve(st, rel_tol=1e-8, allow_noconv=True)
    torch.cuda.synchronize()
    pff._check(mesh.L.pff_trace_set(mesh.h, None, args.iteration))
    a = buf.cpu().numpy().astype(np.int64)
    out = [f"cfg5_{args.n} {args.precision}: {mesh.n_chunks} chunks, {mesh.n_shared} interface nodes"]
    section(a, 0, f"CG iteration {args.iteration} (dmg_iter_chunk)", out)
    section(a, 256 * 1024, "explicit step (step_chunk_kernel)", out)
    print("\n".join(out))


if __name__ == "__main__":
    main()
