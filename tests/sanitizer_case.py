"""One small forward + reverse pass of the CUDA path, meant to be run under compute-sanitizer:

    compute-sanitizer --tool memcheck  python tests/sanitizer_case.py --graphs 1
    compute-sanitizer --tool initcheck python tests/sanitizer_case.py --graphs 0
    compute-sanitizer --tool racecheck python tests/sanitizer_case.py --fused 1      # smem ring of k_fused_he
    compute-sanitizer --tool racecheck python tests/sanitizer_case.py --grid odd     # scalar (V = 1) kernels

Not a pytest test (the sanitizer slows kernels 10-100x); the summaries it produced are kept under profiles/.
The run is C1-shaped (32^3, 8-cell CPML: vector kernels, every box class, design box on the shell) or the odd 14x13x12
grid (scalar kernels, T % k != 0), a few steps long, and ends with a finite, non-zero gradient.
"""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--grid", default="c1", choices=["c1", "odd"])
    ap.add_argument("--nsteps", type=int, default=37)
    ap.add_argument("--graphs", type=int, default=1)
    ap.add_argument("--fused", type=int, default=-1, help="-1 auto, 0 never, 1 forward and reverse marching kernels")
    ap.add_argument("--dtype", type=int, default=3, help="store dtype id (include/fdtd.h); 3 = e4m3 + per-slice scale")
    ap.add_argument("--k", type=int, default=4)
    ap.add_argument("--interp", type=int, default=1)
    ap.add_argument("--persist", type=int, default=-1, help="-1 auto, 0 never, 1 persistent cooperative step kernel")
    args = ap.parse_args()
    import torch
    from paper_2603_24027_b200 import fdtd, workloads as W
    w = W.c1(nsteps=args.nsteps) if args.grid == "c1" else W.tiny(nsteps=args.nsteps)
    sim = fdtd.Sim(torch.from_numpy(w.eps).cuda(), W.DX, W.DT, w.pml, design=w.design, monitor=w.monitor)
    sim.set_graphs(args.graphs)
    if args.fused >= 0:
        sim.set_fused(args.fused)
    if hasattr(sim, "set_persistent") and args.persist >= 0:
        sim.set_persistent(args.persist)
    mon = sim.forward(w.nsteps, w.sources, args.dtype, args.k)
    L, d = W.loss_and_cotangent(w, mon.cpu().numpy())
    grad = sim.reverse(None, torch.from_numpy(d.astype(np.float32)).cuda(), args.interp)
    sim.sync()
    g = grad.cpu().numpy()
    assert np.isfinite(g).all() and np.abs(g).max() > 0
    print(f"sanitizer_case: grid {w.shape} nsteps {w.nsteps} graphs {args.graphs} fused {args.fused} dtype {args.dtype} k {args.k} "
          f"interp {args.interp}: loss {L:.6e} max|grad| {np.abs(g).max():.6e} launches {sim.launch_count()}")


if __name__ == "__main__":
    main()
