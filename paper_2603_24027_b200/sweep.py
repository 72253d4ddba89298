"""Accuracy / memory sweep of the interface store (BASELINE.json configs[4]; the shape of the paper's Fig. 3).

For one workload (default C3, 256x256x128) and a few seeded designs: store dtype in {float32, float16, bfloat16,
float8_e4m3+scale, float8_e4m3+mx32 (a scale byte per 32 values)} x k in {1,2,4,8,16,32} x {linear, cubic}; --paper-fp8 adds the paper's five unscaled float8
flavours (e4m3b11fnuz, e5m2fnuz, e4m3fnuz, e4m3, e3m4).  Reports, per setting, the store bytes
(fdtd_store_bytes), the paper's compression factor (32/bits)*k, the gradient throughput and the
cosine similarity (eq. 2) of grad_eps against the (float32, k = 1, linear) gradient of the same design,
averaged over the designs (PAPER.md:59 averages over 10 gradients).

  python -m paper_2603_24027_b200.sweep [--workload C3] [--nsteps T] [--seeds 3] [--out sweep.json]

Everything numerical runs in the CUDA library; this file only loops over settings and forms the cosine.
"""
import argparse
import dataclasses
import json
import sys
import time

import numpy as np

from . import workloads as W


def run(args):
    import torch
    from . import fdtd
    base_seed = {"C1": 1001, "C2": 1002, "C3": 1003, "C4": 1004}[args.workload]
    dtypes = [W.F32, W.F16, W.BF16, W.F8E4M3_SCALED, W.F8E4M3_MX32] + (list(W.PAPER_FP8) if args.paper_fp8 else [])
    ks = [int(x) for x in args.k.split(",")]
    interps = [W.LINEAR, W.CUBIC] if args.cubic else [W.LINEAR]
    acc = {}
    for si in range(args.seeds):
        kw = {"seed": base_seed + 1000 * si}
        if args.nsteps:
            kw["nsteps"] = args.nsteps
        w = W.BY_NAME[args.workload](**kw)
        if args.field_scale != 1.0:
            w = dataclasses.replace(w, sources=[dataclasses.replace(q, wave=(q.wave * args.field_scale).astype(np.float32))
                                                for q in w.sources])
        eps = torch.from_numpy(w.eps).cuda()
        sim = fdtd.Sim(eps, W.DX, W.DT, w.pml, design=w.design, monitor=w.monitor)
        sim.set_workspace(w.nsteps, W.F32, 1)                  # the largest store of the sweep; reused by every setting
        extra = dict(w.extra)
        ref = None
        for dtype in dtypes:
            for k in ks:
                for interp in interps:
                    if interp == W.CUBIC and k == 1:
                        continue
                    torch.cuda.synchronize()
                    t0 = time.perf_counter()
                    mon = sim.forward(w.nsteps, w.sources, dtype, k)
                    mon_np = mon.cpu().numpy()
                    if w.loss == "pulse_shape" and "target_amp" not in extra:   # fixed once from the first forward run
                        A = np.asarray(w.extra["A"], dtype=np.float64).reshape(mon_np.shape[2:])
                        extra["target_amp"] = 0.5 * float(np.max(np.abs(np.tensordot(mon_np[:, 0].astype(np.float64), A, axes=3))))
                    L, d = W.loss_and_cotangent(w, mon_np, extra)
                    g = sim.reverse(None, torch.from_numpy(d.astype(np.float32)).cuda(), interp)
                    torch.cuda.synchronize()
                    dt = time.perf_counter() - t0
                    g = g.cpu().numpy().astype(np.float64)
                    if ref is None:
                        assert dtype == W.F32 and k == 1 and interp == W.LINEAR
                        ref = g
                    key = (dtype, k, interp)
                    a = acc.setdefault(key, {"cos": [], "bytes": sim.store_bytes(), "sec": []})
                    a["cos"].append(W.cosine_similarity(g, ref) if np.isfinite(g).all() and np.abs(g).max() > 0 else float("nan"))
                    a["sec"].append(dt)
        sim.destroy()
        del sim
    rows = []
    f32k1 = acc[(W.F32, 1, W.LINEAR)]["bytes"]
    for (dtype, k, interp), a in acc.items():
        rows.append({"dtype": W.DTYPE_NAMES[dtype], "k": k, "interp": "cubic" if interp == W.CUBIC else "linear",
                     "store_bytes": int(a["bytes"]), "byte_ratio_vs_f32_k1": f32k1 / a["bytes"],
                     "paper_factor": 32 // W.DTYPE_BITS[dtype] * k, "cosine_mean": float(np.mean(a["cos"])),
                     "cosine_min": float(np.min(a["cos"])), "designs": len(a["cos"]),
                     "mcells_per_s_incl_host_loss": float(w.cells) * w.nsteps / float(np.mean(a["sec"])) / 1e6})
    return {"workload": args.workload, "grid": list(w.shape), "nsteps": w.nsteps, "seeds": args.seeds, "rows": rows}


def to_markdown(res):
    out = [f"Sweep on {res['workload']} {res['grid']} x {res['nsteps']} steps, {res['seeds']} seeded design(s); cosine vs (float32, k=1, linear)\n",
           "| dtype | k | interp | store MB | bytes ratio | (32/bits)*k | cosine mean | cosine min | 1 - cosine mean | Mcell-upd/s (incl. host loss) |",
           "|---|---|---|---|---|---|---|---|---|---|"]
    for r in res["rows"]:
        out.append(f"| {r['dtype']} | {r['k']} | {r['interp']} | {r['store_bytes'] / 1e6:.1f} | {r['byte_ratio_vs_f32_k1']:.2f} | "
                   f"{r['paper_factor']} | {r['cosine_mean']:.6f} | {r['cosine_min']:.6f} | {1.0 - r['cosine_mean']:.2e} | "
                   f"{r['mcells_per_s_incl_host_loss']:.0f} |")
    return "\n".join(out)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--nsteps", type=int, default=0)
    ap.add_argument("--seeds", type=int, default=3)
    ap.add_argument("--k", default="1,2,4,8,16,32")
    ap.add_argument("--no-cubic", dest="cubic", action="store_false")
    ap.add_argument("--paper-fp8", action="store_true", help="add the paper's five unscaled float8 flavours (PAPER.md:53)")
    ap.add_argument("--field-scale", type=float, default=1.0,
                    help="multiply the source amplitude: the unscaled float8 casts depend on the absolute field level")
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    res = run(args)
    if args.out:
        with open(args.out, "w") as f:
            json.dump(res, f, indent=1)
    print(to_markdown(res))


if __name__ == "__main__":
    sys.exit(main())
