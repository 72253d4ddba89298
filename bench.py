#!/usr/bin/env python
"""bench.py — throughput of the time-reversible FDTD gradient loop (forward + reverse) on B200.

One "step" = one pass of the whole hot path over one synthetic workload: fdtd_forward(nsteps) including record /
monitor writes, the (harness) loss cotangent, fdtd_reverse including dequant / interpolate / inject, adjoint and
gradient accumulation.  Metric: Mcell-updates/s = nx*ny*nz*nsteps / (t_forward + t_reverse), whole job.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C1|C3|C4] [--nsteps T] [--impl reference]

N > 1 (under torchrun): the path does not shard (BASELINE.json: one GPU) — N independent replicas with different
seeded designs (the paper's "mean over 10 gradients"), no collective on the data path; weak scaling.
--impl reference times the CPU oracle (as it stands) on the host cores on a bounded sample of the same workload.
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

from paper_2603_24027_b200 import workloads as W  # noqa: E402

METRIC = "Mcell-updates/s fwd+reverse (incl record/inject)"
UNIT = "Mcell-updates/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_ burst)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def make_workload(name, nsteps, seed_offset=0, store=None, k=0):
    w = _make_workload(name, nsteps, seed_offset)
    if store is not None or k:
        import dataclasses
        w = dataclasses.replace(w, store_dtype=w.store_dtype if store is None else store, k=k or w.k)
    return w


STORE_BY_NAME = {v: k for k, v in W.DTYPE_NAMES.items()}


def _make_workload(name, nsteps, seed_offset=0):
    f = W.BY_NAME[name]
    kw = {}
    if nsteps:
        kw["nsteps"] = nsteps
    if seed_offset:
        kw["seed"] = {"C1": 1001, "C2": 1002, "C3": 1003, "C4": 1004}[name] + 1000 * seed_offset
    return f(**kw)


def replica_seed_offset(rank):
    """Replica r of an N-GPU run gets its own seeded design (the paper's batch of independent gradients)."""
    return int(rank)


def reduce_max(values, world, device=None):
    """Max over ranks of a list of floats (device timings): the slowest replica sets the job's time."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def whole_job_value(cells, nsteps, steps, world, total_ms):
    """Mcell-updates/s of the whole job: every replica's cell updates over the slowest replica's time."""
    return float(cells) * nsteps * steps * world / (total_ms * 1e-3) / 1e6


# DRAM bytes per launch of a kernel group (read + write, summed over the group's kernels) from the committed ncu --set full
# captures (profiles/r01d_c2.md, r01e_c3_c2.md, r01c_full.md): what roofline.traffic reports beside the algorithmic bytes.  ncu flushes the caches
# between launches, so on C2 (working set of the order of the L2) arrays that stay in L2 do not appear as writes.
NCU_TRAFFIC = {
    ("C2", "fwd_e"): 88.2e6, ("C2", "fwd_h"): 76.7e6, ("C2", "inv_h"): 32.2e6, ("C2", "adj_h"): 76.6e6,
    ("C2", "grad_inv_e"): 44.3e6, ("C2", "adj_e"): 88.4e6,
    ("C3", "fwd_e"): 364.7e6, ("C3", "fwd_h"): 314.7e6, ("C3", "inv_h"): 175.6e6, ("C3", "adj_h"): 335.2e6,
    ("C3", "grad_inv_e"): 231.8e6, ("C3", "adj_e"): 382.7e6,
    ("C4", "fwd_fused"): 6112.8e6, ("C4", "fwd_fused_slabs"): 3242.1e6,
}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index, period_ms=200):
        self.lines = []
        self.proc = None
        if period_ms <= 0:
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", str(int(period_ms)),
                                          "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.lines:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                c = float(parts[0])
                mx = float(parts[1])
            except ValueError:
                continue
            if t0 - 0.05 <= ts <= t1 + 0.15:
                sm.append(c)
                for n, v in zip(names, parts[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def run_gpu(args, rank, world):
    import torch
    import torch.distributed as dist
    from paper_2603_24027_b200 import fdtd

    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    w = make_workload(args.workload, args.nsteps, seed_offset=replica_seed_offset(rank),
                      store=STORE_BY_NAME[args.store] if args.store else None, k=args.k)
    flags = fdtd.WS_REVERSE | fdtd.WS_HOST_IO
    eps_dev = torch.from_numpy(w.eps).to(dev)
    sim = fdtd.Sim(eps_dev, W.DX, W.DT, w.pml, design=w.design, monitor=w.monitor,
                   store_mode=fdtd.STORE_TANGENTIAL if args.tangential else fdtd.STORE_ALL)
    sim.set_workspace(w.nsteps, w.store_dtype, w.k, flags)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    extra = {}

    def loss_cotangent_dev(mon):
        # harness-level objective on the small monitor tensor (SURVEY layer L4), on the device for the device-timed leg
        L, d = W.loss_and_cotangent(w, mon.cpu().numpy(), extra)
        return L, torch.from_numpy(d.astype(np.float32)).to(dev)

    # one untimed pass fixes the objective's constants (C3's target amplitude) and the cotangent, so that the timed
    # device leg contains only library work
    mon = sim.forward(w.nsteps, w.sources, w.store_dtype, w.k, flags=flags)
    if w.loss == "pulse_shape":
        A = np.asarray(w.extra["A"], dtype=np.float64).reshape(mon.shape[2:])
        extra.update(w.extra)
        extra["target_amp"] = 0.5 * float(np.max(np.abs(np.tensordot(mon[:, 0].cpu().numpy().astype(np.float64), A, axes=3))))
    L0, dmon = loss_cotangent_dev(mon)
    grad = sim.reverse(None, dmon, W.LINEAR)
    sim.sync()
    assert torch.isfinite(grad).all().item(), "gradient is not finite"
    if not args.nsteps:
        assert grad.abs().max().item() > 0, "gradient is zero on the full-length workload"

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def one_step(timed):
        flush.fill_(1)                                # L2 flush between steps (not timed)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        e[0].record()
        sim.forward(w.nsteps, w.sources, w.store_dtype, w.k, flags=flags)
        e[1].record()
        sim.reverse(None, dmon, W.LINEAR)
        e[2].record()
        torch.cuda.synchronize()
        return e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2])

    for _ in range(args.warmup):
        one_step(False)
    barrier()
    sampler = ClockSampler(local, args.clock_sample_ms) if rank == 0 else None
    l0 = sim.launch_count()
    t0 = time.time()
    tf, tr = [], []
    for _ in range(args.steps):
        a, b = one_step(True)
        tf.append(a)
        tr.append(b)
    barrier()
    t1 = time.time()
    launches = sim.launch_count() - l0
    clocks = sampler.stop(t0, t1) if sampler else None
    tot_ms = float(np.sum(tf) + np.sum(tr))
    tot_ms, f_ms, r_ms = reduce_max([tot_ms, float(np.sum(tf)), float(np.sum(tr))], world, dev)
    value = whole_job_value(w.cells, w.nsteps, args.steps, world, tot_ms)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    eps_host = torch.from_numpy(w.eps).pin_memory()
    mon_host = torch.empty(w.monitor_shape(), dtype=torch.float32).pin_memory()
    dmon_host = torch.empty(w.monitor_shape(), dtype=torch.float32).pin_memory()
    lo, hi = w.design
    grad_host = torch.empty([hi[a] - lo[a] for a in range(3)], dtype=torch.float32).pin_memory()

    def e2e_step():
        sim.set_eps_host(eps_host)
        sim.forward_host(w.nsteps, w.sources, w.store_dtype, w.k, mon_host)
        L, d = W.loss_and_cotangent(w, mon_host.numpy(), extra)
        dmon_host.copy_(torch.from_numpy(np.ascontiguousarray(d, dtype=np.float32)))
        sim.reverse_host(dmon_host, W.LINEAR, grad_host)
        return L
    e2e_step()
    barrier()
    ne2e = max(1, min(args.steps, 3))
    te = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(ne2e):
        e2e_step()
    ev1.record()
    barrier()
    e2e_ms = max(ev0.elapsed_time(ev1), 0.0)
    e2e_wall = (time.perf_counter() - te) * 1e3
    e2e_ms = max(e2e_ms, e2e_wall)                      # host work sits between GPU segments: take the longer clock
    e2e_ms = reduce_max([e2e_ms], world, dev)[0]
    amp_bytes = sum(int(np.prod([s.hi[a] - s.lo[a] for a in range(3)])) * 4 for s in w.sources if s.amp is not None)
    e2e = {"value": whole_job_value(w.cells, w.nsteps, ne2e, world, e2e_ms), "unit": UNIT,
           "h2d_bytes_per_step": int(w.eps.nbytes + dmon_host.numel() * 4 + amp_bytes + sum(s.wave.nbytes for s in w.sources)),
           "d2h_bytes_per_step": int(mon_host.numel() * 4 + grad_host.numel() * 4), "steps": ne2e}
    if world > 1:
        dist.barrier()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- per-kernel roofline (rank 0): each stencil kernel timed alone, back to back, CUDA events on its stream ----
    peak, peak_src = load_peaks()
    sim.forward(w.nsteps, w.sources, w.store_dtype, w.k, flags=flags)
    nrec = sim.num_slots() - 1
    fused = sim.uses_fused(w.nsteps)   # large grids: H half-step of step m and E half-step of step m+1 in one marching kernel
    counts = {"fwd_e": 1 if fused else w.nsteps, "fwd_h": 1 if fused else w.nsteps, "inv_h": w.nsteps, "adj_h": w.nsteps,
              "grad_inv_e": w.nsteps, "adj_e": w.nsteps, "record": nrec + 1, "inject_h": w.nsteps, "inject_e": w.nsteps,
              "fwd_fused": w.nsteps - 1, "fwd_fused_slabs": w.nsteps - 1}
    kernels = {}
    for kid, name in enumerate(fdtd.Sim.KERNELS):
        if kid >= 9 and not fused:
            continue
        if 6 <= kid <= 8:
            sim.forward(min(w.nsteps, 4 * w.k), w.sources, w.store_dtype, w.k, flags=flags)
        flush.fill_(1)
        ms, by = sim.profile_kernel(kid, warm=3, reps=20)
        kernels[name] = {"us": ms * 1e3, "algo_bytes": by, "gbs": by / (ms * 1e-3) / 1e9, "launches_per_step": counts[name]}
    tot = sum(v["us"] * v["launches_per_step"] for v in kernels.values())
    for v in kernels.values():
        v["share"] = v["us"] * v["launches_per_step"] / tot
        v["frac"] = v["gbs"] / peak
    dom = max(kernels, key=lambda n: kernels[n]["share"])
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dom]["gbs"] / peak, "traffic": NCU_TRAFFIC.get((args.workload, dom)), "peak_source": peak_src,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum per launch (all kernels of the group), ncu --set full, "
                                  "profiles/r01d_c2.md, r01e_c3_c2.md, r01c_full.md" if (args.workload, dom) in NCU_TRAFFIC else None,
                "how": "kernel group timed alone (its lean and general kernel side by side, as in the step): 20 back-to-back launches "
                       "between CUDA events on the library's stream after 3 warm-up launches; achieved = algorithmic bytes per "
                       "launch (DESIGN.md Roofline) / mean launch time",
                "launch_us": kernels[dom]["us"], "algo_bytes": kernels[dom]["algo_bytes"]}
    # whole-pass effective bandwidth: algorithmic bytes of all stencil launches of one step / measured time
    fwd_names = ("fwd_e", "fwd_h", "fwd_fused", "fwd_fused_slabs")
    algo_fwd = sum(kernels[n]["algo_bytes"] * kernels[n]["launches_per_step"] for n in fwd_names if n in kernels) \
        + kernels["record"]["algo_bytes"] * (nrec + 1)
    algo_rev = sum(kernels[n]["algo_bytes"] for n in ("inv_h", "adj_h", "grad_inv_e", "adj_e", "inject_h", "inject_e")) * w.nsteps
    fwd_gbs = algo_fwd / (f_ms / args.steps * 1e-3) / 1e9
    # the same forward time against the bytes of the two-kernel form (76 B per cell): comparable across paths
    algo_fwd2 = (kernels["fwd_e"]["algo_bytes"] + kernels["fwd_h"]["algo_bytes"]) * w.nsteps + kernels["record"]["algo_bytes"] * (nrec + 1)
    fwd2_gbs = algo_fwd2 / (f_ms / args.steps * 1e-3) / 1e9
    rev_gbs = algo_rev / (r_ms / args.steps * 1e-3) / 1e9

    # ---- CPU baseline: the oracle as it stands on a bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if world == 1 and not args.no_cpu and not args.tangential:
        cpu = cpu_baseline(args.workload, args.cpu_steps)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": tot_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{w.name}: {w.shape[0]}x{w.shape[1]}x{w.shape[2]} f32 Yee grid, {w.pml}-cell CPML, {w.nsteps} steps, "
                               f"{W.DTYPE_NAMES[w.store_dtype]} store, k={w.k}, linear interpolation, loss={w.loss}",
                   "grid": list(w.shape), "pml": w.pml, "nsteps": w.nsteps, "store_dtype": W.DTYPE_NAMES[w.store_dtype], "k": w.k,
                   "store_components": "tangential (12 slices per slot)" if args.tangential else "all six per face (36 slices per slot)",
                   "l2": "256 MB write between timed steps flushes L2; inside a step the working set "
                         f"({13 * w.cells * 4 / 1e6:.0f} MB of fields) is what the workload itself keeps resident",
                   "replicas": world, "parallelism": "replicas only (the path runs on one GPU)"},
        "forward_mcells_per_s": whole_job_value(w.cells, w.nsteps, args.steps, world, f_ms),
        "reverse_mcells_per_s": whole_job_value(w.cells, w.nsteps, args.steps, world, r_ms),
        "forward_ms": f_ms / args.steps, "reverse_ms": r_ms / args.steps,
        "store_bytes": sim_store_bytes(sim, w, flags), "store_bytes_per_step": sim_store_bytes(sim, w, flags) / w.nsteps,
        "store_bytes_f32_k1": (w.nsteps + 1) * sim.slot_values() * (3 if args.tangential else 1) * 4,   # all six components
        "effective_gbs": {"forward": fwd_gbs, "reverse": rev_gbs, "forward_frac_of_peak": fwd_gbs / peak,
                          "reverse_frac_of_peak": rev_gbs / peak, "forward_fused": bool(fused),
                          "forward_two_kernel_equivalent": fwd2_gbs, "forward_two_kernel_equivalent_frac": fwd2_gbs / peak,
                          # also against the nominal HBM3e figure (8000 GB/s)
                          "forward_frac_of_nominal_8000": fwd_gbs / 8000.0, "reverse_frac_of_nominal_8000": rev_gbs / 8000.0},
        "roofline": roofline, "kernels": kernels, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "loss": L0, "grad_abs_max": float(grad.abs().max().item()),
    }
    if cpu is not None:
        out["cpu_baseline"] = cpu
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def sim_store_bytes(sim, w, flags):
    if not sim.store_bytes():
        sim.forward(w.nsteps, w.sources, w.store_dtype, w.k, flags=flags)
    return int(sim.store_bytes())


def oracle_pass(w, nsteps):
    """One forward + reverse of the CPU oracle (f32) on the first nsteps of workload w.  Returns (seconds, cores)."""
    import dataclasses
    from oracle import fdtd_oracle as orc
    srcs = [dataclasses.replace(s, wave=s.wave[:nsteps]) for s in w.sources]
    ws = dataclasses.replace(w, nsteps=nsteps, sources=srcs)
    s = orc.OracleSim(32, ws.eps, ws.pml, W.S)
    s.set_design(*ws.design)
    s.set_monitor(*ws.monitor)
    for q in srcs:
        s.add_source(q.comp, q.lo, q.hi, q.amp, q.wave)
    t0 = time.perf_counter()
    s.forward(nsteps, ws.store_dtype, ws.k)
    tf = time.perf_counter() - t0
    ex = dict(ws.extra)
    ex["target_amp"] = 1.0
    L, d = W.loss_and_cotangent(ws, s.monitor_record(), ex)
    t1 = time.perf_counter()
    s.reverse(None, d, orc.LINEAR)
    tr = time.perf_counter() - t1
    return tf, tr, orc.get_threads()


def cpu_baseline(workload, nsteps):
    w = make_workload(workload, None)
    nsteps = min(nsteps, w.nsteps)
    tf, tr, cores = oracle_pass(w, nsteps)
    cu = float(w.cells) * nsteps
    return {"value": cu / (tf + tr) / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{w.name} grid, first {nsteps} of {w.nsteps} steps, forward + reverse, float32 oracle, "
                      f"{W.DTYPE_NAMES[w.store_dtype]} k={w.k}",
            "forward_mcells_per_s": cu / tf / 1e6, "reverse_mcells_per_s": cu / tr / 1e6, "seconds": tf + tr}


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores; each step = a bounded sample of the workload."""
    if rank != 0:
        return
    w = make_workload(args.workload, None)
    sample = min(args.ref_steps, w.nsteps)
    for _ in range(args.warmup):
        oracle_pass(w, sample)
    t = 0.0
    cores = 0
    for _ in range(args.steps):
        tf, tr, cores = oracle_pass(w, sample)
        t += tf + tr
    value = float(w.cells) * sample * args.steps / t / 1e6
    desc = (f"{w.name} grid, first {sample} of {w.nsteps} steps per bench step, forward + reverse, float32 oracle, "
            f"{W.DTYPE_NAMES[w.store_dtype]} k={w.k}")
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"{w.name}: {w.shape[0]}x{w.shape[1]}x{w.shape[2]} f32 Yee grid, {w.pml}-cell CPML, {w.nsteps} steps, "
                                  f"{W.DTYPE_NAMES[w.store_dtype]} store, k={w.k}, linear interpolation, loss={w.loss}",
                      "sample": desc},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--nsteps", type=int, default=0, help="override the workload's number of time steps")
    ap.add_argument("--cpu-steps", type=int, default=60, help="time steps of the cpu_baseline sample")
    ap.add_argument("--ref-steps", type=int, default=20, help="time steps per bench step of --impl reference")
    ap.add_argument("--store", default="", choices=[""] + sorted(STORE_BY_NAME), help="override the workload's store dtype")
    ap.add_argument("--k", type=int, default=0, help="override the workload's temporal subsampling factor")
    ap.add_argument("--tangential", action="store_true",
                    help="FDTD_STORE_TANGENTIAL: store only the 12 tangential slices per slot (a third of the bytes); no cpu_baseline")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--clock-sample-ms", type=int, default=200, help="nvidia-smi polling period during the timed region")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_gpu(args, rank, world)


if __name__ == "__main__":
    main()
