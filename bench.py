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


# DRAM bytes per launch of a kernel group (dram__bytes_read.sum + dram__bytes_write.sum, summed over the group's kernels) from
# `ncu --set full` captures of THIS build: profiles/ncu_traffic.json, written by `python bench.py --ncu-import <raw.csv> ...`
# from the raw page of a capture and stamped with a hash of the kernel sources.  A stamp that does not match the sources on disk
# means the capture is stale: the traffic is then reported as null (with the reason), never silently reused.
NCU_JSON = os.path.join(ROOT, "profiles", "ncu_traffic.json")
KERNEL_SOURCES = ["fdtd_api.cu", "fdtd_dev.cuh", "fdtd_stencil.cuh", "fdtd_store.cuh", "fdtd_fused.cuh"]
# kernel group -> the kernels whose launches make up one "launch" of the group (names as ncu prints them, prefix match)
GROUP_KERNELS = {
    "fwd_e": ["k_row<0>", "k_lean_curlm<4, 0>", "k_lean_curlm<1, 0>", "k_gen_e"],
    "fwd_h": ["k_row<1>", "k_lean_h", "k_gen_h"],
    "inv_h": ["k_inv_h"],
    "adj_h": ["k_row<2>", "k_lean_curlm<4, 1>", "k_lean_curlm<1, 1>", "k_gen_adj_h"],
    "grad_inv_e": ["k_inv_e<", "k_grad("],
    "adj_e": ["k_row<3>", "k_lean_adj_e", "k_gen_adj_e"],
    "record": ["k_record"],
    "inject_h": ["k_inject"],
    "inject_e": ["k_inject"],
    "fwd_fused": ["k_fused_fp", "k_fused_he"],
    "rev_fused": ["k_fused_ip", "k_fused_he"],
    "grad": ["k_grad("],
    "adj_fused": ["k_fused_ap"],
    "adj_fused_slabs": ["k_gen_adj_h", "k_gen_adj_e"],
    "fwd_fused_slabs": ["k_gen_h", "k_gen_e"],
}


def kernel_source_hash():
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2603_24027_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def load_ncu_traffic(workload):
    """{group: bytes per launch} for the workload, or ({}, reason) when there is no capture of this build."""
    if not os.path.exists(NCU_JSON):
        return {}, "no profiles/ncu_traffic.json"
    with open(NCU_JSON) as f:
        d = json.load(f)
    e = d.get(workload)
    if not e:
        return {}, f"no ncu capture of {workload} in profiles/ncu_traffic.json"
    if e.get("kernel_source_hash") != kernel_source_hash():
        return {}, (f"ncu capture of {workload} is stale: taken from kernel sources {e.get('kernel_source_hash')}, "
                    f"the sources on disk are {kernel_source_hash()}")
    return e["groups"], e.get("source", "profiles/ncu_traffic.json")


def ncu_import(args):
    """bench.py --ncu-import raw.csv --workload W --ncu-note '...': read `ncu -i rep --page raw --csv` output of a capture
    made by `ncu --set full ... python bench.py --workload W --profile-only ...` (every group launched once, in
    Sim.KERNELS order) and store DRAM bytes per group launch in profiles/ncu_traffic.json."""
    import csv
    rows = list(csv.reader(open(args.ncu_import)))
    hdr = rows[0]
    ci = {n: hdr.index(n) for n in ("Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum")}
    units = rows[1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}

    def by(r, n):
        return float(r[ci[n]]) * scale[units[ci[n]]]
    tscale = {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}[units[ci["gpu__time_duration.sum"]]]
    launches = [(r[ci["Kernel Name"]], by(r, "dram__bytes_read.sum"), by(r, "dram__bytes_write.sum"),
                 float(r[ci["gpu__time_duration.sum"]]) * tscale) for r in rows[2:] if "fdtd::" in r[ci["Kernel Name"]]]
    groups, detail, pos = {}, {}, 0
    present = " ".join(l[0] for l in launches)
    for name in active_groups(None, "k_fused_fp" in present or "k_fused_he" in present, "k_fused_ip" in present, "k_fused_ap" in present):
        pref = GROUP_KERNELS[name]
        got = []
        while pos < len(launches) and any(launches[pos][0].replace("void ", "").replace("fdtd::", "").startswith(p) for p in pref) \
                and len(got) < (2 if name not in ("inv_h", "inject_h", "inject_e", "fwd_fused", "rev_fused", "grad", "adj_fused") else 1):
            got.append(launches[pos])
            pos += 1
        if not got:
            continue
        groups[name] = sum(g[1] + g[2] for g in got)
        detail[name] = [{"kernel": g[0][:60], "read": g[1], "write": g[2], "us": g[3]} for g in got]
    d = {}
    if os.path.exists(NCU_JSON):
        with open(NCU_JSON) as f:
            d = json.load(f)
    d[args.workload] = {"kernel_source_hash": kernel_source_hash(), "source": args.ncu_note or os.path.basename(args.ncu_import),
                        "groups": groups, "launches": detail}
    with open(NCU_JSON, "w") as f:
        json.dump(d, f, indent=1)
    print(json.dumps({"workload": args.workload, "groups": groups, "unmatched_launches": len(launches) - pos}))


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


def active_groups(fdtd, fused, fused_rev, fused_adj=False):
    """Names of the kernel groups that the run launches (fdtd.Sim.KERNEL_IDS), in profiling order.  fwd_e / fwd_h stay in the list
    on the fused forward path too (its first and last half-step, and the two-kernel-equivalent figure)."""
    names = ["fwd_e", "fwd_h"]
    names += ["rev_fused", "grad"] if fused_rev else ["inv_h", "grad_inv_e"]
    names += ["adj_fused", "adj_fused_slabs"] if fused_adj else ["adj_h", "adj_e"]
    names += ["record", "inject_h", "inject_e"]
    if fused:
        names += ["fwd_fused", "fwd_fused_slabs"]
    return names


def profile_kernels(sim, fdtd, w, flags, flush, reps, fused, fused_rev, fused_adj=False):
    """Each kernel group timed alone on the library's stream (fdtd_profile_kernel): {name: {us, algo_bytes}}.  Needs a completed
    forward run (record / inject and the z-face injection of the inverse kernels read the store)."""
    out = {}
    for name in active_groups(fdtd, fused, fused_rev, fused_adj):
        flush.fill_(1)
        ms, by = sim.profile_kernel(fdtd.Sim.KERNEL_IDS[name], warm=3 if reps > 1 else 0, reps=reps)
        out[name] = {"us": ms * 1e3, "algo_bytes": by}
    return out


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
    # --profile-only sizes the store for a short run: ncu saves and restores device memory around every replayed pass
    sim.set_workspace(min(w.nsteps, 64) if args.profile_only else w.nsteps, w.store_dtype, w.k, flags)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    extra = {}

    if args.profile_only:
        # one launch of every kernel group, in Sim.KERNELS order, for an `ncu --set full` capture (see --ncu-import)
        import dataclasses
        w = dataclasses.replace(w, nsteps=min(w.nsteps, 64))
        sim.forward(w.nsteps, w.sources, w.store_dtype, w.k, flags=flags)
        fused, fused_rev, fused_adj = sim.uses_fused(w.nsteps), sim.uses_fused_reverse(), sim.uses_fused_adjoint()
        torch.cuda.synchronize()
        torch.cuda.profiler.start()
        k = profile_kernels(sim, fdtd, w, flags, flush, 1, fused, fused_rev, fused_adj)
        torch.cuda.profiler.stop()
        print(json.dumps({"profile_only": True, "workload": args.workload, "kernels": k, "kernel_source_hash": kernel_source_hash()}))
        return

    def loss_cotangent_dev(mon):
        # harness-level objective on the small monitor tensor (SURVEY layer L4), on the device for the device-timed leg
        L, d = W.loss_and_cotangent(w, mon.cpu().numpy(), extra)
        return L, torch.from_numpy(d.astype(np.float32, copy=False)).to(dev)

    state = {"dmon": None, "L0": None, "grad": None}

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def one_step():
        flush.fill_(1)                                # L2 flush between steps (not timed)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        e[0].record()
        mon = sim.forward(w.nsteps, w.sources, w.store_dtype, w.k, flags=flags)
        e[1].record()
        if state["dmon"] is None:
            # first (warm-up) pass: fix the objective's constants (C3's target amplitude) and the loss cotangent once, so that
            # every later pass — all timed ones — contains only library work between the events
            if w.loss == "pulse_shape":
                A = np.asarray(w.extra["A"], dtype=np.float64).reshape(mon.shape[2:])
                extra.update(w.extra)
                extra["target_amp"] = 0.5 * float(np.max(np.abs(np.tensordot(mon[:, 0].cpu().numpy().astype(np.float64), A, axes=3))))
            state["L0"], state["dmon"] = loss_cotangent_dev(mon)
            e[1].record()
        grad = sim.reverse(None, state["dmon"], W.LINEAR)
        e[2].record()
        torch.cuda.synchronize()
        if state["grad"] is None:
            state["grad"] = grad.clone()
        return e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2])

    for _ in range(args.warmup):
        one_step()
    grad = state["grad"]
    assert torch.isfinite(grad).all().item(), "gradient is not finite"
    if not args.nsteps:
        assert grad.abs().max().item() > 0, "gradient is zero on the full-length workload"
    barrier()
    sampler = ClockSampler(local, args.clock_sample_ms) if rank == 0 else None
    l0 = sim.launch_count()
    t0 = time.time()
    tf, tr = [], []
    for _ in range(args.steps):
        a, b = one_step()
        tf.append(a)
        tr.append(b)
    barrier()
    t1 = time.time()
    launches = sim.launch_count() - l0
    clocks = sampler.stop(t0, t1) if sampler else None
    store_bytes = int(sim.store_bytes())
    nrec = sim.num_slots() - 1
    slot_vals = int(sim.slot_values())
    tot_ms = float(np.sum(tf) + np.sum(tr))
    tot_ms, f_ms, r_ms = reduce_max([tot_ms, float(np.sum(tf)), float(np.sum(tr))], world, dev)
    value = whole_job_value(w.cells, w.nsteps, args.steps, world, tot_ms)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    eps_host = torch.from_numpy(w.eps).pin_memory()
    mon_host = torch.empty(w.monitor_shape(), dtype=torch.float32).pin_memory()
    dmon_host = torch.empty(w.monitor_shape(), dtype=torch.float32).pin_memory()
    lo, hi = w.design
    grad_host = torch.empty([hi[a] - lo[a] for a in range(3)], dtype=torch.float32).pin_memory()
    state["dmon"] = None                                 # the device cotangent is not needed any more (7.9 GB on C4)

    def e2e_step():
        sim.set_eps_host(eps_host)
        sim.forward_host(w.nsteps, w.sources, w.store_dtype, w.k, mon_host)
        L, d = W.loss_and_cotangent(w, mon_host.numpy(), extra)
        dmon_host.copy_(torch.from_numpy(np.ascontiguousarray(d, dtype=np.float32)))
        sim.reverse_host(dmon_host, W.LINEAR, grad_host)
        return L
    # the device-timed passes above have warmed the GPU; a pass of the host-buffer path first only where it is cheap
    ne2e = max(1, min(args.steps, 3)) if tot_ms / args.steps < 5e3 else 1
    if tot_ms / args.steps < 5e3:
        e2e_step()
    barrier()
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

    # ---- per-kernel roofline (rank 0): each kernel group timed alone, back to back, CUDA events on its stream ----
    peak, peak_src = load_peaks()
    sim.forward(min(w.nsteps, 64), w.sources, w.store_dtype, w.k, flags=flags)
    fused = sim.uses_fused(w.nsteps)   # H half-step of step m and E half-step of step m+1 in one marching kernel
    fused_rev = sim.uses_fused_reverse()   # large grids: inverse-H and inverse-E of the reverse primal in one marching kernel
    fused_adj = sim.uses_fused_adjoint()   # large grids: adjoint of H and adjoint of E in one marching kernel
    counts = {"fwd_e": 1 if fused else w.nsteps, "fwd_h": 1 if fused else w.nsteps, "inv_h": w.nsteps, "adj_h": w.nsteps,
              "grad_inv_e": w.nsteps, "adj_e": w.nsteps, "record": nrec + 1, "inject_h": w.nsteps, "inject_e": w.nsteps,
              "fwd_fused": w.nsteps - 1, "fwd_fused_slabs": w.nsteps - 1, "rev_fused": w.nsteps, "grad": w.nsteps,
              "adj_fused": w.nsteps, "adj_fused_slabs": w.nsteps}
    kernels = profile_kernels(sim, fdtd, w, flags, flush, 20, fused, fused_rev, fused_adj)
    traffic, traffic_src = load_ncu_traffic(args.workload if not (args.store or args.k or args.tangential) else "-")
    tot = sum(v["us"] * counts[n] for n, v in kernels.items())
    for n, v in kernels.items():
        v["launches_per_step"] = counts[n]
        v["share"] = v["us"] * counts[n] / tot
        # algorithmic bytes (SURVEY 8(d) / DESIGN.md "Roofline") over the measured time: an EFFECTIVE bandwidth
        v["effective_gbs"] = v["algo_bytes"] / (v["us"] * 1e-6) / 1e9
        v["frac"] = v["effective_gbs"] / peak
        # DRAM bytes of the same launch from the ncu capture of this build over the same measured time
        v["dram_bytes"] = traffic.get(n)
        v["dram_gbs"] = traffic[n] / (v["us"] * 1e-6) / 1e9 if n in traffic else None
        v["dram_frac"] = v["dram_gbs"] / peak if n in traffic else None
    dom = max(kernels, key=lambda n: kernels[n]["share"])
    kd = kernels[dom]
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kd["effective_gbs"], "peak": peak, "unit": "GB/s",
                "frac": kd["frac"], "traffic": kd["dram_bytes"], "peak_source": peak_src,
                "traffic_source": ("dram__bytes_read.sum + dram__bytes_write.sum per launch (all kernels of the group), ncu --set full, "
                                   + str(traffic_src)) if kd["dram_bytes"] is not None else f"null: {traffic_src}",
                "dram_frac": kd["dram_frac"],
                "how": "dominant kernel group (largest share of the step) timed alone, its kernels side by side as in the step: 20 "
                       "back-to-back launches between CUDA events on the library's stream after 3 warm-up launches, L2 flushed before "
                       "the series; achieved = ALGORITHMIC bytes per launch (DESIGN.md Roofline; SURVEY 8(d)) / mean launch time; "
                       "dram_frac = ncu DRAM bytes of the same launch / the same time / peak",
                "launch_us": kd["us"], "algo_bytes": kd["algo_bytes"]}
    if dom == "adj_e":
        # SURVEY 8(d)'s table counts the adjoint of the E half-step at 36 B per cell; the kernel also reads ce (S/eps): 40 B
        survey = kd["algo_bytes"] - 4.0 * w.cells
        roofline["survey_bytes"] = survey
        roofline["frac_survey_bytes"] = survey / (kd["us"] * 1e-6) / 1e9 / peak
    # whole-pass effective bandwidth: algorithmic bytes of all stencil launches of one step / measured time
    fwd_names = ("fwd_e", "fwd_h", "fwd_fused", "fwd_fused_slabs")
    algo_fwd = sum(kernels[n]["algo_bytes"] * counts[n] for n in fwd_names if n in kernels) + kernels["record"]["algo_bytes"] * (nrec + 1)
    rev_names = ("rev_fused", "grad", "inv_h", "grad_inv_e", "adj_h", "adj_e", "adj_fused", "adj_fused_slabs", "inject_h", "inject_e")
    algo_rev = sum(kernels[n]["algo_bytes"] for n in rev_names if n in kernels) * w.nsteps
    fwd_gbs = algo_fwd / (f_ms / args.steps * 1e-3) / 1e9
    # the same forward time against the bytes of the two-kernel form (76 B per cell): comparable across paths
    algo_fwd2 = (kernels["fwd_e"]["algo_bytes"] + kernels["fwd_h"]["algo_bytes"]) * w.nsteps + kernels["record"]["algo_bytes"] * (nrec + 1)
    fwd2_gbs = algo_fwd2 / (f_ms / args.steps * 1e-3) / 1e9
    rev_gbs = algo_rev / (r_ms / args.steps * 1e-3) / 1e9

    # ---- CPU baseline: the oracle as it stands on a bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if world == 1 and not args.no_cpu and not args.tangential:
        del sim, flush
        torch.cuda.empty_cache()
        cpu = cpu_baseline(args.workload, args.cpu_steps)

    ws_mb = 13 * w.cells * 4 / 1e6
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": tot_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{w.name}: {w.shape[0]}x{w.shape[1]}x{w.shape[2]} f32 Yee grid, {w.pml}-cell CPML, {w.nsteps} steps, "
                               f"{W.DTYPE_NAMES[w.store_dtype]} store, k={w.k}, linear interpolation, loss={w.loss}",
                   "grid": list(w.shape), "pml": w.pml, "nsteps": w.nsteps, "store_dtype": W.DTYPE_NAMES[w.store_dtype], "k": w.k,
                   "store_components": "tangential (12 slices per slot)" if args.tangential else "all six per face (36 slices per slot)",
                   "l2": (f"inputs larger than L2: every time step streams its working set ({ws_mb:.0f} MB of fields in the reverse run, "
                          f"{7 * w.cells * 4 / 1e6:.0f} MB forward) from HBM; a 256 MB write also flushes L2 between timed steps")
                         if 7 * w.cells * 4 > 1.5 * 126e6 else
                         (f"256 MB write between timed steps flushes L2; inside a step the working set ({ws_mb:.0f} MB of fields) is of "
                          "the order of the 126 MB L2, so per-kernel fractions are effective bandwidths, not DRAM traffic"),
                   "replicas": world, "parallelism": "replicas only (the path runs on one GPU)"},
        "forward_mcells_per_s": whole_job_value(w.cells, w.nsteps, args.steps, world, f_ms),
        "reverse_mcells_per_s": whole_job_value(w.cells, w.nsteps, args.steps, world, r_ms),
        "forward_ms": f_ms / args.steps, "reverse_ms": r_ms / args.steps,
        "store_bytes": store_bytes, "store_bytes_per_step": store_bytes / w.nsteps,
        "store_bytes_f32_k1": (w.nsteps + 1) * slot_vals * (3 if args.tangential else 1) * 4,   # all six components
        "effective_gbs": {"forward": fwd_gbs, "reverse": rev_gbs, "forward_frac_of_peak": fwd_gbs / peak,
                          "reverse_frac_of_peak": rev_gbs / peak, "forward_fused": bool(fused), "reverse_fused": bool(fused_rev), "adjoint_fused": bool(fused_adj),
                          "forward_two_kernel_equivalent": fwd2_gbs, "forward_two_kernel_equivalent_frac": fwd2_gbs / peak,
                          # also against the nominal HBM3e figure (8000 GB/s)
                          "forward_frac_of_nominal_8000": fwd_gbs / 8000.0, "reverse_frac_of_nominal_8000": rev_gbs / 8000.0,
                          "note": "algorithmic bytes (SURVEY 8(d)) / measured time: effective bandwidths, not DRAM counters"},
        "roofline": roofline, "kernels": kernels, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "loss": state["L0"], "grad_abs_max": float(grad.abs().max().item()),
    }
    if cpu is not None:
        out["cpu_baseline"] = cpu
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


class OracleRunner:
    """The CPU oracle (f32), as it stands, on the first `nsteps` time steps of workload w.  Built once (its arrays are
    allocated at construction); every pass resets it to state 0 and runs forward + reverse."""

    def __init__(self, w, nsteps):
        import dataclasses
        from oracle import fdtd_oracle as orc
        self.orc = orc
        srcs = [dataclasses.replace(s, wave=s.wave[:nsteps]) for s in w.sources]
        self.ws = dataclasses.replace(w, nsteps=nsteps, sources=srcs)
        self.s = orc.OracleSim(32, self.ws.eps, self.ws.pml, W.S)
        self.s.set_design(*self.ws.design)
        self.s.set_monitor(*self.ws.monitor)
        for q in srcs:
            self.s.add_source(q.comp, q.lo, q.hi, q.amp, q.wave)

    def one_pass(self):
        """(forward seconds, reverse seconds, threads)"""
        ws, s = self.ws, self.s
        s.reset()
        t0 = time.perf_counter()
        s.forward(ws.nsteps, ws.store_dtype, ws.k)
        tf = time.perf_counter() - t0
        ex = dict(ws.extra)
        ex["target_amp"] = 1.0
        L, d = W.loss_and_cotangent(ws, s.monitor_record(), ex)
        t1 = time.perf_counter()
        s.reverse(None, d, self.orc.LINEAR)
        tr = time.perf_counter() - t1
        return tf, tr, self.orc.get_threads()


def sample_description(w, nsteps, per_step=False):
    first = min(getattr(s.wave, "size", 0) and int(np.argmax(np.abs(s.wave) > 1e-3 * np.abs(s.wave).max())) for s in w.sources) + 1
    quiet = (f"; the source is still below 1e-3 of its peak until step {first}, so the sampled steps run on (near-)zero fields"
             if first > nsteps else "")
    return (f"{w.name} grid, first {nsteps} of {w.nsteps} time steps" + (" per bench step" if per_step else "") +
            f", forward + reverse, float32 oracle, {W.DTYPE_NAMES[w.store_dtype]} k={w.k}{quiet}")


def default_sample_steps(w, seconds):
    """Time steps of the workload that the oracle gets through in about `seconds` (its measured ~40 Mcell-updates/s forward +
    reverse on 16 cores), at least 2 (one stored slot interval needs two states), at most 60."""
    return int(max(2, min(60, seconds * 40e6 / w.cells)))


def cpu_baseline(workload, nsteps):
    w = make_workload(workload, None)
    nsteps = min(nsteps or default_sample_steps(w, 15.0), w.nsteps)
    tf, tr, cores = OracleRunner(w, nsteps).one_pass()
    cu = float(w.cells) * nsteps
    return {"value": cu / (tf + tr) / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": sample_description(w, nsteps),
            "forward_mcells_per_s": cu / tf / 1e6, "reverse_mcells_per_s": cu / tr / 1e6, "seconds": tf + tr}


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores; each step = a bounded sample of the workload."""
    if rank != 0:
        return
    w = make_workload(args.workload, None)
    sample = min(args.ref_steps or default_sample_steps(w, 6.0), w.nsteps)
    runner = OracleRunner(w, sample)
    for _ in range(args.warmup):
        runner.one_pass()
    t = 0.0
    cores = 0
    for _ in range(args.steps):
        tf, tr, cores = runner.one_pass()
        t += tf + tr
    value = float(w.cells) * sample * args.steps / t / 1e6
    desc = sample_description(w, sample, per_step=True)
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
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4"],
                    help="C4 (512^3, 10 000 steps, bf16 k=4: the largest single-GPU configuration, HBM-bound) is the default")
    ap.add_argument("--nsteps", type=int, default=0, help="override the workload's number of time steps")
    ap.add_argument("--cpu-steps", type=int, default=0, help="time steps of the cpu_baseline sample (0: about 15 s of oracle work)")
    ap.add_argument("--ref-steps", type=int, default=0, help="time steps per bench step of --impl reference (0: about 6 s of oracle work)")
    ap.add_argument("--profile-only", action="store_true", help="launch every kernel group once (for an ncu --set full capture) and exit")
    ap.add_argument("--ncu-import", default="", help="raw-page CSV of such a capture: store its DRAM bytes in profiles/ncu_traffic.json")
    ap.add_argument("--ncu-note", default="", help="provenance string stored with --ncu-import")
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
    if args.ncu_import:
        ncu_import(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_gpu(args, rank, world)


if __name__ == "__main__":
    main()
