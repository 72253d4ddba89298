"""Shared test helpers: drive the oracle on a workloads.Workload."""
import numpy as np

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import workloads as W


def make_oracle(w, prec, cpml=orc.CPML_DEFAULTS, with_sources=True, store_mode=0):
    s = orc.OracleSim(prec, w.eps, w.pml, W.S, cpml)
    if store_mode:
        s.set_store_mode(store_mode)
    s.set_design(*w.design)
    s.set_monitor(*w.monitor)
    if with_sources:
        for q in w.sources:
            s.add_source(q.comp, q.lo, q.hi, q.amp, q.wave)
    return s


def oracle_gradient(w, prec, dtype, k, interp=orc.LINEAR, mode=orc.METHOD, eps=None, extra=None, store_mode=0):
    """forward -> loss -> reverse.  Returns dict(L, grad, final, state0, mon, sim)."""
    if eps is not None:
        import dataclasses
        w = dataclasses.replace(w, eps=np.asarray(eps))
    s = make_oracle(w, prec, store_mode=store_mode)
    if mode == orc.STORE_ALL:
        s.set_keep_all(True)
    s.forward(w.nsteps, dtype, k)
    mon = s.monitor_record()
    final = s.fields()
    L, d = W.loss_and_cotangent(w, mon, extra)
    g = s.reverse(None, d, interp, mode)
    return dict(L=L, grad=g, final=final, state0=s.fields(), mon=mon, sim=s, dmon=d)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


# ---- CUDA path (imported lazily so that CPU-only test runs never touch torch.cuda) ----
def gpu_sim(w, cpml=None, store_mode=0, rows=-1):
    import torch
    from paper_2603_24027_b200 import fdtd
    eps = torch.from_numpy(np.ascontiguousarray(w.eps, dtype=np.float32)).cuda()
    return fdtd.Sim(eps, W.DX, W.DT, w.pml, design=w.design, monitor=w.monitor, cpml=cpml, store_mode=store_mode, rows=rows)


def gpu_gradient(w, dtype, k, interp=0, extra=None, sim=None):
    """forward -> loss (harness, numpy on the monitor record) -> reverse, all through the C ABI."""
    import torch
    s = sim or gpu_sim(w)
    mon = s.forward(w.nsteps, w.sources, dtype, k)
    final = s.fields().cpu().numpy().astype(np.float64)
    mon_np = mon.cpu().numpy().astype(np.float64)
    L, d = W.loss_and_cotangent(w, mon_np, extra)
    dmon = torch.from_numpy(d.astype(np.float32)).cuda()
    g = s.reverse(None, dmon, interp)
    state0 = s.fields().cpu().numpy().astype(np.float64)
    return dict(L=L, grad=g.cpu().numpy().astype(np.float64), final=final, state0=state0, mon=mon_np, sim=s, dmon=d)
