"""Shared test helpers: drive the oracle on a workloads.Workload."""
import numpy as np

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import workloads as W


def make_oracle(w, prec, cpml=orc.CPML_DEFAULTS, with_sources=True):
    s = orc.OracleSim(prec, w.eps, w.pml, W.S, cpml)
    s.set_design(*w.design)
    s.set_monitor(*w.monitor)
    if with_sources:
        for q in w.sources:
            s.add_source(q.comp, q.lo, q.hi, q.amp, q.wave)
    return s


def oracle_gradient(w, prec, dtype, k, interp=orc.LINEAR, mode=orc.METHOD, eps=None, extra=None):
    """forward -> loss -> reverse.  Returns dict(L, grad, final, state0, mon, sim)."""
    if eps is not None:
        import dataclasses
        w = dataclasses.replace(w, eps=np.asarray(eps))
    s = make_oracle(w, prec)
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
