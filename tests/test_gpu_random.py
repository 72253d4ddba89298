"""Random small grids, CUDA path against the float32 oracle (`-m gpu`).

The hand-built parity cases of test_gpu_parity.py pick their shapes; these draw them: CPML width 1..10, any extents (so the scalar
V = 1 / 2 kernels and the float4 ones, rows of a single group, one to three z tiles), run length, subsampling k, every store
dtype, both interpolations, store mode, 1-3 random sources with or without amplitude arrays (overlapping ones included), random
design / monitor / cotangent boxes and component masks, graphs on / off, marching kernels automatic / off / forced, row kernels
automatic / off / on.  Every case runs in a guarded workspace (0xFF fill, guard bands: DESIGN.md section 3).  Checked per case: final fields, monitor record and every stored slot bit for bit; loss; gradient within
north_star's 1e-4.  1 200 such cases were run once (two defects found and fixed: unordered sums of overlapping sources, marching
kernels forced onto a single-group interior; both have tests of their own in test_gpu_parity.py); 50 seeded cases stay.
"""
import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import workloads as W
from paper_2603_24027_b200.fdtd import WS_GUARD, WS_REVERSE
from tests.helpers import gpu_gradient, gpu_sim, make_oracle, oracle_gradient, rel_l2

pytestmark = pytest.mark.gpu

DTYPES = [W.F32, W.F16, W.BF16, W.F8E4M3_SCALED, W.F8E4M3_MX32, W.F8E4M3B11FNUZ, W.F8E5M2FNUZ, W.F8E4M3FNUZ, W.F8E4M3, W.F8E3M4]
GRAD_TOL = 1e-4


def _draw(rng, tall_prob=0.25):
    P = int(rng.integers(1, 11))
    if rng.random() < 0.3:
        P = int(rng.choice([4, 8]))                     # widths the marching kernels accept
    dims = [int(rng.integers(2 * P + 3, 2 * P + 3 + 30)) for _ in range(3)]
    if rng.random() < 0.55:
        dims[2] = 4 * ((dims[2] + 3) // 4)              # float4 kernels
    if rng.random() < tall_prob and P <= 8:             # rows that cross a 128-cell tile boundary
        dims[2] = int(rng.choice([128, 132, 136, 140, 256, 260]))
        dims[0], dims[1] = min(dims[0], 2 * P + 12), min(dims[1], 2 * P + 14)
    shape = tuple(dims)
    T = int(rng.integers(2, 45))
    cfg = dict(P=P, shape=shape, T=T, k=int(rng.choice([1, 2, 3, 4, 5, 8, 16])), dtype=int(rng.choice(DTYPES)),
               interp=int(rng.choice([W.LINEAR, W.CUBIC])), eps=rng.uniform(1.0, 12.25, shape).astype(np.float32),
               wave=W.gauss_sine(T, max(2, T // 3), max(1, T // 8)))

    def box(minw, maxw, margin=P):
        lo, hi = [], []
        for a in range(3):
            width = int(rng.integers(minw, min(maxw, shape[a] - 2 * margin) + 1))
            lo.append(int(rng.integers(margin, shape[a] - margin - width + 1)))
            hi.append(lo[-1] + width)
        return tuple(lo), tuple(hi)
    cfg["box"] = box
    srcs = []
    for _ in range(int(rng.integers(1, 4))):
        lo, hi = box(1, 5)
        amp = rng.uniform(0.5, 1.5, tuple(hi[a] - lo[a] for a in range(3))).astype(np.float32) if rng.random() < 0.5 else None
        srcs.append(W.Source(int(rng.integers(0, 3)), lo, hi, amp, cfg["wave"]))
    cfg["srcs"] = srcs
    return cfg


def _knobs(rng):
    return bool(rng.integers(0, 2)), int(rng.choice([-1, -1, 0, 1])), int(rng.choice([-1, 0, 1]))


@pytest.mark.parametrize("seed", range(30000, 30030))
def test_random_grid_flux_loss_against_oracle(seed):
    """Flux loss on an x plane behind the first source, design box around that source (all-components or tangential store)."""
    rng = np.random.default_rng(seed)
    c = _draw(rng)
    P, shape, srcs = c["P"], c["shape"], c["srcs"]
    store_mode = int(rng.choice([0, 0, orc.STORE_TANGENTIAL]))
    dlo, dhi = c["box"](1, 30)
    q = P + 1 if store_mode else P                       # tangential store: the design box stays on the inner interior
    dlo = tuple(max(q, min(dlo[a], srcs[0].lo[a] - 1)) for a in range(3))
    dhi = tuple(min(shape[a] - q, max(dhi[a], srcs[0].hi[a] + 1)) for a in range(3))
    if any(dhi[a] <= dlo[a] for a in range(3)):
        pytest.skip("no room for a design box on the inner interior")
    mx = min(shape[0] - P - 1, srcs[0].hi[0] + 1)
    mon = ((mx, P, P), (mx + 1, shape[1] - P, shape[2] - P), 0b110110)
    w = W.Workload(f"random{seed}", shape, P, c["T"], c["eps"], (dlo, dhi), srcs, mon, "flux_x", c["dtype"], c["k"])
    graphs, fused, rows = _knobs(rng)
    tag = f"{shape} P {P} T {w.nsteps} k {w.k} dtype {w.store_dtype} interp {c['interp']} mode {store_mode} graphs {graphs} fused {fused} rows {rows}"
    o = oracle_gradient(w, 32, w.store_dtype, w.k, c["interp"], store_mode=store_mode)
    s = gpu_sim(w, store_mode=store_mode, rows=rows)
    s.set_graphs(graphs)
    s.set_fused(fused, 0)
    s.set_workspace(w.nsteps, w.store_dtype, w.k, WS_REVERSE | WS_GUARD)    # 0xFF-filled, a guard band behind every sub-array
    g = gpu_gradient(w, w.store_dtype, w.k, interp=c["interp"], sim=s)
    assert s.guard_check() == 0, tag
    assert np.array_equal(g["final"], o["final"]), tag
    assert np.array_equal(g["mon"], o["mon"]), tag
    assert abs(g["L"] - o["L"]) <= 1e-6 * abs(o["L"]), tag
    if np.linalg.norm(o["grad"]) > 1e-30:                # below that the float32 output has underflowed to zero
        assert rel_l2(g["grad"], o["grad"]) <= GRAD_TOL, tag
    inner = (slice(None),) + tuple(slice(q, n - q) for n in shape)
    peak = max(np.abs(o["final"]).max(), 1e-30)
    assert np.abs(g["state0"][inner] - o["state0"][inner]).max() <= 1e-4 * peak, tag
    assert s.store_bytes() == o["sim"].store_bytes(), tag
    s.forward(w.nsteps, srcs, w.store_dtype, w.k)
    of = o["sim"]
    of.reset()
    of.forward(w.nsteps, w.store_dtype, w.k)
    assert s.num_slots() == of.num_slots()
    for j in range(of.num_slots()):
        data, scales = s.slot(j, w.store_dtype)
        od, osc = of.slot(j, w.store_dtype)
        assert np.array_equal(data.cpu().numpy(), od), (tag, j)
        if w.store_dtype == W.F8E4M3_SCALED and store_mode == 0:
            assert np.array_equal(scales.cpu().numpy(), osc), (tag, j)


@pytest.mark.parametrize("seed", range(40000, 40020))
def test_random_cotangents_against_oracle(seed):
    """Random monitor box and component mask with random per-step cotangents, and / or a random cotangent box on the final state
    (which may reach into the CPML), random design box: the gradient is linear in the cotangents, so no loss function is needed."""
    import torch
    rng = np.random.default_rng(seed)
    c = _draw(rng)
    P, shape, srcs, T = c["P"], c["shape"], c["srcs"], c["T"]
    design = c["box"](1, 30)
    mlo, mhi = c["box"](1, 12)
    mmask = int(rng.integers(1, 64))
    w = W.Workload(f"cot{seed}", shape, P, T, c["eps"], design, srcs, (mlo, mhi, mmask), "flux_x", c["dtype"], c["k"])
    graphs, fused, rows = _knobs(rng)
    use_final = rng.random() < 0.6
    use_mon = rng.random() < 0.7 or not use_final
    o = make_oracle(w, 32)
    o.forward(T, w.store_dtype, w.k)
    omon, ofinal = o.monitor_record(), o.fields()
    dmon = (rng.standard_normal(omon.shape) * rng.choice([1.0, 1e-3, 30.0])).astype(np.float32) if use_mon else None
    dfinal = cot = None
    if use_final:
        clo, chi = c["box"](1, 14, margin=1) if rng.random() < 0.3 else c["box"](1, 14)
        cmask = int(rng.integers(1, 64))
        comps = [q for q in range(6) if cmask >> q & 1]
        gbox = rng.standard_normal((len(comps),) + tuple(chi[a] - clo[a] for a in range(3))).astype(np.float32)
        dfinal = np.zeros((6,) + shape)
        for ci, q in enumerate(comps):
            dfinal[q, clo[0]:chi[0], clo[1]:chi[1], clo[2]:chi[2]] = gbox[ci]
        cot = (clo, chi, cmask, torch.from_numpy(gbox).cuda())
    og = o.reverse(dfinal, None if dmon is None else dmon.astype(np.float64), c["interp"])
    s = gpu_sim(w, rows=rows)
    s.set_graphs(graphs)
    s.set_fused(fused, 0)
    s.set_workspace(T, w.store_dtype, w.k, WS_REVERSE | WS_GUARD)
    gmon = s.forward(T, srcs, w.store_dtype, w.k).cpu().numpy()
    tag = f"{shape} P {P} T {T} k {w.k} dtype {w.store_dtype} interp {c['interp']} mon {mlo}-{mhi} mask {mmask:06b} final {use_final} dmon {use_mon} graphs {graphs} fused {fused} rows {rows}"
    assert np.array_equal(s.fields().cpu().numpy().astype(np.float64), ofinal), tag
    assert np.array_equal(gmon.astype(np.float64), omon), tag
    gg = s.reverse(cot, None if dmon is None else torch.from_numpy(dmon).cuda(), c["interp"]).cpu().numpy().astype(np.float64)
    assert s.guard_check() == 0, tag
    if np.linalg.norm(og) > 1e-30:
        assert rel_l2(gg, og) <= GRAD_TOL, tag
    else:
        assert np.abs(gg).max() <= 1e-30, tag
