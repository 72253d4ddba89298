"""Seeded synthetic workloads shaped like the paper's nanophotonic inverse-design problems.

This module serves BOTH the CPU oracle's tests and the CUDA path (tests, bench.py): it holds the input
generators (permittivity maps, sources, monitor/design boxes) and the objective functions that turn
recorded monitor values into a scalar loss and its cotangent.  It holds NONE of the method's arithmetic
(no field update, no codec, no interpolation) and imports neither oracle/ nor the CUDA binding.

The paper's own workload (Si grating coupler in FDTDX) is not reproducible here; these
inputs take its shapes — Si (12.25) / SiO2 (2.085) permittivities, 20 nm cells, a 220 nm = 11-cell
device layer, a 1550 nm carrier (~136 steps per period), PML on all faces, flux /
energy / pulse-shape objectives — and stand in for it.  Recipes: DESIGN.md "Input recipe", following
BASELINE.json `configs` C1..C4.

Field component indices: 0..2 = Ex,Ey,Ez ; 3..5 = Hx,Hy,Hz.  Boxes are half-open [lo, hi).
"""
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

C0 = 299792458.0
DX = 20e-9
COURANT_FACTOR = 0.99
DT = COURANT_FACTOR * DX / (C0 * np.sqrt(3.0))        # PAPER.md:39 eq. (1)  -> 3.81e-17 s
S = C0 * DT / DX                              # Courant number 0.99/sqrt(3)
WAVELENGTH = 1550e-9
OMEGA_DT = 2.0 * np.pi * C0 * DT / WAVELENGTH  # rad per step; 2*pi/135.59 ("approximately 136")
EPS_SI, EPS_SIO2 = 12.25, 2.085

# store dtypes / interpolation (the ids of include/fdtd.h)
F32, F16, BF16, F8E4M3_SCALED = 0, 1, 2, 3
F8E4M3_MX32 = 5    # micro-scaled E4M3: a power-of-two scale byte per block of 32 values (R20)
F8E4M3B11FNUZ, F8E5M2FNUZ, F8E4M3FNUZ, F8E4M3, F8E3M4 = 10, 11, 12, 13, 14   # the paper's unscaled flavours
PAPER_FP8 = (F8E4M3B11FNUZ, F8E5M2FNUZ, F8E4M3FNUZ, F8E4M3, F8E3M4)
LINEAR, CUBIC = 0, 1
DTYPE_NAMES = {F32: "float32", F16: "float16", BF16: "bfloat16", F8E4M3_SCALED: "float8_e4m3+scale",
               F8E4M3_MX32: "float8_e4m3+mx32",
               F8E4M3B11FNUZ: "float8_e4m3b11fnuz", F8E5M2FNUZ: "float8_e5m2fnuz", F8E4M3FNUZ: "float8_e4m3fnuz",
               F8E4M3: "float8_e4m3", F8E3M4: "float8_e3m4"}
DTYPE_BITS = {F32: 32, F16: 16, BF16: 16, F8E4M3_SCALED: 8, F8E4M3_MX32: 8, **{d: 8 for d in PAPER_FP8}}


@dataclass
class Source:
    comp: int
    lo: Tuple[int, int, int]
    hi: Tuple[int, int, int]
    amp: Optional[np.ndarray]          # float32 [hi-lo] or None (= 1)
    wave: np.ndarray                   # float32 [nsteps]; wave[m-1] is added in step m


@dataclass
class Workload:
    name: str
    shape: Tuple[int, int, int]
    pml: int
    nsteps: int
    eps: np.ndarray                    # float32 [nx,ny,nz]
    design: Tuple[Tuple[int, int, int], Tuple[int, int, int]]
    sources: List[Source]
    monitor: Tuple[Tuple[int, int, int], Tuple[int, int, int], int]   # lo, hi, comp_mask
    loss: str                          # "final_E2" | "flux_x" | "pulse_shape"
    store_dtype: int
    k: int
    extra: dict = field(default_factory=dict)

    @property
    def cells(self):
        return int(np.prod(self.shape))

    def monitor_shape(self):
        lo, hi, mask = self.monitor
        return (self.nsteps, bin(mask).count("1")) + tuple(hi[a] - lo[a] for a in range(3))


def gauss_sine(nsteps, n0, tau):
    """wave[m-1] = exp(-((m-n0)/tau)^2/2) * sin(OMEGA_DT*(m-n0)), m = 1..nsteps."""
    m = np.arange(1, nsteps + 1, dtype=np.float64)
    return (np.exp(-0.5 * ((m - n0) / tau) ** 2) * np.sin(OMEGA_DT * (m - n0))).astype(np.float32)


def ramped_cw(nsteps, ramp):
    m = np.arange(1, nsteps + 1, dtype=np.float64)
    return ((1.0 - np.exp(-(m / ramp) ** 2)) * np.sin(OMEGA_DT * m)).astype(np.float32)


def c1(nsteps=200, seed=1001):
    """BASELINE.json configs[0]: 32^3, 8-cell CPML, Ez dipole, 16^3 design region = the whole interior."""
    n, P = 32, 8
    eps = np.ones((n, n, n), dtype=np.float32)
    eps[8:24, 8:24, 8:24] = np.random.default_rng(seed).uniform(EPS_SIO2, EPS_SI, (16, 16, 16)).astype(np.float32)
    src = Source(2, (16, 16, 16), (17, 17, 17), None, gauss_sine(nsteps, 60, 20))
    return Workload("C1", (n, n, n), P, nsteps, eps, ((8, 8, 8), (24, 24, 24)), [src],
                    ((22, 8, 8), (23, 24, 24), 0b000111), "final_E2", F32, 1)


def c2(nsteps=2000, seed=1002, n=128, P=12):
    """BASELINE.json configs[1]: 128^3, 12-cell CPML, Si slab in SiO2, 64x64 design patch, line source, flux loss."""
    assert n == 128
    eps = np.full((n, n, n), EPS_SIO2, dtype=np.float32)
    eps[:, :, 58:69] = EPS_SI
    eps[32:96, 32:96, 58:69] = np.random.default_rng(seed).uniform(EPS_SIO2, EPS_SI, (64, 64, 11)).astype(np.float32)
    i = np.arange(24, 104, dtype=np.float64)
    amp = np.exp(-((i - 64.0) / 16.0) ** 2).astype(np.float32).reshape(80, 1, 1)
    n0, tau = (400, 120) if nsteps >= 800 else (nsteps // 3, max(nsteps // 10, 4))
    src = Source(1, (24, 64, 96), (104, 65, 97), amp, gauss_sine(nsteps, n0, tau))
    return Workload("C2", (n, n, n), P, nsteps, eps, ((32, 32, 58), (96, 96, 69)), [src],
                    ((104, 44, 52), (105, 84, 76), 0b110110), "flux_x", BF16, 4)


def c3(nsteps=5000, seed=1003):
    """BASELINE.json configs[2]: 256x256x128, 16-cell CPML, Si strip waveguide, binary-plus-noise design, pulse-shape loss."""
    shape, P = (256, 256, 128), 16
    eps = np.full(shape, EPS_SIO2, dtype=np.float32)
    eps[:, 116:141, 58:69] = EPS_SI
    rng = np.random.default_rng(seed)
    b = rng.integers(0, 2, (32, 32)).astype(np.float64)
    b = np.kron(b, np.ones((4, 4)))
    rho = np.clip(b + 0.1 * rng.standard_normal((128, 128)), 0.0, 1.0)
    eps[64:192, 64:192, 58:69] = (EPS_SIO2 + rho * (EPS_SI - EPS_SIO2)).astype(np.float32)[:, :, None]
    j = np.arange(108, 149, dtype=np.float64).reshape(-1, 1)
    kk = np.arange(54, 73, dtype=np.float64).reshape(1, -1)
    A = np.exp(-((j - 128.0) / 8.0) ** 2 - ((kk - 63.0) / 4.0) ** 2).astype(np.float32)
    full = nsteps >= 3000
    n0, tau = (1100, 272) if full else (nsteps // 4, max(nsteps // 12, 4))
    src = Source(1, (24, 108, 54), (25, 149, 73), A.reshape(1, 41, 19), gauss_sine(nsteps, n0, tau))
    tgt_n0, tgt_tau = (2600, 400) if full else (int(0.6 * nsteps), max(nsteps // 8, 4))
    return Workload("C3", shape, P, nsteps, eps, ((64, 64, 58), (192, 192, 69)), [src],
                    ((232, 108, 54), (233, 149, 73), 0b000010), "pulse_shape", F16, 8,
                    {"A": A, "target_n0": tgt_n0, "target_tau": tgt_tau})


def c4(nsteps=10000, seed=1004, n=512):
    """BASELINE.json configs[3]: 512^3, 16-cell CPML, random multi-slab eps, 256^3 design, 8x8 dipole array."""
    P = 16
    rng = np.random.default_rng(seed)
    eps = np.empty((n, n, n), dtype=np.float32)
    z = 0
    while z < n:
        t = int(rng.integers(8, 65))
        eps[:, :, z:z + t] = np.float32(rng.uniform(1.0, EPS_SI))
        z += t
    q = n // 4
    eps[q:3 * q, q:3 * q, q:3 * q] = rng.uniform(1.0, EPS_SI, (2 * q, 2 * q, 2 * q)).astype(np.float32)
    signs = rng.choice([-1.0, 1.0], size=(8, 8)).astype(np.float32)
    wave = ramped_cw(nsteps, 500.0 if nsteps >= 2000 else max(nsteps / 4.0, 2.0))
    step = (n - 2 * (n // 8)) // 8                       # 48 at n = 512
    srcs = []
    for a in range(8):
        for b in range(8):
            i, j, kz = n // 8 + step * a, n // 8 + step * b, (n * 48) // 512
            kz = max(kz, P + 1)
            srcs.append(Source(2, (i, j, kz), (i + 1, j + 1, kz + 1), np.full((1, 1, 1), signs[a, b], np.float32), wave))
    kmon = (n * 448) // 512
    return Workload("C4", (n, n, n), P, nsteps, eps, ((q, q, q), (3 * q, 3 * q, 3 * q)), srcs,
                    ((q, q, kmon), (3 * q, 3 * q, kmon + 1), 0b000111), "final_E2", BF16, 4)


def tiny(shape=(14, 13, 12), P=3, nsteps=24, seed=7, store_dtype=F32, k=1):
    """A tiny mixed workload for finite-difference and store-all checks: design box touches inner cells,
    face-, edge- and corner-shell cells; two sources; a monitor on E and H; loss = final + per-step terms."""
    rng = np.random.default_rng(seed)
    eps = rng.uniform(1.0, 4.0, shape).astype(np.float32)
    lo = (P, P, P)
    hi = (P + 4, P + 3, shape[2] - P)
    c = tuple(s // 2 for s in shape)
    w1 = (np.sin(0.5 * np.arange(1, nsteps + 1)) * np.exp(-0.5 * ((np.arange(1, nsteps + 1) - 8) / 4.0) ** 2)).astype(np.float32)
    w2 = (0.5 * np.cos(0.4 * np.arange(1, nsteps + 1))).astype(np.float32)
    srcs = [Source(2, c, tuple(x + 1 for x in c), None, w1),
            Source(0, (P, P + 1, P + 1), (P + 2, P + 3, P + 2), rng.uniform(0.5, 1.5, (2, 2, 1)).astype(np.float32), w2)]
    mon = ((shape[0] - P - 2, P, P), (shape[0] - P - 1, shape[1] - P, shape[2] - P), 0b110110)
    return Workload("tiny", tuple(shape), P, nsteps, eps, (lo, hi), srcs, mon, "flux_x", store_dtype, k)


BY_NAME = {"C1": c1, "C2": c2, "C3": c3, "C4": c4, "tiny": tiny}


# ----------------------------------------------------------------------------------------------------
# Objectives (harness level: SURVEY.md layer L4; PAPER.md:45,51 measure Poynting flux through detectors).
# Each returns (L, dmon) with dmon = dL/d(monitor record), same shape as the record, float64.
# E and H are taken as stored (co-indexed, half a step apart): synthetic objectives (R19).
# ----------------------------------------------------------------------------------------------------
def loss_and_cotangent(w: Workload, mon: np.ndarray, extra: Optional[dict] = None):
    mon = np.asarray(mon)
    # float32 records (the CUDA path's own output) keep their type where the cotangent is a copy / sign flip / doubling of
    # the record (exact in float32): no 8-byte copy of a 30 MB record on the host.  Sums are accumulated in float64.
    if not (mon.dtype == np.float32 and w.loss in ("final_E2", "flux_x")):
        mon = mon.astype(np.float64, copy=False)
    assert mon.shape == w.monitor_shape(), (mon.shape, w.monitor_shape())
    d = np.empty_like(mon) if w.loss == "flux_x" else np.zeros_like(mon)   # flux_x fills every component
    if w.loss == "final_E2":                       # L = sum_c sum_plane E_c(T)^2
        L = float(np.sum(mon[-1].astype(np.float64) ** 2))
        d[-1] = 2.0 * mon[-1]
    elif w.loss == "flux_x":                       # mask Ey,Ez,Hy,Hz -> record order (Ey,Ez,Hy,Hz); L = -sum (Ey*Hz - Ez*Hy)
        ey, ez, hy, hz = mon[:, 0], mon[:, 1], mon[:, 2], mon[:, 3]
        L = float(-(np.einsum("mxyz,mxyz->", ey, hz, dtype=np.float64) - np.einsum("mxyz,mxyz->", ez, hy, dtype=np.float64)))
        np.negative(hz, out=d[:, 0])
        d[:, 1] = hy
        d[:, 2] = ez
        np.negative(ey, out=d[:, 3])
    elif w.loss == "pulse_shape":                  # a_m = sum A*Ey^m ; L = sum_m (a_m - T_m)^2
        A = np.asarray(w.extra["A"], dtype=np.float64).reshape(mon.shape[2:])
        a = np.tensordot(mon[:, 0], A, axes=3)
        ex = extra or w.extra
        At = ex.get("target_amp")
        if At is None:
            At = 0.5 * float(np.max(np.abs(a)))
        m = np.arange(1, w.nsteps + 1, dtype=np.float64)
        T = At * np.exp(-0.5 * ((m - w.extra["target_n0"]) / w.extra["target_tau"]) ** 2) * np.sin(OMEGA_DT * (m - w.extra["target_n0"]))
        L = float(np.sum((a - T) ** 2))
        d[:, 0] = 2.0 * (a - T)[:, None, None, None] * A[None]
    else:
        raise ValueError(w.loss)
    return L, d


def cosine_similarity(x, y):
    """PAPER.md:55 eq. (2)."""
    x = np.asarray(x, dtype=np.float64).ravel()
    y = np.asarray(y, dtype=np.float64).ravel()
    return float(np.dot(x, y) / (np.linalg.norm(x) * np.linalg.norm(y)))
