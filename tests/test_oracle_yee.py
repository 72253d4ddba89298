"""Pins for the oracle's Yee update, CPML and time reversal (CPU only).

Each test checks the oracle against something the paper or the mathematics fixes — never against itself.
"""
import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import workloads as W
from tests.helpers import make_oracle, rel_l2


def test_time_step_matches_paper(golden):
    g = golden("paper_values.txt")
    dt = orc.cfl_dt(g["dx_m"], g["courant_factor"])
    assert abs(dt - g["dt_s"]) < 0.005e-17                           # printed to 3 significant digits
    assert abs(W.DT - dt) < 1e-30 and abs(orc.courant_number(g["dx_m"], dt) - 0.99 / np.sqrt(3)) < 1e-15
    period = 1550e-9 / g["c_m_per_s"]
    assert abs(period - g["period_1550nm_s"]) < 0.005e-15
    assert round(period / dt) == g["steps_per_period"]                # "approximately 136"
    assert abs(2 * np.pi / W.OMEGA_DT - period / dt) < 1e-9


def _mode_fields(shape, plane_axes, m, n, S):
    """E0 = sin(m pi u/Nu) sin(n pi v/Nv) on the component normal to the (u,v) plane; H^{1/2} = -(S/2) curl+(E0)."""
    u_ax, v_ax = plane_axes
    c = 3 - u_ax - v_ax
    idx = np.indices(shape).astype(np.float64)
    e0 = np.sin(m * np.pi * idx[u_ax] / shape[u_ax]) * np.sin(n * np.pi * idx[v_ax] / shape[v_ax])
    f = np.zeros((6,) + tuple(shape))
    f[c] = e0

    def dplus(a, arr):
        up = np.zeros_like(arr)
        sl_src = [slice(None)] * 3
        sl_dst = [slice(None)] * 3
        sl_src[a] = slice(1, None)
        sl_dst[a] = slice(0, -1)
        up[tuple(sl_dst)] = arr[tuple(sl_src)]
        return up - arr
    # curl+(E)_h = d_{h+1}+ E_{h+2} - d_{h+2}+ E_{h+1}
    for h in range(3):
        a1, b1, a2, b2 = (h + 1) % 3, (h + 2) % 3, (h + 2) % 3, (h + 1) % 3
        f[3 + h] = -(S / 2.0) * (dplus(a1, f[b1]) - dplus(a2, f[b2]))
    return f, c, e0


@pytest.mark.parametrize("plane_axes,mn", [((0, 1), (1, 2)), ((1, 2), (2, 1)), ((2, 0), (1, 1)), ((0, 1), (3, 2))])
@pytest.mark.parametrize("eps_r", [1.0, 2.25])
def test_yee_numerical_dispersion_closed_form(plane_axes, mn, eps_r):
    """Standing wave in a PEC box = two Yee plane waves: E^n = E^0 cos(w n dt) with
    sin^2(w dt/2) = (S^2/eps_r) [sin^2(m pi/2Nu) + sin^2(n pi/2Nv)]  (Taflove, ref. 26 PAPER.md:115)."""
    shape = (11, 9, 10)
    S = W.S
    f0, c, e0 = _mode_fields(shape, plane_axes, mn[0], mn[1], S / np.sqrt(1.0) )
    # H^{1/2} must use the medium: H^{-1/2} = (S/2) curl+(E0) is independent of eps (H update has no eps)
    sim = orc.OracleSim(64, np.full(shape, eps_r), 0, S)
    sim.set_fields(f0)
    u_ax, v_ax = plane_axes
    s2 = (S * S / eps_r) * (np.sin(mn[0] * np.pi / (2 * shape[u_ax])) ** 2 + np.sin(mn[1] * np.pi / (2 * shape[v_ax])) ** 2)
    wdt = 2.0 * np.arcsin(np.sqrt(s2))
    nsteps = 400
    worst = 0.0
    done = 0
    for n in (1, 7, 50, 400):
        sim.forward(n - done, orc.NATIVE, 1)
        done = n
        f = sim.fields()
        worst = max(worst, np.abs(f[c] - e0 * np.cos(wdt * n)).max())
        others = [x for x in range(3) if x != c]
        assert np.abs(f[others]).max() < 1e-13
    assert worst < 5e-13, worst


def test_energy_conserved_in_lossless_pec_cavity():
    """W = sum eps E^n.E^n + sum H^{n+1/2}.H^{n-1/2} is an exact invariant of the leapfrog scheme for any eps(r)."""
    rng = np.random.default_rng(3)
    shape = (9, 8, 7)
    eps = rng.uniform(1.0, 12.25, shape)
    f = rng.standard_normal((6,) + shape)
    idx = np.indices(shape)
    for c in range(3):                                   # tangential E on the low PEC walls is zero
        f[c][(idx[(c + 1) % 3] == 0) | (idx[(c + 2) % 3] == 0)] = 0.0
    sim = orc.OracleSim(64, eps, 0, W.S)
    sim.set_fields(f)
    prev = f
    Ws = []
    for n in range(60):
        sim.forward(1, orc.NATIVE, 1)
        cur = sim.fields()
        Ws.append(np.sum(eps[None] * cur[:3] ** 2) + np.sum(cur[3:] * prev[3:]))
        prev = cur
    Ws = np.array(Ws)
    assert np.abs(Ws - Ws[0]).max() / abs(Ws[0]) < 1e-13
    assert np.abs(prev[:3]).max() > 0.1                  # the state is not trivially decaying


@pytest.mark.parametrize("prec,tol", [(64, 1e-13), (32, 2e-5)])
def test_round_trip_without_pml(prec, tol):
    """Forward T steps then pure time reversal (P = 0, sources replayed) returns the initial state."""
    rng = np.random.default_rng(5)
    shape = (10, 9, 8)
    eps = rng.uniform(1.0, 12.25, shape)
    f = rng.standard_normal((6,) + shape)
    idx = np.indices(shape)
    for c in range(3):
        f[c][(idx[(c + 1) % 3] == 0) | (idx[(c + 2) % 3] == 0)] = 0.0
    if prec == 32:
        f = f.astype(np.float32).astype(np.float64)
    sim = orc.OracleSim(prec, eps, 0, W.S)
    sim.add_source(1, (3, 3, 3), (5, 4, 6), rng.uniform(0.5, 1.5, (2, 1, 3)), np.sin(0.3 * np.arange(1, 101)))
    sim.set_fields(f)
    sim.forward(100, orc.NATIVE, 1)
    mid = sim.fields()
    assert rel_l2(mid, f) > 0.5                           # the run really moved the state
    sim.reverse(None, None, orc.LINEAR, orc.PURE_REVERSAL)
    assert np.abs(sim.fields() - f).max() < tol * np.abs(f).max()


def test_round_trip_with_pml_uncompressed_store():
    """With PML, f64, an uncompressed store and k = 1 the interior state 0 is recovered to rounding."""
    w = W.tiny(nsteps=40)
    s = make_oracle(w, 64)
    s.forward(w.nsteps, orc.NATIVE, 1)
    final = s.fields()
    s.reverse(None, None, orc.LINEAR, orc.METHOD)
    P = w.pml
    st0 = s.fields()[:, P:w.shape[0] - P, P:w.shape[1] - P, P:w.shape[2] - P]
    assert np.abs(final).max() > 1e-3
    assert np.abs(st0).max() < 1e-14


def test_cpml_with_zero_sigma_is_plain_yee():
    """sigma = 0 (kappa = 1): every CPML term vanishes, fields identical to a PML-free run, bit for bit."""
    w = W.tiny(nsteps=30)
    a = orc.OracleSim(32, w.eps, w.pml, W.S, (0.0, 1.0, 0.01, 3.0))
    b = orc.OracleSim(32, w.eps, 0, W.S)
    for s in (a, b):
        for q in w.sources:
            s.add_source(q.comp, q.lo, q.hi, q.amp, q.wave)
        s.forward(w.nsteps, orc.F32, 1)
    assert np.array_equal(a.fields(), b.fields())
    c = make_oracle(w, 32)
    c.forward(w.nsteps, orc.F32, 1)
    assert not np.array_equal(c.fields(), b.fields())     # the default CPML does absorb


def test_cpml_reflection_bound():
    """Default CPML (R5; constants unpinned against the paper) vs a big-domain reference whose walls are
    out of causal reach: reflection error <= 1e-2 of the peak at P = 8 (SURVEY.md 8(c) c-4 probe: 7.5e-3); sigma = 0 (bare PEC wall) is O(1)."""
    n, P, T = 36, 8, 130
    big = 112
    off = (big - n) // 2
    wave = W.gauss_sine(T, 30, 8)                          # broadband pulse
    c = n // 2
    mon_lo, mon_hi = (P, P, P), (P + 2, n - P, n - P)     # two planes next to the PML, away from the dipole's near field

    def run(N, P_, o, cpml):
        s = orc.OracleSim(32, np.ones((N, N, N)), P_, W.S, cpml)
        s.add_source(2, (c + o, c + o, c + o), (c + o + 1,) * 3, None, wave)
        s.set_monitor(tuple(x + o for x in mon_lo), tuple(x + o for x in mon_hi), 0b000100)
        s.forward(T, orc.F32, 1)
        return s.monitor_record()
    ref = run(big, 0, off, orc.CPML_DEFAULTS)              # wall echo needs >= 102 cells = 178 steps > T: not reached
    got = run(n, P, 0, orc.CPML_DEFAULTS)
    bare = run(n, P, 0, (0.0, 1.0, 0.0, 3.0))
    peak = np.abs(ref).max()
    assert np.abs(got - ref).max() / peak < 1e-2
    assert np.abs(bare - ref).max() / peak > 0.5


def test_cpml_profile_staggering_and_mirror_symmetry():
    """The CPML constants are a reading (R5: the paper prints none), but WHERE the profile is sampled is fixed by the
    Yee staggering: E-type terms sit at integer positions i, H-type terms at half-integer positions i + 1/2, and the absorber
    starts at the interface planes x = P and x = N - P.  With kappa = 1 the tables give back the graded conductivity,
    sigma + alpha = -ln b, so:
      (1) against the physical depth (P - x or x - (N - P)) the E samples (integer depths) and the H samples (half-integer
          depths) interleave on ONE strictly increasing curve sigma(depth) — a half-cell mix-up of the two tables breaks the
          interleaving;
      (2) the layout is mirror-symmetric about the middle of the grid: E(i) = E(N - i), H(i) = H(N - 1 - i);
      (3) the interior (shell included) is plain Yee: b-terms irrelevant, c = 0, 1/kappa - 1 = 0."""
    N, P = 40, 10
    s = orc.OracleSim(64, np.ones((N, N, N)), P, W.S)
    sf, kmax, amax, m = orc.CPML_DEFAULTS
    assert kmax == 1.0
    for axis in range(3):
        bE, cE, kE, bH, cH, kH = s.tables(axis)
        # (3)
        assert np.all(cE[P:N - P + 1] == 0) and np.all(kE == 0) and np.all(kH == 0)
        assert np.all(cH[P:N - P] == 0)
        assert np.all(cE[:P] != 0) and np.all(cE[N - P + 1:] != 0) and np.all(cH[:P] != 0) and np.all(cH[N - P:] != 0)
        # (2)
        i = np.arange(1, N)
        assert np.allclose(bE[i], bE[N - i], rtol=0, atol=1e-15) and np.allclose(cE[i], cE[N - i], rtol=0, atol=1e-15)
        i = np.arange(0, N)
        assert np.allclose(bH[i], bH[N - 1 - i], rtol=0, atol=1e-15) and np.allclose(cH[i], cH[N - 1 - i], rtol=0, atol=1e-15)
        # (1) low slab: depth of E node i is P - i (i = 0 .. P-1), of H node i is P - i - 1/2
        depth = np.concatenate([P - np.arange(P), P - np.arange(P) - 0.5])
        loss = np.concatenate([-np.log(bE[:P]), -np.log(bH[:P])])          # sigma + alpha at that depth
        alpha = amax * (1.0 - depth / P)
        sigma = loss - alpha
        order = np.argsort(depth)
        d_sorted, s_sorted = depth[order], sigma[order]
        assert np.all(np.diff(d_sorted) == 0.5)                               # 0.5, 1.0, 1.5, ... P: E and H alternate
        assert np.all(np.diff(s_sorted) > 0)
        # one power law through all 2P samples: sigma = sigma_max * (depth / P)^m with a single sigma_max
        smax = s_sorted / (d_sorted / P) ** m
        assert np.allclose(smax, smax[-1], rtol=1e-10)
        assert abs(smax[-1] - sf * (m + 1) * W.S) <= 1e-7 * smax[-1]            # W.S is rounded to f32 inside the oracle
