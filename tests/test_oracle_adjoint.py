"""Pins for the oracle's adjoint propagation, gradient and store-based reverse run (CPU only)."""
import dataclasses

import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import workloads as W
from tests.helpers import make_oracle, oracle_gradient, rel_l2


@pytest.mark.parametrize("cpml", [orc.CPML_DEFAULTS, (0.8, 3.0, 0.05, 3.0), (1.1, 1.0, 0.0, 2.0)])
def test_adjoint_step_is_the_transpose_of_the_forward_step(cpml):
    """Dot-product test <A x, y> = <x, A^T y> for one full step (E half-step, H half-step, CPML psi included)."""
    rng = np.random.default_rng(11)
    shape, P = (9, 8, 7), 2
    s = orc.OracleSim(64, rng.uniform(1.0, 12.25, shape), P, W.S, cpml)
    N = int(np.prod(shape))
    for trial in range(3):
        x = rng.standard_normal(18 * N)
        y = rng.standard_normal(18 * N)
        Ax = s.apply_step(x)
        Aty = s.apply_step_transpose(y)
        lhs, rhs = float(Ax @ y), float(x @ Aty)
        assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), np.linalg.norm(Ax) * np.linalg.norm(y) * 1e-2), (lhs, rhs)
    # the operator is not symmetric/trivial: the transpose differs from the forward map
    assert rel_l2(s.apply_step_transpose(x), s.apply_step(x)) > 0.1


def test_method_equals_plain_definition_store_all():
    """Time reversal + uncompressed f64 store (k = 1) reproduces back-propagation through stored states."""
    w = W.tiny(nsteps=30)
    a = oracle_gradient(w, 64, orc.NATIVE, 1, mode=orc.METHOD)
    b = oracle_gradient(w, 64, orc.NATIVE, 1, mode=orc.STORE_ALL)
    assert np.abs(b["grad"]).max() > 0
    assert rel_l2(a["grad"], b["grad"]) < 1e-11
    assert abs(a["L"] - b["L"]) == 0


def _loss_only(w, eps):
    w2 = dataclasses.replace(w, eps=eps)
    s = make_oracle(w2, 64)
    s.forward(w2.nsteps, orc.NATIVE, 1)
    return W.loss_and_cotangent(w2, s.monitor_record())[0]


@pytest.mark.parametrize("loss", ["flux_x", "final_E2"])
def test_gradient_matches_central_finite_differences(loss):
    """dL/d eps_r from the reverse run vs central differences in f64, on inner, face-, edge- and corner-shell cells."""
    w = W.tiny(nsteps=36)
    if loss == "final_E2":
        lo, hi, _ = w.monitor
        w = dataclasses.replace(w, loss="final_E2", monitor=(lo, hi, 0b000111))
    eps = w.eps.astype(np.float64)
    w = dataclasses.replace(w, eps=eps)
    g = oracle_gradient(w, 64, orc.NATIVE, 1)["grad"]
    g_all = oracle_gradient(w, 64, orc.NATIVE, 1, mode=orc.STORE_ALL)["grad"]
    (lo, hi) = w.design
    P = w.pml
    cells = [(lo[0] + 1, lo[1] + 1, lo[2] + 2),            # inner interior
             (lo[0], lo[1] + 1, lo[2] + 2),                # on the x-low face of the shell
             (lo[0], lo[1], lo[2] + 3),                    # shell edge
             (lo[0], lo[1], lo[2]),                        # shell corner (low)
             (lo[0] + 2, lo[1] + 2, hi[2] - 1),            # z-high face of the shell
             (lo[0], lo[1], hi[2] - 1)]                    # shell corner (z high)
    assert hi[2] - 1 == w.shape[2] - P - 1 and lo[0] == P
    scale = np.abs(g).max()
    assert scale > 0
    for c in cells:
        h = 1e-5 * eps[c]
        ep, em = eps.copy(), eps.copy()
        ep[c] += h
        em[c] -= h
        fd = (_loss_only(w, ep) - _loss_only(w, em)) / (2 * h)
        d = tuple(c[a] - lo[a] for a in range(3))
        assert abs(g[d] - fd) < 2e-6 * scale, (c, g[d], fd)
        assert abs(g_all[d] - fd) < 2e-6 * scale, (c, g_all[d], fd)


def test_f32_k1_store_is_identical_to_uncompressed_store():
    """float32, k = 1 is the baseline: its store-based reverse must equal a reverse fed from an
    uncompressed copy of the fields, bit for bit."""
    w = W.tiny(nsteps=30)
    a = oracle_gradient(w, 32, orc.F32, 1)
    b = oracle_gradient(w, 32, orc.NATIVE, 1)
    assert np.array_equal(a["grad"], b["grad"]) and np.array_equal(a["state0"], b["state0"])
    assert a["sim"].store_bytes() == b["sim"].store_bytes() == 31 * a["sim"].slot_values() * 4


def test_worked_example_c1(golden):
    """C1 against the survey's independent float64 numpy probe (tests/golden/survey_worked_example_c1.txt)."""
    g = golden("survey_worked_example_c1.txt")
    w = W.c1()
    r = oracle_gradient(w, 64, orc.NATIVE, 1)
    assert abs(r["L"] / g["loss"] - 1) < 1e-5
    assert abs(np.abs(r["grad"]).max() / g["max_abs_grad"] - 1) < 5e-4        # printed to 4 digits
    assert abs(np.abs(r["final"][:3]).max() / g["final_max_abs_E"] - 1) < 2e-4
    P = w.pml
    assert np.abs(r["state0"][:, P:-P, P:-P, P:-P]).max() < g["state0_residual"]
    r32 = oracle_gradient(w, 32, orc.F32, 1)
    assert rel_l2(r32["final"], r["final"]) < 2 * g["f32_vs_f64_fields"]
    assert rel_l2(r32["grad"], r["grad"]) < 1e-5
    assert W.cosine_similarity(r32["grad"], r["grad"]) > 1 - 1e-9


def test_compressed_store_degrades_gracefully():
    """PAPER.md:63 (qualitative): 16-bit storage and moderate k keep the gradient direction; the store shrinks by
    (32/bits)*k."""
    w = W.c1()
    base = oracle_gradient(w, 32, orc.F32, 1)
    nslots1 = base["sim"].num_slots()
    assert nslots1 == w.nsteps + 1
    for dtype, k, min_cos in [(orc.BF16, 1, 0.9999), (orc.F16, 4, 0.999), (orc.E4M3_SCALED, 4, 0.99), (orc.F32, 8, 0.98)]:
        r = oracle_gradient(w, 32, dtype, k)
        cs = W.cosine_similarity(r["grad"], base["grad"])
        assert cs > min_cos, (dtype, k, cs)
        assert r["sim"].num_slots() == w.nsteps // k + 1
        eb = {orc.F32: 4, orc.F16: 2, orc.BF16: 2, orc.E4M3_SCALED: 1}[dtype]
        expect = r["sim"].num_slots() * (r["sim"].slot_values() * eb + (144 if dtype == orc.E4M3_SCALED else 0))
        assert r["sim"].store_bytes() == expect


def test_last_interval_when_nsteps_not_multiple_of_k():
    """DESIGN.md R10: slots at m = 0, k, 2k, ... plus the final state; the last interval is shorter."""
    w = W.tiny(nsteps=22)
    s = make_oracle(w, 32)
    s.forward(w.nsteps, orc.F32, 4)
    assert [s.slot_step(j) for j in range(s.num_slots())] == [0, 4, 8, 12, 16, 20, 22]
    # at stored steps the fetched value is the stored value itself (no interpolation arithmetic)
    data, _ = s.slot(5, orc.F32)
    vals = data.view(np.float32)
    off = s.slice_offset(2, 4)
    assert s.fetch(20, 2, 4, 3) == float(vals[off + 3])
    data6, _ = s.slot(6, orc.F32)
    v6 = data6.view(np.float32)
    assert s.fetch(22, 2, 4, 3) == float(v6[off + 3])
    a, b = np.float32(vals[off + 3]), np.float32(v6[off + 3])
    mid = s.fetch(21, 2, 4, 3)                             # halfway through the short interval [20, 22]
    assert abs(mid - 0.5 * (float(a) + float(b))) <= 1e-7 * max(abs(float(a)), abs(float(b)), 1e-30)


def _inner_design(w):
    P = w.pml
    return dataclasses.replace(w, design=(tuple([P + 1] * 3), tuple(n - P - 1 for n in w.shape)))


@pytest.mark.parametrize("shape,P", [((14, 13, 12), 3), ((11, 12, 10), 2)])
def test_tangential_only_store_reconstructs_the_inner_interior_and_the_gradient(shape, P):
    """the inner interior reads from the shell only H tangential to the LOW faces and E tangential to the HIGH
    faces.  Pins: (1) with those 12 slices alone (f64, k = 1) the reverse run returns the inner interior to state 0 to
    rounding; (2) its gradient equals back-propagation through stored states (plain definition) and the all-six-components
    run; (3) the store is exactly 1/3 (equal-sized slices per face)."""
    w = _inner_design(W.tiny(shape=shape, P=P, nsteps=30))
    full = oracle_gradient(w, 64, orc.NATIVE, 1)
    tang = oracle_gradient(w, 64, orc.NATIVE, 1, store_mode=orc.STORE_TANGENTIAL)
    plain = oracle_gradient(w, 64, orc.NATIVE, 1, mode=orc.STORE_ALL)
    peak = np.abs(full["final"]).max()
    inner = (slice(None),) + tuple(slice(P + 1, n - P - 1) for n in shape)
    assert np.abs(tang["state0"][inner]).max() <= 1e-13 * peak
    assert np.abs(plain["grad"]).max() > 0
    assert rel_l2(tang["grad"], plain["grad"]) < 1e-10
    assert rel_l2(tang["grad"], full["grad"]) < 1e-10
    assert tang["sim"].slot_values() * 3 == full["sim"].slot_values()
    assert tang["sim"].store_bytes() * 3 == full["sim"].store_bytes()
    # the forward run is untouched by the store mode
    assert np.array_equal(tang["final"], full["final"]) and tang["L"] == full["L"]


def test_tangential_only_store_compressed_matches_full_store_on_the_inner_interior():
    """Under compression (bf16, k = 4; fp8+scale, k = 3) the inner interior sees the same injected values in both store
    modes, so the float32 gradient is the same to rounding of the accumulation; scales are per slice in both."""
    w = _inner_design(W.tiny(nsteps=26))
    for dtype, k in [(orc.BF16, 4), (orc.E4M3_SCALED, 3)]:
        full = oracle_gradient(w, 32, dtype, k)
        tang = oracle_gradient(w, 32, dtype, k, store_mode=orc.STORE_TANGENTIAL)
        assert rel_l2(tang["grad"], full["grad"]) < 1e-6
        assert tang["sim"].slot_values() * 3 == full["sim"].slot_values()
