"""Pins for the oracle's minifloat codec and temporal interpolation (CPU only).

Library routines used as independent references: ml_dtypes (the casts JAX `astype` goes through, which is what
the paper ran: PAPER.md:27,53), torch CPU casts and numpy float16.
"""
import ml_dtypes
import numpy as np
import pytest
import torch

from oracle import fdtd_oracle as orc
from paper_2603_24027_b200 import workloads as W

ML = {orc.F16: np.float16, orc.BF16: ml_dtypes.bfloat16, orc.E4M3FN: ml_dtypes.float8_e4m3fn,
      orc.E4M3B11FNUZ: ml_dtypes.float8_e4m3b11fnuz, orc.E5M2FNUZ: ml_dtypes.float8_e5m2fnuz,
      orc.E4M3FNUZ: ml_dtypes.float8_e4m3fnuz, orc.E4M3: ml_dtypes.float8_e4m3, orc.E3M4: ml_dtypes.float8_e3m4}
BITS = {orc.F16: 16, orc.BF16: 16}


def _codes(dtype):
    nb = BITS.get(dtype, 8)
    return np.arange(1 << nb, dtype=np.uint32), (np.uint16 if nb == 16 else np.uint8)


@pytest.mark.parametrize("dtype", sorted(ML))
def test_decode_table_matches_library(dtype):
    codes, ut = _codes(dtype)
    lib = codes.astype(ut).view(ML[dtype]).astype(np.float64)
    mine = np.array([orc.decode_code(dtype, c) for c in codes])
    assert np.array_equal(np.isnan(lib), np.isnan(mine))
    ok = ~np.isnan(lib)
    assert np.array_equal(lib[ok], mine[ok])
    assert orc.format_max(dtype) == float(np.nanmax(lib[np.isfinite(lib)]))


@pytest.mark.parametrize("dtype", sorted(ML))
def test_encode_is_round_to_nearest_even_like_library(dtype):
    codes, ut = _codes(dtype)
    table = codes.astype(ut).view(ML[dtype]).astype(np.float64)
    fin = np.sort(np.unique(table[np.isfinite(table)]))
    # every representable value maps to itself; every midpoint ties to even; plus random values at many scales
    mids = 0.5 * (fin[1:] + fin[:-1])
    rng = np.random.default_rng(0)
    rnd = (rng.standard_normal(200000) * np.exp(rng.uniform(-12, 8, 200000))).astype(np.float32).astype(np.float64)
    rnd = rnd[np.abs(rnd) <= fin.max()]
    xs = np.concatenate([fin, mids, rnd, np.nextafter(mids, np.inf), np.nextafter(mids, -np.inf)])
    xs = xs.astype(np.float32).astype(np.float64) if dtype not in (orc.F16, orc.BF16) else xs
    # the oracle's encoder takes the f32 value promoted to double; feed the library the same f32 value
    xs32 = xs.astype(np.float32)
    with np.errstate(over="ignore"):
        lib = xs32.astype(ML[dtype]).astype(np.float64)
    mine = np.array([orc.decode_code(dtype, orc.encode_value(dtype, float(x))) for x in xs32])
    same = (lib == mine) | (np.isnan(lib) & np.isnan(mine))
    assert same.all(), (xs32[~same][:5], lib[~same][:5], mine[~same][:5])
    # encode(decode(c)) == c for every non-NaN code
    for c in codes[:: max(1, len(codes) // 4096)]:
        v = orc.decode_code(dtype, int(c))
        if np.isnan(v):
            continue
        assert orc.encode_value(dtype, v) == int(c), (dtype, c, v)


def test_slice_codecs_match_torch_cpu_casts():
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(100000) * np.exp(rng.uniform(-30, 3, 100000))).astype(np.float32)
    x[:7] = [0.0, -0.0, 1e-45, -1e-40, 65504.0, 6.1e-5, 5.9e-8]
    t = torch.from_numpy(x)
    c16, _ = orc.encode(orc.F16, x)
    assert np.array_equal(c16.view(np.uint16), t.to(torch.float16).view(torch.int16).numpy().view(np.uint16))
    cb, _ = orc.encode(orc.BF16, x)
    assert np.array_equal(cb.view(np.uint16), t.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16))
    assert np.array_equal(orc.decode(orc.F16, c16), t.to(torch.float16).float().numpy())
    assert np.array_equal(orc.decode(orc.BF16, cb), t.to(torch.bfloat16).float().numpy())
    y = np.clip(x, -448, 448)
    c8, _ = orc.encode(orc.E4M3FN, y)
    assert np.array_equal(c8, torch.from_numpy(y).to(torch.float8_e4m3fn).view(torch.uint8).numpy())
    cf, sc = orc.encode(orc.F32, x)
    assert sc == 1.0 and np.array_equal(cf.view(np.float32).view(np.uint32), x.view(np.uint32))


def test_scaled_e4m3_slice_codec():
    """DESIGN.md R13/R14: per-slice absmax scale, clamp to +-448 before the cast, RNE, scale 0 for an all-zero slice."""
    rng = np.random.default_rng(2)
    for amp in (1e-7, 3.3e-3, 1.0, 4e4):
        x = (amp * rng.standard_normal(5000)).astype(np.float32)
        codes, sc = orc.encode(orc.E4M3_SCALED, x)
        amax = np.abs(x).max()
        assert sc == np.float32(amax) / np.float32(448.0)
        assert not np.any((codes & 0x7F) == 0x7F)                      # never the NaN code
        imax = int(np.argmax(np.abs(x)))
        assert (codes[imax] & 0x7F) == 0x7E                            # amax lands on +-448
        # independent reference: torch's e4m3fn cast of the same scaled, clamped f32 values
        inv = np.float32(448.0) / np.float32(amax)
        y = np.clip((x * inv).astype(np.float32), -448, 448)
        ref = torch.from_numpy(y).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
        assert np.array_equal(codes, ref)
        back = orc.decode(orc.E4M3_SCALED, codes, sc)
        normal = np.abs(y) >= 2.0 ** -6
        assert np.all(np.abs(back[normal] - x[normal]) <= (2.0 ** -4) * np.abs(x[normal]) * (1 + 1e-6))
        assert np.all(np.abs(back - x) <= (2.0 ** -10) * sc * (1 + 1e-6) + (2.0 ** -4) * np.abs(x))
    z, sc = orc.encode(orc.E4M3_SCALED, np.zeros(17, np.float32))
    assert sc == 0.0 and not z.any() and not orc.decode(orc.E4M3_SCALED, z, sc).any()


def test_microscaled_e4m3_slice_codec():
    """DESIGN.md R20: blocks of 32 values, block scale 2^X with X = the smallest integer such that amax * 2^-X <= 448 (clamped to
    [-127, 127]) stored as X + 127, code = e4m3fn(clamp(x * 2^-X, +-448)).  References: ml_dtypes' float8_e8m0fnu (the scale byte) and float8_e4m3fn (the
    element cast), torch's e4m3fn cast, and properties no formula-retyping can fake (error bound, scale equivariance, block
    independence, ragged tail)."""
    rng = np.random.default_rng(7)
    n = 32 * 40 + 13                                                     # ragged last block
    x = (rng.standard_normal(n) * np.exp(rng.uniform(-25, 6, n))).astype(np.float32)
    x[64:96] = 0.0                                                       # an all-zero block
    x[96:128] *= np.float32(1e-38)                                       # a block of f32 subnormals / tiny values
    x[128] = np.float32(3.0e38)                                          # near the f32 maximum
    x[160:192] = np.float32(2.0 ** -5) * np.arange(-16, 16, dtype=np.float32)   # exactly representable: must round-trip
    x[192:224] = np.float32(448.0 * 2.0 ** -20) * np.linspace(-1, 1, 32, dtype=np.float32)   # amax exactly 448 * 2^X: lower X
    x[224:256] = np.float32(449.0 * 2.0 ** -20) * np.linspace(-1, 1, 32, dtype=np.float32)   # just above: X one higher
    codes, bs = orc.encode_mx(x)
    assert codes.shape == (n,) and bs.shape == (41,)
    assert not np.any((codes & 0x7F) == 0x7F)                            # never the NaN code
    back = orc.decode_mx(codes, bs)
    nb = len(bs)
    pad = np.zeros(nb * 32, np.float32)
    pad[:n] = x
    amax = np.abs(pad).reshape(nb, 32).max(axis=1)
    # the scale byte, read as ml_dtypes' e8m0: a power of two with  224 * scale < amax <= 448 * scale  (unless clamped)
    scale = bs.view(ml_dtypes.float8_e8m0fnu).astype(np.float64)
    assert np.array_equal(scale, 2.0 ** (bs.astype(np.int64) - 127))
    nz = amax > 448.0 * 2.0 ** -127
    assert np.all(scale[nz] * 224.0 < amax[nz]) and np.all(amax[nz] <= scale[nz] * 448.0)
    assert np.any(amax[nz] > scale[nz] * 256.0) and np.any(amax[nz] <= scale[nz] * 256.0)     # both binades occur
    assert np.all(bs[amax == 0] == 0) and np.all(bs[~nz] == 0)           # X clamps at -127
    # elements: the library cast of the scaled, clamped value
    y = np.clip(pad.astype(np.float64) / np.repeat(scale, 32), -448, 448).astype(np.float32)[:n]
    assert np.array_equal(codes, y.astype(ml_dtypes.float8_e4m3fn).view(np.uint8))
    assert np.array_equal(codes, torch.from_numpy(y).to(torch.float8_e4m3fn).view(torch.uint8).numpy())
    assert np.array_equal(back.astype(np.float64), codes.view(ml_dtypes.float8_e4m3fn).astype(np.float64) * np.repeat(scale, 32)[:n])
    # error bound: 3 mantissa bits -> 2^-4 relative, or half the subnormal step 2^-10 * scale; nothing is ever clipped
    sc_el = np.repeat(scale, 32)[:n]
    err = np.abs(back.astype(np.float64) - x.astype(np.float64))
    assert np.all(err <= np.maximum(2.0 ** -4 * np.abs(x.astype(np.float64)), 2.0 ** -10 * sc_el))
    assert np.all(np.abs(pad.astype(np.float64) / np.repeat(scale, 32)) <= 448.0)
    assert np.array_equal(back[160:192], x[160:192]) and not back[64:96].any()
    assert int(bs[6]) == 127 - 20 and int(bs[7]) == 127 - 19 and (codes[192] & 0x7F) == 0x7E      # 0x7E = 448
    # the largest value of each block keeps at least its leading bit: never flushed
    imax = np.abs(pad).reshape(nb, 32).argmax(axis=1) + 32 * np.arange(nb)
    keep = imax[nz]
    assert np.all(np.abs(np.pad(back, (0, nb * 32 - n))[keep]) >= 0.5 * np.abs(pad[keep]))
    # power-of-two equivariance: x * 2^j -> same codes, scale byte + j
    c2, b2 = orc.encode_mx((x[:64] * np.float32(2.0 ** 11)).astype(np.float32))
    assert np.array_equal(c2, codes[:64]) and np.array_equal(b2.astype(int), bs[:2].astype(int) + 11)
    # block independence: changing block 5 leaves every other block's bytes alone
    x2 = x.copy()
    x2[5 * 32:6 * 32] *= np.float32(1000.0)
    c3, b3 = orc.encode_mx(x2)
    other = np.ones(n, bool)
    other[5 * 32:6 * 32] = False
    assert np.array_equal(c3[other], codes[other]) and np.array_equal(np.delete(b3, 5), np.delete(bs, 5))
    # a field-sized value next to a 10^6 times larger one in ANOTHER block survives (the per-slice scale would flush it, R13)
    z = np.zeros(64, np.float32)
    z[0], z[40] = 1.0, 1.0e-6
    cz, bz = orc.encode_mx(z)
    assert abs(orc.decode_mx(cz, bz)[40] / 1.0e-6 - 1) < 2.0 ** -4
    cs, sc = orc.encode(orc.E4M3_SCALED, z)
    assert orc.decode(orc.E4M3_SCALED, cs, sc)[40] == 0.0


def test_microscaled_store_bytes_and_fetch():
    """Slot = slot_values codes + one byte per block of 32 (per slice, ragged tail counted); fetch decodes through it."""
    eps = np.ones((14, 13, 12))
    s = orc.OracleSim(32, eps, 2, W.S)
    wave = np.sin(0.3 * np.arange(24))
    s.add_source(2, (6, 6, 6), (7, 7, 7), None, wave)
    s.forward(24, orc.E4M3_MX32, 4)
    blocks = sum(6 * ((s.face_size(f) + 31) // 32) for f in range(6))
    assert s.store_bytes() == s.num_slots() * (s.slot_values() + blocks)
    data, _ = s.slot(3, orc.E4M3_MX32)
    assert data.size == s.slot_values() + blocks
    f, comp = 4, 2
    fs, off, bo = s.face_size(f), s.slice_offset(f, comp), s.block_offset(f, comp)
    vals = orc.decode_mx(data[off:off + fs], data[s.slot_values() + bo:s.slot_values() + bo + (fs + 31) // 32])
    assert np.array_equal(vals.astype(np.float64), s.fetch_face(12, f, comp))     # state 12 = slot 3, exact
    assert np.abs(vals).max() > 0
    # against the uncompressed run: within the codec's error bound of the true slice
    t = orc.OracleSim(32, eps, 2, W.S)
    t.add_source(2, (6, 6, 6), (7, 7, 7), None, wave)
    t.forward(24, orc.F32, 4)
    true = t.fetch_face(12, f, comp)
    assert np.all(np.abs(vals - true) <= 2.0 ** -3 * np.abs(true) + 2.0 ** -9 * np.abs(true).max())


def test_paper_formats_fail_by_underflow_unscaled():
    """PAPER.md:63 ranking has a cause the oracle reproduces: e4m3fnuz / e4m3 / e3m4 flush field-sized values
    (1e-3) to zero, e4m3b11fnuz / e5m2fnuz keep them."""
    x = np.float32(1.0e-3)
    kept = {d: orc.decode_code(d, orc.encode_value(d, float(x))) for d in ML if d not in (orc.F16, orc.BF16)}
    assert kept[orc.E4M3B11FNUZ] != 0 and kept[orc.E5M2FNUZ] != 0
    assert abs(kept[orc.E4M3B11FNUZ] / x - 1) < 2 ** -4
    assert kept[orc.E4M3] == 0 or abs(kept[orc.E4M3] / x - 1) > 0.2
    assert kept[orc.E3M4] == 0


# ---- interpolation (PAPER.md:47 linear; cubic = BASELINE.json option) ----
def test_linear_interpolation_exact_on_affine_data_and_at_nodes():
    rng = np.random.default_rng(4)
    for _ in range(200):
        a, b = rng.standard_normal(2)
        k = int(rng.integers(1, 33))
        assert orc.lerp64(a, b, 0, k) == a
        for num in range(k + 1):
            exact = a + (b - a) * num / k
            assert abs(orc.lerp64(a, b, num, k) - exact) <= 4e-16 * max(abs(a), abs(b))
        a32, b32 = np.float32(a), np.float32(b)
        assert orc.lerp(a32, b32, 0, k) == a32
        v = orc.lerp(a32, b32, k // 2, k)
        assert abs(v - (float(a32) + (float(b32) - float(a32)) * (k // 2) / k)) <= 3e-7 * max(abs(a), abs(b))


def test_cubic_interpolation_exact_on_cubic_polynomials():
    rng = np.random.default_rng(6)
    for _ in range(100):
        c = rng.standard_normal(4)
        k = int(rng.integers(2, 33))
        p = lambda t: ((c[3] * t + c[2]) * t + c[1]) * t + c[0]     # noqa: E731  (t in units of k)
        for num in range(k):
            v = orc.cubic64(p(-1.0), p(0.0), p(1.0), p(2.0), num, k)
            assert abs(v - p(num / k)) <= 1e-13 * (1 + np.abs(c).sum())
        assert orc.cubic64(p(-1.0), p(0.0), p(1.0), p(2.0), 0, k) == pytest.approx(p(0.0), abs=1e-15)


@pytest.mark.parametrize("k", [2, 4, 8, 16, 32])
def test_interpolation_error_on_the_papers_sine(k):
    """Fig. 1b idea: a 1550 nm carrier (~136 steps per period) sampled every k steps.
    Linear error <= (w k dt)^2/8, cubic <= (9/384)(w k dt)^4 of the amplitude (textbook interpolation bounds)."""
    w = W.OMEGA_DT
    n = np.arange(0, 40 * 136)
    f = lambda m: np.sin(w * m + 0.3)                                # noqa: E731
    err_lin = err_cub = 0.0
    for m in n:
        j, num = divmod(int(m), k)
        a, b = f(j * k), f((j + 1) * k)
        err_lin = max(err_lin, abs(orc.lerp64(a, b, num, k) - f(m)))
        err_cub = max(err_cub, abs(orc.cubic64(f((j - 1) * k), a, b, f((j + 2) * k), num, k) - f(m)))
    bl, bc = (w * k) ** 2 / 8, (9.0 / 384.0) * (w * k) ** 4
    assert err_lin <= bl * 1.0001 and err_lin >= 0.8 * bl * (1 - (w * k) ** 2 / 12)       # the bound is nearly attained
    assert err_cub <= bc * 1.0001 and err_cub >= 0.5 * bc * (1 - (w * k) ** 2)
    if k <= 8:
        assert err_lin < 2e-2                                         # "linear interpolation provides sufficient accuracy"


def test_compression_factor_matches_paper(golden):
    """compression factor = (32/bits)*k vs float32, k=1; 8-bit, k = 16 -> 64x."""
    g = golden("paper_values.txt")
    T = 1600
    eps = np.ones((8, 8, 8))
    wave = np.zeros(T)
    sizes = {}
    for dtype, k in [(orc.F32, 1), (orc.E4M3B11FNUZ, 16), (orc.BF16, 4)]:
        s = orc.OracleSim(32, eps, 2, W.S)
        s.add_source(2, (4, 4, 4), (5, 5, 5), None, wave)
        s.forward(T, dtype, k)
        sizes[(dtype, k)] = s.store_bytes()
        assert s.num_slots() == T // k + 1
    ratio = sizes[(orc.F32, 1)] / sizes[(orc.E4M3B11FNUZ, 16)]
    assert ratio == pytest.approx(4 * (T + 1) / (T // 16 + 1))
    assert abs(ratio / g["compression_e4m3_k16"] - 1) < 0.02           # -> 64 as T grows (slot-0 overhead)
    assert sizes[(orc.F32, 1)] / sizes[(orc.BF16, 4)] == pytest.approx(2 * (T + 1) / (T // 4 + 1))


# ---------------------------------------------------------------------------------------------------------
# The fetch PATH of the cubic option (slot choice j0-1 .. j0+2 and the fall-back rules of DESIGN.md R11 / SURVEY c-7),
# pinned through the real record -> fetch route.  With a Courant number of 0 the curl terms vanish, so a source with
# wave[m-1] = p(m) - p(m-1) leaves E^m = p(m) on its box: the interface values are a known cubic polynomial in the step
# index (integers, exact in f32 and f64).  Expected values come from p alone: p(n) where R11 says "cubic", the chord
# between the two bracketing stored values where it says "linear" (first interval, last interval, any interval whose
# neighbouring slots are not k apart), p(n) at stored steps.  A one-slot shift or a wrong fall-back condition fails it.
# ---------------------------------------------------------------------------------------------------------
def _p_cubic(m):
    m = np.asarray(m, dtype=np.float64)
    return 2.0 * m ** 3 - 45.0 * m ** 2 + 210.0 * m


@pytest.mark.parametrize("prec,dtype", [(64, orc.NATIVE), (32, orc.F32), (32, orc.NATIVE)])
@pytest.mark.parametrize("T,k", [(23, 4), (24, 4), (17, 5), (9, 3), (7, 4), (3, 4)])
def test_cubic_fetch_path_slot_choice_and_fallbacks(prec, dtype, T, k):
    n, P = 8, 2
    s = orc.OracleSim(prec, np.ones((n, n, n)), P, 0.0)
    wave = _p_cubic(np.arange(1, T + 1)) - _p_cubic(np.arange(0, T))
    # Ez on the whole low-x interface plane (face 0: plane i = P, cross-section [P, n-P)^2)
    s.add_source(2, (P, P, P), (P + 1, n - P, n - P), None, wave)
    s.forward(T, dtype, k)
    stored = list(range(0, T + 1, k)) + ([T] if T % k else [])
    assert [s.slot_step(j) for j in range(s.num_slots())] == stored
    face, comp = 0, 2
    nfs = s.face_size(face)
    for nstate in range(T + 1):
        if nstate in stored:
            kind, want = "exact", float(_p_cubic(nstate))
        else:
            j0 = nstate // k
            m0, m1 = stored[j0], stored[j0 + 1]
            cubic = j0 >= 1 and j0 + 2 < len(stored) and m1 - m0 == k and stored[j0 + 2] - m1 == k
            if cubic:
                kind, want = "cubic", float(_p_cubic(nstate))
            else:
                kind = "linear"
                want = float(_p_cubic(m0) + (nstate - m0) / (m1 - m0) * (_p_cubic(m1) - _p_cubic(m0)))
        got = s.fetch_face(nstate, face, comp, orc.CUBIC)
        assert got.shape == (nfs,)
        tol = (1e-6 if prec == 32 or dtype == orc.F32 else 1e-12) * max(1.0, float(np.max(np.abs(_p_cubic(stored)))))
        if kind == "exact":
            tol = 0.0
        assert np.max(np.abs(got - want)) <= tol, (T, k, nstate, kind, float(got[0]), want)
        # the linear option on the same store: chord everywhere between stored steps
        lin = s.fetch(nstate, face, comp, 0, orc.LINEAR)
        if nstate not in stored:
            j0 = nstate // k
            m0, m1 = stored[j0], stored[j0 + 1]
            chord = float(_p_cubic(m0) + (nstate - m0) / (m1 - m0) * (_p_cubic(m1) - _p_cubic(m0)))
            assert abs(lin - chord) <= max(tol, 1e-12)
    # the cubic and the chord differ on the cubic intervals (the test can tell them apart)
    if len(stored) >= 5 and k > 1:
        n_mid = stored[1] + 1
        assert abs(float(_p_cubic(n_mid)) - s.fetch(n_mid, face, comp, 0, orc.LINEAR)) > 1.0
    # components that have no source stay zero in every slot
    assert np.all(s.fetch_face(min(T, k + 1), face, 0, orc.CUBIC) == 0.0)
