// fdtd_store.cuh — the paper's contribution as kernels: record / quantise / subsample and
// dequantise / interpolate / inject (row R1), plus the small source / monitor / cotangent kernels.
// PAPER.md:35 (cast to a smaller bit-width, cast back in the reverse run), PAPER.md:47 (every k-th step, linear
// interpolation).  Codec readings: DESIGN.md R12-R14; interpolation arithmetic: R11.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>

#include "fdtd_dev.cuh"

namespace fdtd {

// 0..3: BASELINE.json's store types.  10..14: the paper's five unscaled float8 flavours (ids as in fdtd.h).
// 5: micro-scaled E4M3 (blocks of 32 values share a power-of-two scale byte; R20).
enum { DT_F32 = 0, DT_F16 = 1, DT_BF16 = 2, DT_E4M3S = 3, DT_MX32 = 5,
       DT_E4M3B11FNUZ = 10, DT_E5M2FNUZ = 11, DT_E4M3FNUZ = 12, DT_E4M3 = 13, DT_E3M4 = 14 };

// Interface store: slot j = state min(j*k, nsteps); inside a slot
// [face 0..5][comp 0..5][u][v] in the store dtype; face = 2*axis + side, plane index P (low) / n-P-1 (high),
// (u,v) = the two other axes in increasing order, interior extent only.  36 f32 scales per slot (fp8 only).
struct StoreDev {
  char* base;
  size_t slot_bytes;
  float* scales;        // [nslots][36]
  unsigned* amax;       // [nslots][36] bit pattern of max|x| per slice (fp8)
  int nslots, nsteps, k, dtype;
  int mode;             // 0: all six components on every face; 1: tangential only (H on the low faces, E on the high faces)
  long long slot_values;
  long long val_off[7];   // prefix sums of ncomp(mode)*face_size  (value index of face f)
  long long cell_off[7];  // prefix sums of face_size    (shell-cell index of face f)
  int du[6], dv[6];
  // micro-scaled store (DT_MX32): a slot is [codes: slot_values bytes][block scales]; a slice has ceil(face/32) blocks
  long long blk_off[7];   // prefix sums of ncomp(mode)*blocks(face): block index of face f inside a slot
  long long blkc_off[7];  // prefix sums of blocks(face)  (what cell_off is for cells)
};

__device__ __forceinline__ int elem_bytes(int dt) { return dt == DT_F32 ? 4 : ((dt == DT_F16 || dt == DT_BF16) ? 2 : 1); }

// ---- value codecs (round-to-nearest-even, subnormals kept) ----
template <int DT> struct Codec;
template <> struct Codec<DT_F32> {
  typedef float code_t;
  static __device__ __forceinline__ code_t enc(float x, float) { return x; }
  static __device__ __forceinline__ float dec(code_t c, float) { return c; }
};
template <> struct Codec<DT_F16> {
  typedef unsigned short code_t;
  static __device__ __forceinline__ code_t enc(float x, float) { return __half_as_ushort(__float2half_rn(x)); }
  static __device__ __forceinline__ float dec(code_t c, float) { return __half2float(__ushort_as_half(c)); }
};
template <> struct Codec<DT_BF16> {
  typedef unsigned short code_t;
  static __device__ __forceinline__ code_t enc(float x, float) { return __bfloat16_as_ushort(__float2bfloat16_rn(x)); }
  static __device__ __forceinline__ float dec(code_t c, float) { return __uint_as_float((unsigned)c << 16); }
};
template <> struct Codec<DT_E4M3S> {   // OCP E4M3 (max 448) after a per-slice scale: code = e4m3(clamp(x*inv, +-448))
  typedef unsigned char code_t;
  static __device__ __forceinline__ code_t enc(float x, float inv) {
    float y = x * inv;
    y = fminf(448.0f, fmaxf(-448.0f, y));
    return (code_t)__nv_cvt_float_to_fp8(y, __NV_SATFINITE, __NV_E4M3);
  }
  static __device__ __forceinline__ float dec(code_t c, float scale) {
    const __half_raw h = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)c, __NV_E4M3);
    return __half2float(__half(h)) * scale;
  }
};

// Micro-scaled E4M3 (R20): the element cast is the scaled one's, the scale is 2^X per block of 32 values with
// X = the smallest integer with amax * 2^-X <= 448, clamped to [-127, 127], stored as the byte X + 127 (the block maximum lands
// in (224, 448], nothing is clipped).  Multiplying by 2^-X / 2^X is exact.
template <> struct Codec<DT_MX32> : Codec<DT_E4M3S> {};
__device__ __forceinline__ int mx_exponent(unsigned amax_bits) {   // f32 bits of max|x|
  // floor(log2 amax) - 8, one more where the mantissa is above 1.75 (448 = 1.75 * 2^8); f32 subnormals fall below the clamp
  return max((int)(amax_bits >> 23) - 135 + ((amax_bits & 0x7fffffu) > 0x600000u ? 1 : 0), -127);
}
__device__ __forceinline__ float mx_pow2(int k) {   // 2^k, k in [-127, 127] (2^-127 is an f32 subnormal)
  return k > -127 ? __uint_as_float((unsigned)(k + 127) << 23) : __uint_as_float(0x00400000u);
}
__device__ __forceinline__ float mx_scale(unsigned char byte) { return mx_pow2((int)byte - 127); }

// Software minifloat cast for the paper's unscaled float8 flavours (e4m3b11fnuz, e5m2fnuz, e4m3fnuz, e4m3,
// e3m4; "f" = finite only, "n" = a NaN code exists, "uz" = no negative zero).  EB exponent bits, MB mantissa bits.
// Value-level rule (R12): e = max(floor(log2|x|), 1-BIAS), q = 2^(e-MB), result = sign * q * RNE(|x|/q); above the
// largest finite value IEEE flavours give inf, fn / fnuz flavours NaN (what an XLA / ml_dtypes astype does); fnuz has a
// single zero (0x00) and a single NaN (0x80).  The hardware has no conversion for these types, so this is integer code.
enum { FL_IEEE = 0, FL_FN = 1, FL_FNUZ = 2 };
template <int EB, int MB, int BIAS, int FL>
struct MiniFloat {
  typedef unsigned char code_t;
  static constexpr unsigned EALL = (1u << EB) - 1u, MALL = (1u << MB) - 1u, SIGN = 1u << (EB + MB);
  static __device__ __forceinline__ float pow2(int k) { return __uint_as_float((unsigned)(127 + k) << 23); }   // k in [-126, 127]
  static __device__ __forceinline__ code_t enc(float x, float) {
    const unsigned u = __float_as_uint(x);
    const unsigned sbit = (u >> 31) ? SIGN : 0u;
    const unsigned nan_code = FL == FL_FNUZ ? SIGN : (FL == FL_FN ? (sbit | (EALL << MB) | MALL) : (sbit | (EALL << MB) | (1u << (MB - 1))));
    const unsigned inf_code = FL == FL_IEEE ? (sbit | (EALL << MB)) : nan_code;
    const unsigned zero_code = FL == FL_FNUZ ? 0u : sbit;
    const unsigned au = u & 0x7fffffffu;
    if (au > 0x7f800000u) return (code_t)nan_code;
    if (au == 0x7f800000u) return (code_t)inf_code;
    const float a = __uint_as_float(au);
    int e = (int)(au >> 23) - 127;                 // floor(log2 a) for normal a; f32 subnormals fall below every 1-BIAS
    e = max(e, 1 - BIAS);
    int r = (int)rintf(a * pow2(MB - e));          // exact product (power of two), round-to-nearest-even; r <= 2^(MB+1)
    if (r == (2 << MB)) { r = 1 << MB; ++e; }
    const int emax = FL == FL_IEEE ? (int)EALL - 1 - BIAS : (int)EALL - BIAS;
    const int rmax = FL == FL_FN ? (2 << MB) - 2 : (2 << MB) - 1;
    if (e > emax || (e == emax && r > rmax)) return (code_t)inf_code;
    if (r == 0) return (code_t)zero_code;
    if (r < (1 << MB)) return (code_t)(sbit | (unsigned)r);                       // subnormal: exponent field 0
    return (code_t)(sbit | ((unsigned)(e + BIAS) << MB) | ((unsigned)r - (1u << MB)));
  }
  static __device__ __forceinline__ float dec(code_t c, float) {
    const unsigned sign = (c >> (EB + MB)) & 1u, ef = (c >> MB) & EALL, mf = c & MALL;
    if (FL == FL_FNUZ && c == SIGN) return __uint_as_float(0x7fc00000u);
    if (FL == FL_FN && ef == EALL && mf == MALL) return __uint_as_float(0x7fc00000u);
    if (FL == FL_IEEE && ef == EALL) return mf ? __uint_as_float(0x7fc00000u) : __uint_as_float(sign ? 0xff800000u : 0x7f800000u);
    const float v = ef == 0 ? (float)mf * pow2(1 - BIAS - MB) : (float)((1u << MB) + mf) * pow2((int)ef - BIAS - MB);
    return sign ? -v : v;
  }
};
template <> struct Codec<DT_E4M3B11FNUZ> : MiniFloat<4, 3, 11, FL_FNUZ> {};
template <> struct Codec<DT_E5M2FNUZ> : MiniFloat<5, 2, 16, FL_FNUZ> {};
template <> struct Codec<DT_E4M3FNUZ> : MiniFloat<4, 3, 8, FL_FNUZ> {};
template <> struct Codec<DT_E4M3> : MiniFloat<4, 3, 7, FL_IEEE> {};
template <> struct Codec<DT_E3M4> : MiniFloat<3, 4, 3, FL_IEEE> {};

// ---- temporal interpolation, all in f32 (R11) ----
__device__ __forceinline__ float lerp_value(float a, float b, int num, int den) {
  const float w = (float)num / (float)den;
  return fmaf(w, b - a, a);
}
__device__ __forceinline__ float cubic_value(float vm1, float v0, float v1, float v2, int num, int den) {
  const float t = (float)num / (float)den;
  const float wm1 = -t * (t - 1.0f) * (t - 2.0f) / 6.0f;
  const float w0 = (t + 1.0f) * (t - 1.0f) * (t - 2.0f) / 2.0f;
  const float w1 = -(t + 1.0f) * t * (t - 2.0f) / 2.0f;
  const float w2 = (t + 1.0f) * t * (t - 1.0f) / 6.0f;
  return (wm1 * vm1 + w0 * v0) + (w1 * v1 + w2 * v2);
}

// which slots bracket state n, and how to combine them
struct FetchPlan {
  int mode;        // 0 = exact slot j[1]; 1 = linear j[1], j[2]; 2 = cubic j[0..3]
  int j[4];
  int num, den;
};
__device__ __host__ __forceinline__ int slot_step(int j, int k, int nsteps) {
  const long long s = (long long)j * k;
  return s < nsteps ? (int)s : nsteps;
}
__device__ __host__ __forceinline__ FetchPlan make_plan(int nstate, int nsteps, int k, int nslots, int interp) {
  FetchPlan p;
  p.mode = 0; p.num = 0; p.den = 1; p.j[0] = p.j[1] = p.j[2] = p.j[3] = 0;
  if (nstate == nsteps) { p.j[1] = nslots - 1; return p; }
  const int j0 = nstate / k, m0 = j0 * k;
  p.j[1] = j0;
  if (nstate == m0) return p;
  const int m1 = slot_step(j0 + 1, k, nsteps);
  p.j[2] = j0 + 1;
  p.num = nstate - m0;
  p.den = m1 - m0;
  p.mode = 1;
  if (interp == 1 && j0 >= 1 && j0 + 2 < nslots && m1 - m0 == k && slot_step(j0 + 2, k, nsteps) - m1 == k) {
    p.mode = 2;
    p.j[0] = j0 - 1;
    p.j[3] = j0 + 2;
    p.den = k;
  }
  return p;
}

template <int DT>
__device__ __forceinline__ float fetch_value(const StoreDev& s, const FetchPlan& p, int slice, long long vidx, long long bidx) {
  typedef typename Codec<DT>::code_t code_t;
  auto val = [&](int j) {
    const char* slot = s.base + (size_t)j * s.slot_bytes;
    const code_t c = reinterpret_cast<const code_t*>(slot)[vidx];
    float sc = 1.0f;
    if (DT == DT_E4M3S) sc = s.scales[(size_t)j * 36 + slice];
    if (DT == DT_MX32) sc = mx_scale(reinterpret_cast<const unsigned char*>(slot)[s.slot_values + bidx]);
    return Codec<DT>::dec(c, sc);
  };
  const float a = val(p.j[1]);
  if (p.mode == 0) return a;
  const float b = val(p.j[2]);
  if (p.mode == 1) return lerp_value(a, b, p.num, p.den);
  return cubic_value(val(p.j[0]), a, b, val(p.j[3]), p.num, p.den);
}

// cell of element e of face f
__device__ __forceinline__ void face_cell(const Dev& d, const StoreDev& s, int f, long long e, int c[3]) {
  const int a = f >> 1, side = f & 1;
  const int b0 = a == 0 ? 1 : 0, b1 = a == 2 ? 1 : 2;
  const int u = (int)(e / s.dv[f]), v = (int)(e % s.dv[f]);
  c[a] = side ? d.n[a] - d.P - 1 : d.P;
  c[b0] = d.P + u;
  c[b1] = d.P + v;
}
__device__ __forceinline__ int find_face(const long long* off, long long t) {
  int f = 0;
#pragma unroll
  for (int g = 1; g < 6; ++g) f += (t >= off[g]);
  return f;
}
__device__ __forceinline__ const float* field_ptr(const Dev& d, int comp) { return comp < 3 ? d.E[comp] : d.H[comp - 3]; }

__device__ __forceinline__ int cur_step(int m_base, const int* step_dev) { return m_base + (step_dev ? *step_dev : 0); }
__device__ __forceinline__ int record_slot(const StoreDev& s, int m) {
  return (m == s.nsteps) ? s.nslots - 1 : m / s.k;
}

// ---------------------------------------------------------------------------------------------------------
// Record (row A5).  Phase 1 (fp8 only): per-slice absmax, warp-reduced, one atomicMax per (warp, slice).
// Phase 2: gather the 36 slices from the field arrays, cast, write the slot.
// ---------------------------------------------------------------------------------------------------------
// half = 0: the three E components, 1: the three H components, 2: all six.  The two halves of a slot can be written
// by different launches: E^m is final after the E half-step, H^{m+1/2} after the H half-step.
// coff: prefix sums of the per-face slice length that t enumerates — cell_off (t = value) or blkc_off (t = block of 32 values).
struct RecItem { int f, comp, rank; long long e; };   // rank: position of the component among those the face stores
// Tangential store (mode 1): the inner interior reads from the shell only H tangential to the LOW faces
// (through d^- in the inverse-E update) and E tangential to the HIGH faces (through d^+ in the inverse-H update); a face
// keeps those two components, in increasing component order.
__device__ __forceinline__ int tangential_comp(int axis, int rank) { return axis == 0 ? 1 + rank : (axis == 1 ? 2 * rank : rank); }
__device__ __forceinline__ bool record_item_tangential(const long long* coff, long long t, int half, RecItem& it) {
  // half 0: E on the three high faces, half 1: H on the three low faces, half 2: E part then H part
  for (int h = (half == 2 ? 0 : half); h <= (half == 2 ? 1 : half); ++h) {
    for (int a = 0; a < 3; ++a) {
      const int f = 2 * a + (h == 0 ? 1 : 0);
      const long long fs = coff[f + 1] - coff[f];
      if (t < 2 * fs) {
        const int rank = (int)(t / fs);
        it.f = f;
        it.rank = rank;
        it.comp = tangential_comp(a, rank) + (h == 1 ? 3 : 0);
        it.e = t - rank * fs;
        return true;
      }
      t -= 2 * fs;
    }
  }
  return false;
}
__device__ __forceinline__ bool record_item(const StoreDev& s, const long long* coff, long long t, int half, RecItem& it) {
  if (s.mode == 1) return record_item_tangential(coff, t, half, it);
  const int nc = half == 2 ? 6 : 3;
  if (t >= coff[6] * nc) return false;
  // t enumerates [face][comp in half][element]; coff = prefix sums of face sizes
  int f = 0;
#pragma unroll
  for (int g = 1; g < 6; ++g) f += (t >= coff[g] * nc);
  const long long fs = coff[f + 1] - coff[f];
  const long long r = t - coff[f] * nc;
  it.f = f;
  it.comp = (int)(r / fs) + (half == 1 ? 3 : 0);
  it.rank = it.comp;
  it.e = r % fs;
  return true;
}
__device__ __forceinline__ long long value_index(const StoreDev& s, const RecItem& it, long long e) {
  return s.val_off[it.f] + it.rank * (s.cell_off[it.f + 1] - s.cell_off[it.f]) + e;
}

__global__ void __launch_bounds__(256) k_record_amax(const __grid_constant__ Dev d, const __grid_constant__ StoreDev s,
                                                      int m_base, const int* step_dev, int half) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  RecItem it;
  if (!record_item(s, s.cell_off, t, half, it)) return;
  const int slot = record_slot(s, cur_step(m_base, step_dev));
  const int f = it.f, comp = it.comp;
  int c[3];
  face_cell(d, s, f, it.e, c);
  const float x = field_ptr(d, comp)[((long long)c[0] * d.n[1] + c[1]) * d.n[2] + c[2]];
  const unsigned bits = __float_as_uint(fabsf(x));
  const unsigned key = f * 6 + comp;
  const unsigned act = __activemask();
  const unsigned peers = __match_any_sync(act, key);
  const unsigned mx = __reduce_max_sync(peers, bits);
  if ((threadIdx.x & 31) == (__ffs(peers) - 1)) atomicMax(&s.amax[(size_t)slot * 36 + key], mx);
}

template <int DT>
__global__ void __launch_bounds__(256) k_record(const __grid_constant__ Dev d, const __grid_constant__ StoreDev s,
                                                int m_base, const int* step_dev, int half) {
  typedef typename Codec<DT>::code_t code_t;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  RecItem it;
  if (!record_item(s, s.cell_off, t, half, it)) return;
  const int slot = record_slot(s, cur_step(m_base, step_dev));
  const int f = it.f, comp = it.comp;
  const long long e = it.e;
  int c[3];
  face_cell(d, s, f, e, c);
  const float x = field_ptr(d, comp)[((long long)c[0] * d.n[1] + c[1]) * d.n[2] + c[2]];
  float inv = 1.0f;
  if (DT == DT_E4M3S) {
    const float amax = __uint_as_float(s.amax[(size_t)slot * 36 + f * 6 + comp]);
    inv = amax > 0.0f ? 448.0f / amax : 0.0f;
    if (e == 0) s.scales[(size_t)slot * 36 + f * 6 + comp] = amax > 0.0f ? amax / 448.0f : 0.0f;
  }
  reinterpret_cast<code_t*>(s.base + (size_t)slot * s.slot_bytes)[value_index(s, it, e)] = Codec<DT>::enc(x, inv);
}

// Micro-scaled record (DT_MX32, R20): one warp = one block of 32 consecutive values of a slice; the block's absmax
// is one redux.max over the lanes, so there is no slice-wide pass and no atomic.  Lane 0 writes the scale byte behind the codes.
__global__ void __launch_bounds__(256) k_record_mx(const __grid_constant__ Dev d, const __grid_constant__ StoreDev s,
                                                   int m_base, const int* step_dev, int half) {
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  RecItem it;
  if (!record_item(s, s.blkc_off, w, half, it)) return;   // warp-uniform
  const int slot = record_slot(s, cur_step(m_base, step_dev));
  const int f = it.f;
  const long long fs = s.cell_off[f + 1] - s.cell_off[f];
  const long long e = it.e * 32 + lane;
  float x = 0.0f;
  if (e < fs) {
    int c[3];
    face_cell(d, s, f, e, c);
    x = field_ptr(d, it.comp)[((long long)c[0] * d.n[1] + c[1]) * d.n[2] + c[2]];
  }
  const int X = mx_exponent(__reduce_max_sync(0xffffffffu, __float_as_uint(fabsf(x))));
  unsigned char* slotp = reinterpret_cast<unsigned char*>(s.base + (size_t)slot * s.slot_bytes);
  if (e < fs) slotp[value_index(s, it, e)] = Codec<DT_MX32>::enc(x, mx_pow2(-X));
  if (lane == 0) slotp[s.slot_values + s.blk_off[f] + it.rank * (s.blkc_off[f + 1] - s.blkc_off[f]) + it.e] = (unsigned char)(X + 127);
}

// ---------------------------------------------------------------------------------------------------------
// Dequantise / interpolate / inject (row R1).  One thread = one shell cell of one face, three components
// (magnetic = 0: E, 1: H).  Where faces overlap (edges, corners) the lowest face index wins (R9).
// E injection also takes the shell-cell gradient term in its dE form:
//   acc += sum_c lE_c * (E_old - E_new)_c / ce      on design ∩ shell.
// ---------------------------------------------------------------------------------------------------------
// Eold: where the shell E of state m sits (read for the gradient term); Eout / Hout: where the injected values go.  The same
// arrays in the in-place path; old / new buffer in the fused reverse path (fdtd_fused.cuh).
struct InjIO {
  const float* Eold[3];
  float* Eout[3];
  float* Hout[3];
};
template <int DT>
__global__ void __launch_bounds__(256) k_inject(const __grid_constant__ Dev d, const __grid_constant__ StoreDev s,
                                                int m_base, const int* step_dev, int magnetic, int interp,
                                                const __grid_constant__ InjIO io, int nfaces) {
  // nfaces = 6, or 4 where the inverse kernels inject the interior cells of the two z faces themselves (fdtd_stencil.cuh, ZF);
  // the z faces' edge cells belong to an x or y face anyway
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= s.cell_off[nfaces]) return;
  const int nstate = cur_step(m_base, step_dev) - 1;
  const int f = find_face(s.cell_off, t);
  const long long e = t - s.cell_off[f];
  int c[3];
  face_cell(d, s, f, e, c);
  const int a = f >> 1;
  // does a lower-index face contain this cell?
  for (int g = 0; g < a; ++g)
    if (c[g] == d.P || c[g] == d.n[g] - d.P - 1) return;
  if ((f & 1) && d.P == d.n[a] - d.P - 1) return;
  const bool tang = s.mode == 1;
  if (tang && ((f & 1) != (magnetic ? 0 : 1))) return;   // tangential store: H lives on the low faces, E on the high ones
  const FetchPlan p = make_plan(nstate, s.nsteps, s.k, s.nslots, interp);
  const long long q = ((long long)c[0] * d.n[1] + c[1]) * d.n[2] + c[2];
  const long long fs = (long long)s.du[f] * s.dv[f];
  const long long nb = s.blkc_off[f + 1] - s.blkc_off[f], b0 = s.blk_off[f] + (e >> 5);   // DT_MX32: block of element e
  float nv[3];
#pragma unroll
  for (int cc = 0; cc < 3; ++cc) {
    const int comp = magnetic ? 3 + cc : cc;
    if (tang) {
      if (cc == a) continue;
      const int rank = cc > a ? cc - 1 : cc;      // position among the two components tangential to axis a
      nv[cc] = fetch_value<DT>(s, p, f * 6 + comp, s.val_off[f] + rank * fs + e, b0 + rank * nb);
    } else {
      nv[cc] = fetch_value<DT>(s, p, f * 6 + comp, s.val_off[f] + comp * fs + e, b0 + comp * nb);
    }
  }
  if (magnetic) {
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
      if (!tang || cc != a) io.Hout[cc][q] = nv[cc];
    return;
  }
  if (tang) {   // the design box lies in the inner interior (checked on the host): no shell gradient term
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
      if (cc != a) io.Eout[cc][q] = nv[cc];
    return;
  }
  const bool des = d.has_design && c[0] >= d.dlo[0] && c[0] < d.dhi[0] && c[1] >= d.dlo[1] && c[1] < d.dhi[1] &&
                   c[2] >= d.dlo[2] && c[2] < d.dhi[2];
  if (des) {
    const double ce = (double)d.ce[q];
    double sacc = 0.0;
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
      const float dE = io.Eold[cc][q] - nv[cc];
      sacc += (double)d.lE[cc][q] * ((double)dE / ce);
    }
    const long long ei = ((long long)(c[0] - d.dlo[0]) * (d.dhi[1] - d.dlo[1]) + (c[1] - d.dlo[1])) * (d.dhi[2] - d.dlo[2]) +
                         (c[2] - d.dlo[2]);
    d.acc[ei] += sacc;
  }
#pragma unroll
  for (int cc = 0; cc < 3; ++cc) io.Eout[cc][q] = nv[cc];
}

// ---------------------------------------------------------------------------------------------------------
// Small kernels: sources, monitor, cotangents, boxes
// ---------------------------------------------------------------------------------------------------------
struct SrcDev {
  int comp;
  int lo[3], hi[3];
  const float* amp;      // device, [hi-lo] or nullptr
  long long wave_off;    // into waves[]
};

// E_comp += sign * (amp * wave[m-1]) on each source box; blockIdx.y = source (R8)
__global__ void k_sources(const __grid_constant__ Dev d, const SrcDev* __restrict__ src, const float* __restrict__ waves,
                          int m_base, const int* step_dev, float sign, int x0, int x1) {
  const SrcDev s = src[blockIdx.y];
  const int ey = s.hi[1] - s.lo[1], ez = s.hi[2] - s.lo[2];
  const long long cells = (long long)(s.hi[0] - s.lo[0]) * ey * ez;
  const int m = cur_step(m_base, step_dev);
  const float w = waves[s.wave_off + m - 1];
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < cells; t += (long long)gridDim.x * blockDim.x) {
    const int kk = (int)(t % ez), jj = (int)((t / ez) % ey), ii = (int)(t / ((long long)ez * ey));
    if (s.lo[0] + ii < x0 || s.lo[0] + ii >= x1) continue;   // x clip (chunked launches)
    const float amp = s.amp ? s.amp[t] : 1.0f;
    const float v = amp * w;
    atomicAdd(&d.E[s.comp][((long long)(s.lo[0] + ii) * d.n[1] + (s.lo[1] + jj)) * d.n[2] + (s.lo[2] + kk)], sign * v);
  }
}

struct BoxDev {
  int lo[3], hi[3];
  unsigned mask;
  int ncomp;
};

// mode 0: rec[(m-1)][ci][box] = F_comp        (monitor write, forward)
// mode 1: lambda_comp += rec[(m-1)][ci][box]   (monitor cotangent, reverse)
// mode 2: out[ci][box] = F_comp                (fdtd_get_box; m ignored)
// mode 3: lambda_comp += rec[ci][box]          (dL/dfinal)
// half: 0 = E components only, 1 = H components only, 2 = all (the fused forward path writes a monitor row in two parts)
__global__ void k_box(const __grid_constant__ Dev d, const __grid_constant__ BoxDev b, float* rec, int m_base,
                      const int* step_dev, int mode, int half) {
  const int ex = b.hi[0] - b.lo[0], ey = b.hi[1] - b.lo[1], ez = b.hi[2] - b.lo[2];
  const long long bc = (long long)ex * ey * ez;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= bc * b.ncomp) return;
  const int ci = (int)(t / bc);
  const long long r = t % bc;
  int comp = 0, seen = -1;
  for (int c = 0; c < 6; ++c)
    if (b.mask >> c & 1) { if (++seen == ci) { comp = c; break; } }
  if ((half == 0 && comp >= 3) || (half == 1 && comp < 3)) return;
  if (mode == 0 && cur_step(m_base, step_dev) < 1) return;   // state 0 has no monitor row
  const int kk = (int)(r % ez), jj = (int)((r / ez) % ey), ii = (int)(r / ((long long)ez * ey));
  const long long q = ((long long)(b.lo[0] + ii) * d.n[1] + (b.lo[1] + jj)) * d.n[2] + (b.lo[2] + kk);
  long long off = t;
  if (mode == 0 || mode == 1) off += (long long)(cur_step(m_base, step_dev) - 1) * b.ncomp * bc;
  if (mode == 0 || mode == 2) rec[off] = (comp < 3 ? d.E[comp] : d.H[comp - 3])[q];
  else (comp < 3 ? d.lE[comp] : d.lH[comp - 3])[q] += rec[off];
}

// debugging aid (fdtd_debug_guard_check): bytes of a guard band that no longer hold the 0xFF fill pattern
__global__ void k_guard_count(const unsigned char* p, size_t n, unsigned long long* bad) {
  unsigned c = 0;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) c += p[t] != 0xFFu;
  if (c) atomicAdd(bad, (unsigned long long)c);
}
__global__ void k_tick(int* step_dev, int delta) { *step_dev += delta; }
__global__ void k_set_int(int* p, int v) { *p = v; }

// ce = fl(S * fl(1/eps)) (R3); also the minimum of eps for validation
__global__ void k_make_ce(const float* __restrict__ eps, float* __restrict__ ce, long long N, float S) {
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N; t += (long long)gridDim.x * blockDim.x) {
    const float inv = 1.0f / eps[t];
    ce[t] = S * inv;
  }
}
__global__ void k_min_eps(const float* __restrict__ eps, long long N, unsigned* out_bits) {
  float m = 3.0e38f;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N; t += (long long)gridDim.x * blockDim.x) {
    const float e = eps[t];
    m = (e == e) ? fminf(m, e) : -1.0f;
  }
  m = fmaxf(m, 0.0f);   // negative / NaN -> 0 (fails the >= 1 check); keeps the uint ordering valid
  const unsigned r = __reduce_min_sync(0xffffffffu, __float_as_uint(m));
  if ((threadIdx.x & 31) == 0) atomicMin(out_bits, r);
}

// grad_eps = -(1/eps)^2 * S * acc  over the design box (row R3, end of DESIGN.md R9), evaluated in f64
__global__ void k_grad_finalize(const __grid_constant__ Dev d, const float* __restrict__ eps, float* __restrict__ out) {
  const int ey = d.dhi[1] - d.dlo[1], ez = d.dhi[2] - d.dlo[2];
  const long long cells = (long long)(d.dhi[0] - d.dlo[0]) * ey * ez;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= cells) return;
  const int kk = (int)(t % ez), jj = (int)((t / ez) % ey), ii = (int)(t / ((long long)ez * ey));
  const long long q = ((long long)(d.dlo[0] + ii) * d.n[1] + (d.dlo[1] + jj)) * d.n[2] + (d.dlo[2] + kk);
  const double ie = 1.0 / (double)eps[q];
  out[t] = (float)(-(ie * ie) * (double)d.S * d.acc[t]);
}

// ---- stand-alone codec kernels (same device functions as above) ----
__global__ void k_codec_amax(const float* __restrict__ x, size_t n, unsigned* out_bits) {
  unsigned m = 0;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x)
    m = max(m, __float_as_uint(fabsf(x[t])));
  m = __reduce_max_sync(0xffffffffu, m);
  if ((threadIdx.x & 31) == 0) atomicMax(out_bits, m);
}
template <int DT>
__global__ void k_codec_encode(const float* __restrict__ x, size_t n, void* codes, float* scale, const unsigned* amax_bits) {
  typedef typename Codec<DT>::code_t code_t;
  float inv = 1.0f, sc = 1.0f;
  if (DT == DT_E4M3S) {
    const float amax = __uint_as_float(*amax_bits);
    inv = amax > 0.0f ? 448.0f / amax : 0.0f;
    sc = amax > 0.0f ? amax / 448.0f : 0.0f;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *scale = sc;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x)
    reinterpret_cast<code_t*>(codes)[t] = Codec<DT>::enc(x[t], inv);
}
// DT_MX32: codes[n] followed by ceil(n/32) scale bytes in the same buffer (the slot convention); one warp per block
__global__ void k_codec_encode_mx(const float* __restrict__ x, size_t n, unsigned char* codes) {
  const size_t nblk = (n + 31) / 32;
  const int lane = threadIdx.x & 31;
  for (size_t b = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; b < nblk; b += ((size_t)gridDim.x * blockDim.x) >> 5) {
    const size_t t = b * 32 + lane;
    const float v = t < n ? x[t] : 0.0f;
    const int X = mx_exponent(__reduce_max_sync(0xffffffffu, __float_as_uint(fabsf(v))));
    if (t < n) codes[t] = Codec<DT_MX32>::enc(v, mx_pow2(-X));
    if (lane == 0) codes[n + b] = (unsigned char)(X + 127);
  }
}
struct FetchArgs {
  const void* codes[4];
  float scales[4];
};
template <int DT>
__global__ void k_codec_fetch(const __grid_constant__ FetchArgs a, int mode, int num, int den, size_t n, float* out) {
  typedef typename Codec<DT>::code_t code_t;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
    auto val = [&](int j) {
      const float sc = DT == DT_MX32 ? mx_scale(reinterpret_cast<const unsigned char*>(a.codes[j])[n + (t >> 5)]) : a.scales[j];
      return Codec<DT>::dec(reinterpret_cast<const code_t*>(a.codes[j])[t], sc);
    };
    const float v0 = val(1);
    float r = v0;
    if (mode == 1) r = lerp_value(v0, val(2), num, den);
    else if (mode == 2) r = cubic_value(val(0), v0, val(2), val(3), num, den);
    out[t] = r;
  }
}

}  // namespace fdtd
