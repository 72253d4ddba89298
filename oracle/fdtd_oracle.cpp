// oracle/fdtd_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this.  It shares no code with the CUDA path under
// paper_2603_24027_b200/csrc/.
//
// A plain, slow CPU restatement of the hot path of arxiv/paper_2603_24027 ("Numerical field
// optimization for enhanced efficiency in time-reversible gradient computation of ... FDTD
// simulations"), templated on float / double:
//
//   * Yee leapfrog E/H updates with CPML slabs        (CPML = ref. 17)
//   * record of the six volume/PML interface slices,
//     cast to a smaller bit-width, every k-th step      (PAPER.md:35 bit-width, PAPER.md:47 subsampling)
//   * reverse run: invert the interior updates, cast the stored values back, linearly interpolate,
//     inject them at the interface slices, and carry the adjoint fields backwards
//                                                       ("begins at the final time step ...
//                                                        propagates backward", PAPER.md:35 inject, :47 interp)
//   * dL/d(eps) accumulated over the design box
//
// Everything the paper leaves open (staggering, normalisation, CPML constants, order of injection,
// rounding order) follows the readings R1..R19 listed in DESIGN.md; each function names the reading.
// No blocking, fusion or reordering: every phase is its own loop nest over the whole grid; OpenMP is
// applied to the outermost loop only.
//
// Pin status (see tests/test_oracle_*.py): Yee update -> discrete dispersion closed form; energy
// invariant; forward/reverse round trip; adjoint -> dot-product test and store-all back-propagation;
// gradient -> central finite differences (f64); codec -> exhaustive + torch / ml_dtypes / numpy casts;
// interpolation -> polynomial exactness and sinusoid error bound; dt -> the paper's printed value;
// tangential-only store (store_mode 1) -> inner interior back to state 0 and gradient = store-all back-propagation;
// micro-scaled e4m3 (dtype 5) -> ml_dtypes float8_e4m3fn / float8_e8m0fnu casts, error bound, scale equivariance.
// fetch path (slot choice of the cubic option, fall-back to linear on the first / last / short interval, exact return at
// stored steps) -> a run with Courant number 0 whose interface values are a known cubic polynomial in the step index
// (tests/test_oracle_codec.py::test_cubic_fetch_path_slot_choice_and_fallbacks).
// CPML constants: PARITY UNPINNED against the paper (it prints none); pinned only by "sigma=0 reduces
// to plain Yee" and a reflection bound.
// Edge / corner ownership at injection ("the lowest-numbered face that contains the cell wins", reading R7/R9; it only
// matters under per-slice scales, where two faces hold differently rounded copies of one cell): PARITY UNPINNED, a reading.
//
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <limits>
#include <omp.h>
#include <vector>

namespace {

// =====================================================================================================
// 1. Minifloat codec ("converting the recorded field values to smaller bit-widths";
//    PAPER.md:53 format list).  Value-level definition, reading R12/R13:
//    for x != 0:  e = max(floor(log2|x|), 1-bias),  q = 2^(e-mbits),  result = sign(x) * q * RNE(|x|/q);
//    above the largest finite value: IEEE flavours -> inf, "fn"/"fnuz" flavours -> NaN.
// =====================================================================================================
enum Flavour { IEEE = 0, FN = 1, FNUZ = 2 };
struct Fmt { int ebits, mbits, bias, flavour; };

// store dtype ids (0..3 are the product's; >= 10 are the paper's unscaled float8 flavours, oracle only)
// 5 = micro-scaled e4m3: blocks of 32 values share one power-of-two scale (SURVEY 8(f)-1 "finer scale granularity";
// DESIGN.md reading R20)
enum { DT_F32 = 0, DT_F16 = 1, DT_BF16 = 2, DT_E4M3_SCALED = 3, DT_NATIVE = 4, DT_E4M3_MX32 = 5,
       DT_E4M3B11FNUZ = 10, DT_E5M2FNUZ = 11, DT_E4M3FNUZ = 12, DT_E4M3 = 13, DT_E3M4 = 14, DT_E4M3FN = 15 };

bool fmt_of(int dtype, Fmt* f) {
  switch (dtype) {
    case DT_F16:         *f = {5, 10, 15, IEEE};  return true;
    case DT_BF16:        *f = {8, 7, 127, IEEE};  return true;
    case DT_E4M3_SCALED:
    case DT_E4M3_MX32:
    case DT_E4M3FN:      *f = {4, 3, 7, FN};      return true;
    case DT_E4M3B11FNUZ: *f = {4, 3, 11, FNUZ};   return true;
    case DT_E5M2FNUZ:    *f = {5, 2, 16, FNUZ};   return true;
    case DT_E4M3FNUZ:    *f = {4, 3, 8, FNUZ};    return true;
    case DT_E4M3:        *f = {4, 3, 7, IEEE};    return true;
    case DT_E3M4:        *f = {3, 4, 3, IEEE};    return true;
  }
  return false;
}
int elem_bytes(int dtype, int native_bytes) {
  if (dtype == DT_F32) return 4;
  if (dtype == DT_NATIVE) return native_bytes;
  if (dtype == DT_F16 || dtype == DT_BF16) return 2;
  return 1;
}

double fmt_max(const Fmt& f) {
  int emax_field = (1 << f.ebits) - 1;
  if (f.flavour == IEEE) return std::ldexp(2.0 - std::ldexp(1.0, -f.mbits), emax_field - 1 - f.bias);
  if (f.flavour == FN)   return std::ldexp(2.0 - std::ldexp(2.0, -f.mbits), emax_field - f.bias);  // mantissa all-ones is NaN
  return std::ldexp(2.0 - std::ldexp(1.0, -f.mbits), emax_field - f.bias);                          // FNUZ: every code finite
}

double fmt_decode(const Fmt& f, uint32_t code) {
  const int nb = 1 + f.ebits + f.mbits;
  const uint32_t sign = (code >> (nb - 1)) & 1u;
  const uint32_t ef = (code >> f.mbits) & ((1u << f.ebits) - 1u);
  const uint32_t mf = code & ((1u << f.mbits) - 1u);
  const uint32_t eall = (1u << f.ebits) - 1u, mall = (1u << f.mbits) - 1u;
  const double nan = std::numeric_limits<double>::quiet_NaN();
  if (f.flavour == FNUZ && sign && ef == 0 && mf == 0) return nan;
  if (f.flavour == FN && ef == eall && mf == mall) return nan;
  if (f.flavour == IEEE && ef == eall) {
    if (mf) return nan;
    return sign ? -INFINITY : INFINITY;
  }
  double v = (ef == 0) ? std::ldexp((double)mf, 1 - f.bias - f.mbits)
                       : std::ldexp(1.0 + std::ldexp((double)mf, -f.mbits), (int)ef - f.bias);
  return sign ? -v : v;
}

uint32_t fmt_encode(const Fmt& f, double x) {
  const int nb = 1 + f.ebits + f.mbits;
  const uint32_t eall = (1u << f.ebits) - 1u, mall = (1u << f.mbits) - 1u;
  const uint32_t sbit = std::signbit(x) ? (1u << (nb - 1)) : 0u;
  uint32_t nan_code, inf_code;
  if (f.flavour == FNUZ) { nan_code = 1u << (nb - 1); inf_code = nan_code; }
  else if (f.flavour == FN) { nan_code = sbit | (eall << f.mbits) | mall; inf_code = nan_code; }
  else { nan_code = sbit | (eall << f.mbits) | (1u << (f.mbits - 1)); inf_code = sbit | (eall << f.mbits); }
  if (std::isnan(x)) return nan_code;
  double a = std::fabs(x);
  if (std::isinf(a)) return inf_code;
  if (a == 0.0) return (f.flavour == FNUZ) ? 0u : sbit;
  int ex;  std::frexp(a, &ex);                      // a = m * 2^ex, m in [0.5,1)  =>  floor(log2 a) = ex-1
  int e = std::max(ex - 1, 1 - f.bias);
  double q = std::ldexp(1.0, e - f.mbits);
  double r = std::nearbyint(a / q);                 // default rounding mode: round-to-nearest-even; a/q exact
  double v = r * q;
  if (v > fmt_max(f)) return inf_code;
  if (v == 0.0) return (f.flavour == FNUZ) ? 0u : sbit;
  uint32_t ef, mf;
  double minnormal = std::ldexp(1.0, 1 - f.bias);
  if (v < minnormal) { ef = 0; mf = (uint32_t)std::ldexp(v, -(1 - f.bias - f.mbits)); }
  else {
    int ev;  std::frexp(v, &ev);  ev -= 1;
    ef = (uint32_t)(ev + f.bias);
    mf = (uint32_t)std::ldexp(std::ldexp(v, -ev) - 1.0, f.mbits);
  }
  return sbit | (ef << f.mbits) | mf;
}

void put_code(uint8_t* dst, size_t i, int eb, uint32_t c) {
  if (eb == 1) dst[i] = (uint8_t)c; else { uint16_t h = (uint16_t)c; std::memcpy(dst + 2 * i, &h, 2); }
}
uint32_t get_code(const uint8_t* src, size_t i, int eb) {
  if (eb == 1) return src[i];
  uint16_t h;  std::memcpy(&h, src + 2 * i, 2);  return h;
}

// Encode one slice of f32 values.  DT_E4M3_SCALED follows DESIGN.md reading R13/R14:
// amax = max|x|; inv = amax>0 ? 448/amax : 0; code = e4m3fn_rne(clamp(fl(x*inv), -448, 448));
// scale = amax>0 ? amax/448 : 0  (all f32, round-to-nearest).
void encode_slice(int dtype, const float* x, size_t n, uint8_t* out, float* scale) {
  *scale = 1.0f;
  if (dtype == DT_F32) { std::memcpy(out, x, 4 * n); return; }
  Fmt f;  fmt_of(dtype, &f);
  const int eb = elem_bytes(dtype, 4);
  if (dtype == DT_E4M3_SCALED) {
    float amax = 0.0f;
    for (size_t i = 0; i < n; ++i) amax = std::max(amax, std::fabs(x[i]));
    float inv = (amax > 0.0f) ? 448.0f / amax : 0.0f;
    *scale = (amax > 0.0f) ? amax / 448.0f : 0.0f;
    for (size_t i = 0; i < n; ++i) {
      float y = x[i] * inv;
      y = std::min(448.0f, std::max(-448.0f, y));
      put_code(out, i, eb, fmt_encode(f, (double)y));
    }
    return;
  }
  for (size_t i = 0; i < n; ++i) put_code(out, i, eb, fmt_encode(f, (double)x[i]));
}

// Micro-scaled e4m3 (DT_E4M3_MX32; PAPER.md:35 cast to 8 bits, SURVEY 8(f)-1 finer scale granularity; reading R20).
// The slice is cut into blocks of 32 consecutive values (the last one may be shorter).  Per block:
//   amax = max|x|;  X = the smallest integer with amax * 2^-X <= 448 (e4m3's largest value), clamped to [-127, 127]
//   (amax = 0 -> X = -127), so the block maximum lands in (224, 448] and nothing is ever clipped;
//   code_i = e4m3fn_rne(clamp(x_i * 2^-X, -448, 448));  the block scale is stored as one byte X + 127.
// Decoding: value = e4m3fn(code) * 2^X.  Both multiplications are by powers of two and exact.
const int MX_BLOCK = 32;
size_t mx_blocks(size_t n) { return (n + MX_BLOCK - 1) / MX_BLOCK; }
int mx_block_exponent(const float* x, size_t n) {
  float amax = 0.0f;
  for (size_t i = 0; i < n; ++i) amax = std::max(amax, std::fabs(x[i]));
  if (!(amax > 0.0f)) return -127;
  int ex;  std::frexp((double)amax, &ex);            // amax = m * 2^ex, m in [0.5,1)  =>  floor(log2 amax) = ex-1
  int X = ex - 1 - 8;                                // 8 = exponent of e4m3's top binade [256, 512)
  if (std::ldexp((double)amax, -X) > 448.0) X += 1;  // the top binade ends at 448
  return std::min(127, std::max(-127, X));
}
void encode_slice_mx(const float* x, size_t n, uint8_t* codes, uint8_t* bscale) {
  Fmt f;  fmt_of(DT_E4M3_MX32, &f);
  for (size_t b = 0; b < mx_blocks(n); ++b) {
    const size_t i0 = b * MX_BLOCK, i1 = std::min(n, i0 + MX_BLOCK);
    const int X = mx_block_exponent(x + i0, i1 - i0);
    bscale[b] = (uint8_t)(X + 127);
    for (size_t i = i0; i < i1; ++i) {
      double y = std::ldexp((double)x[i], -X);
      y = std::min(448.0, std::max(-448.0, y));
      codes[i] = (uint8_t)fmt_encode(f, y);
    }
  }
}
float decode_value_mx(const uint8_t* codes, const uint8_t* bscale, size_t i) {
  Fmt f;  fmt_of(DT_E4M3_MX32, &f);
  return (float)std::ldexp(fmt_decode(f, codes[i]), (int)bscale[i / MX_BLOCK] - 127);
}

// "We convert the stored values back to the larger bit-widths".
float decode_value(int dtype, const uint8_t* src, size_t i, float scale) {
  if (dtype == DT_F32) { float v; std::memcpy(&v, src + 4 * i, 4); return v; }
  Fmt f;  fmt_of(dtype, &f);
  float v = (float)fmt_decode(f, get_code(src, i, elem_bytes(dtype, 4)));   // exact: every format is a subset of f32
  if (dtype == DT_E4M3_SCALED) v = v * scale;
  return v;
}

// Temporal interpolation, PAPER.md:47 ("subsampling at every k-th time step and applying linear
// interpolation"); arithmetic = DESIGN.md reading R11.  X = float for the reduced dtypes, T for native.
template <class X> X lerp_value(X a, X b, int num, int den) {
  X w = (X)num / (X)den;
  return std::fma(w, b - a, a);
}
// 4-point Lagrange on uniformly spaced slots (cubic is BASELINE.json's optional extra, not the paper's).
template <class X> X cubic_value(X vm1, X v0, X v1, X v2, int num, int den) {
  X t = (X)num / (X)den;
  X wm1 = -t * (t - 1) * (t - 2) / 6;
  X w0 = (t + 1) * (t - 1) * (t - 2) / 2;
  X w1 = -(t + 1) * t * (t - 2) / 2;
  X w2 = (t + 1) * t * (t - 1) / 6;
  return (wm1 * vm1 + w0 * v0) + (w1 * v1 + w2 * v2);
}

// =====================================================================================================
// 2. The simulation
// =====================================================================================================
struct CpmlParams { double sigma_factor, kappa_max, alpha_max, grade_m; };

template <class T> struct Source {
  int comp, lo[3], hi[3];
  std::vector<T> amp;      // empty = 1
  std::vector<T> wave;     // wave[m-1] is added in step m
};
struct Box { int lo[3], hi[3]; size_t cells() const { return (size_t)(hi[0]-lo[0]) * (hi[1]-lo[1]) * (hi[2]-lo[2]); } };

struct Slot { int step; std::vector<uint8_t> data; float scale[36]; };

template <class T> struct Sim {
  int n[3], P;  size_t N, st[3];
  T S;                                   // Courant number c*dt/dx  (eq. 1)
  std::vector<T> eps, ce;                // ce = fl(S * fl(1/eps))   (reading R3)
  std::vector<T> E[3], H[3], psiE[3][2], psiH[3][2];
  std::vector<T> bE[3], cE[3], kE[3], bH[3], cH[3], kH[3];   // per-axis CPML tables; k* = 1/kappa - 1
  std::vector<Source<T>> src;
  bool has_design = false, has_monitor = false;  Box design, monitor;  unsigned mon_mask = 0;
  std::vector<T> mon_record;             // [nsteps][ncomp][box]
  // run state
  int nsteps = 0, k = 1, dtype = DT_F32;
  std::vector<Slot> slots;
  bool keep_all = false;  std::vector<std::vector<T>> all_states;   // store-all mode (plain definition of the gradient)
  // adjoint
  std::vector<T> lE[3], lH[3], lpsiE[3][2], lpsiH[3][2];

  size_t idx(int i, int j, int kk) const { return ((size_t)i * n[1] + j) * n[2] + kk; }
  bool slab(int a, int i) const { return P > 0 && (i < P || i >= n[a] - P); }
  bool interior(const int* c) const { for (int a = 0; a < 3; ++a) if (c[a] < P || c[a] >= n[a] - P) return false; return true; }
  bool inner(const int* c) const { for (int a = 0; a < 3; ++a) if (c[a] < P + 1 || c[a] >= n[a] - P - 1) return false; return true; }
  bool in_box(const Box& b, const int* c) const { for (int a = 0; a < 3; ++a) if (c[a] < b.lo[a] || c[a] >= b.hi[a]) return false; return true; }
  size_t box_index(const Box& b, const int* c) const {
    return ((size_t)(c[0]-b.lo[0]) * (b.hi[1]-b.lo[1]) + (c[1]-b.lo[1])) * (b.hi[2]-b.lo[2]) + (c[2]-b.lo[2]);
  }

  // ---- CPML coefficient tables (ref. 17; all constants are DESIGN.md reading R5 — the paper prints none) ----
  void build_tables(const CpmlParams& p) {
    for (int a = 0; a < 3; ++a) {
      int Na = n[a];
      bE[a].assign(Na, 0); cE[a].assign(Na, 0); kE[a].assign(Na, 0);
      bH[a].assign(Na, 0); cH[a].assign(Na, 0); kH[a].assign(Na, 0);
      if (P == 0) continue;
      double sigma_max = p.sigma_factor * (p.grade_m + 1.0) * (double)S;
      for (int i = 0; i < Na; ++i) {
        double rE = std::max(std::max((double)(P - i) / P, (double)(i - (Na - P)) / P), 0.0);
        double rH = std::max(std::max((P - i - 0.5) / P, (i + 0.5 - (Na - P)) / P), 0.0);
        for (int h = 0; h < 2; ++h) {
          double rho = h ? rH : rE;
          double b = 0, c = 0, kk = 0;
          if (rho > 0) {
            double sig = sigma_max * std::pow(rho, p.grade_m);
            double kap = 1.0 + (p.kappa_max - 1.0) * std::pow(rho, p.grade_m);
            double alp = p.alpha_max * (1.0 - rho);
            b = std::exp(-(sig / kap + alp));
            double den = sig * kap + kap * kap * alp;
            c = (den > 0) ? sig / den * (b - 1.0) : 0.0;
            kk = 1.0 / kap - 1.0;
          }
          (h ? bH : bE)[a][i] = (T)b;  (h ? cH : cE)[a][i] = (T)c;  (h ? kH : kE)[a][i] = (T)kk;
        }
      }
    }
  }

  void init(int nx, int ny, int nz, int P_, double S_, const double* eps_in, const CpmlParams& p) {
    n[0] = nx; n[1] = ny; n[2] = nz; P = P_;  N = (size_t)nx * ny * nz;
    st[0] = (size_t)ny * nz; st[1] = nz; st[2] = 1;
    S = (T)S_;
    eps.resize(N); ce.resize(N);
    for (size_t q = 0; q < N; ++q) { eps[q] = (T)eps_in[q];  T inv = (T)1 / eps[q];  ce[q] = S * inv; }
    build_tables(p);
    reset();
  }
  void reset() {
    for (int c = 0; c < 3; ++c) {
      E[c].assign(N, 0); H[c].assign(N, 0);
      for (int t = 0; t < 2; ++t) { psiE[c][t].assign(N, 0); psiH[c][t].assign(N, 0); }
    }
    slots.clear(); all_states.clear(); nsteps = 0;
  }

  // ---- forward E half-step (Yee, ref. 26; reading R1/R2 staggering; R3 canonical arithmetic) ----
  //   E_c += S*inv_eps*( d_a1^- H_b1 - d_a2^- H_b2 ),  a1=c+1,b1=c+2 (sign +);  a2=c+2,b2=c+1 (sign -)
  //   in the a-slab:  psi = b*psi + c*d ;  E_c += (+/-) S*inv_eps*( (1/kappa-1)*d + psi )
  //   tangential E on the three low walls is held at 0 (PEC).
  void step_E() {
    for (int c = 0; c < 3; ++c) {
      const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        if (cc[a1] == 0 || cc[a2] == 0) { E[c][q] = 0; continue; }
        T d1 = H[b1][q] - H[b1][q - st[a1]];
        T d2 = H[b2][q] - H[b2][q - st[a2]];
        T e = std::fma(ce[q], d1 - d2, E[c][q]);
        if (slab(a1, cc[a1])) {
          T ps = std::fma(bE[a1][cc[a1]], psiE[c][0][q], cE[a1][cc[a1]] * d1);
          psiE[c][0][q] = ps;
          e = std::fma(ce[q], std::fma(kE[a1][cc[a1]], d1, ps), e);
        }
        if (slab(a2, cc[a2])) {
          T ps = std::fma(bE[a2][cc[a2]], psiE[c][1][q], cE[a2][cc[a2]] * d2);
          psiE[c][1][q] = ps;
          e = std::fma(-ce[q], std::fma(kE[a2][cc[a2]], d2, ps), e);
        }
        E[c][q] = e;
      }
    }
  }
  // soft additive sources: E_c += amp * wave[m-1]   (reading R8; PAPER.md:51 has a plane-wave source, out of scope)
  void add_sources(int m, T sign) {
    for (auto& s : src) {
      Box b; for (int a = 0; a < 3; ++a) { b.lo[a] = s.lo[a]; b.hi[a] = s.hi[a]; }
      T w = s.wave[m - 1];
      for (int i = s.lo[0]; i < s.hi[0]; ++i) for (int j = s.lo[1]; j < s.hi[1]; ++j) for (int kk = s.lo[2]; kk < s.hi[2]; ++kk) {
        const int cc[3] = {i, j, kk};
        T amp = s.amp.empty() ? (T)1 : s.amp[box_index(b, cc)];
        T v = amp * w;
        E[s.comp][idx(i, j, kk)] += sign * v;
      }
    }
  }
  // ---- forward H half-step:  H_c -= S*( d_a1^+ E_b1 - d_a2^+ E_b2 ), ghost E[N] = 0 (PEC on the high walls) ----
  void step_H() {
    for (int c = 0; c < 3; ++c) {
      const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        T up1 = (cc[a1] + 1 < n[a1]) ? E[b1][q + st[a1]] : (T)0;
        T up2 = (cc[a2] + 1 < n[a2]) ? E[b2][q + st[a2]] : (T)0;
        T d1 = up1 - E[b1][q];
        T d2 = up2 - E[b2][q];
        T h = std::fma(-S, d1 - d2, H[c][q]);
        if (slab(a1, cc[a1])) {
          T ps = std::fma(bH[a1][cc[a1]], psiH[c][0][q], cH[a1][cc[a1]] * d1);
          psiH[c][0][q] = ps;
          h = std::fma(-S, std::fma(kH[a1][cc[a1]], d1, ps), h);
        }
        if (slab(a2, cc[a2])) {
          T ps = std::fma(bH[a2][cc[a2]], psiH[c][1][q], cH[a2][cc[a2]] * d2);
          psiH[c][1][q] = ps;
          h = std::fma(S, std::fma(kH[a2][cc[a2]], d2, ps), h);
        }
        H[c][q] = h;
      }
    }
  }

  // ---- interface slices ("interface slices between the simulation volume and PML"; reading R6/R7) ----
  // face f = 2*axis + side; plane index P (low) or n-P-1 (high); cross-section = interior extent of the other two axes.
  int M(int a) const { return n[a] - 2 * P; }
  size_t face_size(int f) const { int a = f / 2; return (size_t)M((a + 1) % 3) * M((a + 2) % 3); }
  // Which components a face stores.  store_mode 0 (reading R6): all six.  store_mode 1 ("tangential"): only
  // what the inner interior ever reads from the shell — the inverse-E update reads H on the LOW faces through d^-, and
  // only its two components tangential to the face; the inverse-H update reads E on the HIGH faces through d^+, again
  // the two tangential ones.  12 slices instead of 36; the shell itself is then not reconstructed.
  int store_mode = 0;
  bool stored(int f, int comp) const {
    if (store_mode == 0) return true;
    const int a = f / 2, side = f % 2;
    if (side == 0) return comp >= 3 && comp - 3 != a;
    return comp < 3 && comp != a;
  }
  int ncomp_stored(int f) const { int c = 0; for (int comp = 0; comp < 6; ++comp) c += stored(f, comp); return c; }
  int nslices() const { int c = 0; for (int f = 0; f < 6; ++f) c += ncomp_stored(f); return c; }
  size_t slot_values() const { size_t s = 0; for (int f = 0; f < 6; ++f) s += ncomp_stored(f) * face_size(f); return s; }
  // micro-scaled store: a slot is [codes: slot_values bytes][block scales: slot_blocks bytes]; the blocks of a slice follow
  // the slices' own order
  size_t face_blocks(int f) const { return mx_blocks(face_size(f)); }
  size_t slot_blocks() const { size_t s = 0; for (int f = 0; f < 6; ++f) s += ncomp_stored(f) * face_blocks(f); return s; }
  size_t block_offset(int f, int comp) const {
    size_t o = 0;
    for (int g = 0; g < f; ++g) o += ncomp_stored(g) * face_blocks(g);
    int rank = 0;
    for (int c = 0; c < comp; ++c) rank += stored(f, c);
    return o + rank * face_blocks(f);
  }
  size_t slice_offset(int f, int comp) const {
    size_t o = 0;
    for (int g = 0; g < f; ++g) o += ncomp_stored(g) * face_size(g);
    int rank = 0;
    for (int c = 0; c < comp; ++c) rank += stored(f, c);
    return o + rank * face_size(f);
  }
  // cell of element (u,v) of face f; (u,v) run over the two remaining axes in increasing axis order, v fastest
  size_t face_cell(int f, int u, int v) const {
    int a = f / 2, side = f % 2;  int c[3];
    int b0 = (a == 0) ? 1 : 0, b1 = (a == 2) ? 1 : 2;
    c[a] = side ? n[a] - P - 1 : P;  c[b0] = P + u;  c[b1] = P + v;
    return idx(c[0], c[1], c[2]);
  }
  int face_dim(int f, int which) const { int a = f / 2; int b0 = (a == 0) ? 1 : 0, b1 = (a == 2) ? 1 : 2; return M(which ? b1 : b0); }

  T* field(int comp) { return comp < 3 ? E[comp].data() : H[comp - 3].data(); }

  // record state m  (PAPER.md:35 cast to smaller bit-width; :47 every k-th step)
  void record(int m) {
    Slot s;  s.step = m;
    const int eb = elem_bytes(dtype, sizeof(T));
    s.data.assign(slot_values() * eb + (dtype == DT_E4M3_MX32 ? slot_blocks() : 0), 0);
    for (int f = 0; f < 6; ++f) for (int comp = 0; comp < 6; ++comp) {
      s.scale[f * 6 + comp] = 1.0f;
      if (!stored(f, comp)) continue;
      const size_t fs = face_size(f), off = slice_offset(f, comp);
      const int du = face_dim(f, 0), dv = face_dim(f, 1);
      const T* F = field(comp);
      s.scale[f * 6 + comp] = 1.0f;
      if (dtype == DT_NATIVE) {
        for (int u = 0; u < du; ++u) for (int v = 0; v < dv; ++v)
          std::memcpy(&s.data[(off + (size_t)u * dv + v) * eb], &F[face_cell(f, u, v)], eb);
      } else {
        std::vector<float> tmp(fs);
        for (int u = 0; u < du; ++u) for (int v = 0; v < dv; ++v) tmp[(size_t)u * dv + v] = (float)F[face_cell(f, u, v)];
        if (dtype == DT_E4M3_MX32) encode_slice_mx(tmp.data(), fs, &s.data[off], &s.data[slot_values() + block_offset(f, comp)]);
        else encode_slice(dtype, tmp.data(), fs, &s.data[off * eb], &s.scale[f * 6 + comp]);
      }
    }
    slots.push_back(std::move(s));
  }

  // fetch the shell value of (face f, comp, element e) for state nstate (reading R10/R11)
  template <class X> X slot_value(const Slot& s, int f, int comp, size_t e) const {
    size_t off = slice_offset(f, comp);
    if (dtype == DT_NATIVE) { T v; std::memcpy(&v, &s.data[(off + e) * sizeof(T)], sizeof(T)); return (X)v; }
    if (dtype == DT_E4M3_MX32) return (X)decode_value_mx(&s.data[off], &s.data[slot_values() + block_offset(f, comp)], e);
    return (X)decode_value(dtype, &s.data[off * elem_bytes(dtype, 4)], e, s.scale[f * 6 + comp]);
  }
  template <class X> X fetch_x(int nstate, int f, int comp, size_t e, int interp) const {
    int j0 = nstate / k;
    if (nstate == nsteps) return slot_value<X>(slots.back(), f, comp, e);
    int m0 = j0 * k;
    const Slot& s0 = slots[j0];
    if (nstate == m0) return slot_value<X>(s0, f, comp, e);
    const Slot& s1 = slots[j0 + 1];
    int m1 = s1.step;
    X a = slot_value<X>(s0, f, comp, e), b = slot_value<X>(s1, f, comp, e);
    bool cubic_ok = interp == 1 && j0 >= 1 && (size_t)(j0 + 2) < slots.size() && m1 - m0 == k && slots[j0 + 2].step - m1 == k;
    if (cubic_ok) {
      X vm1 = slot_value<X>(slots[j0 - 1], f, comp, e), v2 = slot_value<X>(slots[j0 + 2], f, comp, e);
      return cubic_value<X>(vm1, a, b, v2, nstate - m0, k);
    }
    return lerp_value<X>(a, b, nstate - m0, m1 - m0);
  }
  T fetch(int nstate, int f, int comp, size_t e, int interp) const {
    if (dtype == DT_NATIVE) return fetch_x<T>(nstate, f, comp, e, interp);
    return (T)fetch_x<float>(nstate, f, comp, e, interp);     // all in f32, promoted afterwards (reading R11)
  }

  void write_monitor(int m) {
    if (!has_monitor) return;
    size_t bc = monitor.cells();  int ncomp = __builtin_popcount(mon_mask);
    size_t base = (size_t)(m - 1) * ncomp * bc;  int ci = 0;
    for (int comp = 0; comp < 6; ++comp) if (mon_mask >> comp & 1) {
      const T* F = field(comp);
      for (int i = monitor.lo[0]; i < monitor.hi[0]; ++i) for (int j = monitor.lo[1]; j < monitor.hi[1]; ++j) for (int kk = monitor.lo[2]; kk < monitor.hi[2]; ++kk) {
        const int cc[3] = {i, j, kk};
        mon_record[base + ci * bc + box_index(monitor, cc)] = F[idx(i, j, kk)];
      }
      ++ci;
    }
  }
  void snapshot() {
    std::vector<T> s(6 * N);
    for (int c = 0; c < 6; ++c) std::memcpy(&s[c * N], field(c), N * sizeof(T));
    all_states.push_back(std::move(s));
  }

  // forward run from the CURRENT state (normally zeros), state m = (E^m, H^{m+1/2})   (reading R2)
  void forward(int nsteps_, int dtype_, int k_) {
    nsteps = nsteps_; dtype = dtype_; k = k_;
    slots.clear(); all_states.clear();
    if (has_monitor) mon_record.assign((size_t)nsteps * __builtin_popcount(mon_mask) * monitor.cells(), 0);
    record(0);  if (keep_all) snapshot();
    for (int m = 1; m <= nsteps; ++m) {
      step_E();  add_sources(m, (T)1);  step_H();
      write_monitor(m);
      if (m % k == 0 || m == nsteps) record(m);
      if (keep_all) snapshot();
    }
  }
  size_t store_bytes() const {
    size_t b = 0;
    for (auto& s : slots) b += s.data.size() + (dtype == DT_E4M3_SCALED ? nslices() * 4 : 0);
    return b;
  }

  // ---------------------------------------------------------------------------------------------------
  // Reverse run  (step order = DESIGN.md reading R9)
  // ---------------------------------------------------------------------------------------------------
  void alloc_adjoint() {
    for (int c = 0; c < 3; ++c) {
      lE[c].assign(N, 0); lH[c].assign(N, 0);
      for (int t = 0; t < 2; ++t) { lpsiE[c][t].assign(N, 0); lpsiH[c][t].assign(N, 0); }
    }
  }
  void add_monitor_cotangent(int m, const double* dmon) {
    if (!has_monitor || !dmon) return;
    size_t bc = monitor.cells();  int ncomp = __builtin_popcount(mon_mask);
    size_t base = (size_t)(m - 1) * ncomp * bc;  int ci = 0;
    for (int comp = 0; comp < 6; ++comp) if (mon_mask >> comp & 1) {
      T* L = comp < 3 ? lE[comp].data() : lH[comp - 3].data();
      for (int i = monitor.lo[0]; i < monitor.hi[0]; ++i) for (int j = monitor.lo[1]; j < monitor.hi[1]; ++j) for (int kk = monitor.lo[2]; kk < monitor.hi[2]; ++kk) {
        const int cc[3] = {i, j, kk};
        L[idx(i, j, kk)] += (T)dmon[base + ci * bc + box_index(monitor, cc)];
      }
      ++ci;
    }
  }
  // inverse of step_H on the inner interior:  H^{m-1/2} = H^{m+1/2} + S*curl^+(E^m)
  void inverse_H() {
    for (int c = 0; c < 3; ++c) {
      const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
      #pragma omp parallel for schedule(static)
      for (int i = P + 1; i < n[0] - P - 1; ++i) for (int j = P + 1; j < n[1] - P - 1; ++j) for (int kk = P + 1; kk < n[2] - P - 1; ++kk) {
        const size_t q = idx(i, j, kk);
        T d1 = E[b1][q + st[a1]] - E[b1][q];
        T d2 = E[b2][q + st[a2]] - E[b2][q];
        H[c][q] = std::fma(S, d1 - d2, H[c][q]);
      }
    }
  }
  // transpose of step_H acting on (lE, lpsiH); lH passes through.
  //   per H term (c,a,b,s): g = -S*s*lH_c ; phi = lpsiH + g ; lE_b -= d_a^-( g/kappa + cH*phi ) ; lpsiH = bH*phi
  // written per output component e:  lE_e -= S*curl^-(lH)_e  (plain part), then the slab parts.
  void adjoint_H() {
    std::vector<T> W(N);
    for (int e = 0; e < 3; ++e) {
      const int a1 = (e + 1) % 3, b1 = (e + 2) % 3, a2 = (e + 2) % 3, b2 = (e + 1) % 3;
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        if (cc[a1] == 0 || cc[a2] == 0) { lE[e][q] = 0; continue; }       // PEC-masked nodes carry no cotangent
        T d1 = lH[b1][q] - lH[b1][q - st[a1]];
        T d2 = lH[b2][q] - lH[b2][q - st[a2]];
        lE[e][q] = std::fma(-S, d1 - d2, lE[e][q]);
      }
    }
    if (P == 0) return;
    // slab parts: H term (c, t): t=0 -> axis a=c+1, field b=c+2, sign +;  t=1 -> axis a=c+2, field b=c+1, sign -
    for (int c = 0; c < 3; ++c) for (int t = 0; t < 2; ++t) {
      const int a = t ? (c + 2) % 3 : (c + 1) % 3, b = t ? (c + 1) % 3 : (c + 2) % 3;
      const T coef = t ? S : -S;                                           // g = -S*s*lH_c
      const int other = t ? (c + 1) % 3 : (c + 2) % 3;                      // E_b is masked where idx[a]==0 or idx[other']==0
      (void)other;
      std::fill(W.begin(), W.end(), (T)0);
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        if (!slab(a, cc[a])) continue;
        T g = coef * lH[c][q];
        T phi = lpsiH[c][t][q] + g;
        W[q] = std::fma(cH[a][cc[a]], phi, kH[a][cc[a]] * g);
        lpsiH[c][t][q] = bH[a][cc[a]] * phi;
      }
      const int m1 = (b + 1) % 3, m2 = (b + 2) % 3;                         // mask axes of E_b
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        if (cc[m1] == 0 || cc[m2] == 0) continue;
        T lo = (cc[a] > 0) ? W[q - st[a]] : (T)0;
        lE[b][q] -= (W[q] - lo);
      }
    }
  }
  void inject(int nstate, bool magnetic, int interp) {
    // a cell on an edge or corner of the shell belongs to the lowest-index face that contains it (reading R9): only that
    // face writes it, and it writes the components it stores
    for (int f = 0; f < 6; ++f) for (int cidx = 0; cidx < 3; ++cidx) {
      int comp = magnetic ? 3 + cidx : cidx;  T* F = field(comp);
      if (!stored(f, comp)) continue;
      const int a = f / 2, side = f % 2;
      const int b0 = (a == 0) ? 1 : 0, b1 = (a == 2) ? 1 : 2;
      const int du = face_dim(f, 0), dv = face_dim(f, 1);
      for (int u = 0; u < du; ++u) for (int v = 0; v < dv; ++v) {
        int c[3];  c[a] = side ? n[a] - P - 1 : P;  c[b0] = P + u;  c[b1] = P + v;
        bool lower = side == 1 && P == n[a] - P - 1;
        for (int g = 0; g < a; ++g) lower = lower || c[g] == P || c[g] == n[g] - P - 1;
        if (lower) continue;
        F[face_cell(f, u, v)] = fetch(nstate, f, comp, (size_t)u * dv + v, interp);
      }
    }
  }
  bool on_shell(const int* c) const {
    if (!interior(c)) return false;
    for (int a = 0; a < 3; ++a) if (c[a] == P || c[a] == n[a] - P - 1) return true;
    return false;
  }
  // grad_inv accumulator, design ∩ inner interior:  acc += sum_c lE_c * curl^-(H^{m-1/2})_c   (S applied at the end)
  void grad_inner(std::vector<double>& acc) {
    if (!has_design) return;
    #pragma omp parallel for schedule(static)
    for (int i = design.lo[0]; i < design.hi[0]; ++i) for (int j = design.lo[1]; j < design.hi[1]; ++j) for (int kk = design.lo[2]; kk < design.hi[2]; ++kk) {
      const int cc[3] = {i, j, kk};
      if (!inner(cc)) continue;
      const size_t q = idx(i, j, kk);  double s = 0;
      for (int c = 0; c < 3; ++c) {
        const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
        T d1 = H[b1][q] - H[b1][q - st[a1]];
        T d2 = H[b2][q] - H[b2][q - st[a2]];
        T curl = d1 - d2;
        s += (double)lE[c][q] * (double)curl;
      }
      acc[box_index(design, cc)] += s;
    }
  }
  // inverse of step_E on the inner interior: E^{m-1} = (E^m - src) - S*inv_eps*curl^-(H^{m-1/2})
  void inverse_E() {
    for (int c = 0; c < 3; ++c) {
      const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
      #pragma omp parallel for schedule(static)
      for (int i = P + 1; i < n[0] - P - 1; ++i) for (int j = P + 1; j < n[1] - P - 1; ++j) for (int kk = P + 1; kk < n[2] - P - 1; ++kk) {
        const size_t q = idx(i, j, kk);
        T d1 = H[b1][q] - H[b1][q - st[a1]];
        T d2 = H[b2][q] - H[b2][q - st[a2]];
        E[c][q] = std::fma(-ce[q], d1 - d2, E[c][q]);
      }
    }
  }
  // inject E on the shell; shell ∩ design gradient in the dE form:  curl = (Eold - Enew)/ce   (reading R9)
  void inject_E_with_grad(int nstate, int interp, std::vector<double>& acc) {
    std::vector<T> old[3];
    if (has_design) for (int c = 0; c < 3; ++c) old[c] = E[c];
    inject(nstate, false, interp);
    if (!has_design) return;
    for (int i = design.lo[0]; i < design.hi[0]; ++i) for (int j = design.lo[1]; j < design.hi[1]; ++j) for (int kk = design.lo[2]; kk < design.hi[2]; ++kk) {
      const int cc[3] = {i, j, kk};
      if (!on_shell(cc)) continue;
      const size_t q = idx(i, j, kk);  double s = 0;
      for (int c = 0; c < 3; ++c) {
        T dE = old[c][q] - E[c][q];
        s += (double)lE[c][q] * ((double)dE / (double)ce[q]);
      }
      acc[box_index(design, cc)] += s;
    }
  }
  // transpose of step_E acting on (lH, lpsiE); lE passes through.
  //   per E term (c,a,b,s): g = S*inv_eps*s*lE_c ; phi = lpsiE + g ; lH_b -= d_a^+( g/kappa + cE*phi ) ; lpsiE = bE*phi
  // per output component h:  lH_h += curl^+(G)_h,  G_c = ce*lE_c ; then the slab parts.
  void adjoint_E() {
    std::vector<T> G[3], W(N);
    for (int c = 0; c < 3; ++c) { G[c].resize(N); for (size_t q = 0; q < N; ++q) G[c][q] = ce[q] * lE[c][q]; }
    for (int h = 0; h < 3; ++h) {
      const int a1 = (h + 1) % 3, b1 = (h + 2) % 3, a2 = (h + 2) % 3, b2 = (h + 1) % 3;
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        T up1 = (cc[a1] + 1 < n[a1]) ? G[b1][q + st[a1]] : (T)0;
        T up2 = (cc[a2] + 1 < n[a2]) ? G[b2][q + st[a2]] : (T)0;
        T d1 = up1 - G[b1][q];
        T d2 = up2 - G[b2][q];
        lH[h][q] = lH[h][q] + (d1 - d2);
      }
    }
    if (P == 0) return;
    for (int c = 0; c < 3; ++c) for (int t = 0; t < 2; ++t) {
      const int a = t ? (c + 2) % 3 : (c + 1) % 3, b = t ? (c + 1) % 3 : (c + 2) % 3;
      std::fill(W.begin(), W.end(), (T)0);
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        if (!slab(a, cc[a])) continue;
        if (cc[(c + 1) % 3] == 0 || cc[(c + 2) % 3] == 0) continue;        // PEC-masked E_c node: step_E skips it, so does its transpose
        T g = t ? -G[c][q] : G[c][q];
        T phi = lpsiE[c][t][q] + g;
        W[q] = std::fma(cE[a][cc[a]], phi, kE[a][cc[a]] * g);
        lpsiE[c][t][q] = bE[a][cc[a]] * phi;
      }
      #pragma omp parallel for schedule(static)
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        T up = (cc[a] + 1 < n[a]) ? W[q + st[a]] : (T)0;
        lH[b][q] -= (up - W[q]);
      }
    }
  }

  // mode 0: the method (time reversal + store).  mode 1: plain definition — every state comes from the
  // store-all snapshots (needs keep_all).  mode 2: pure time reversal, no injection (PEC box, P = 0 pin).
  void reverse(const double* dfinal, const double* dmon, int interp, int mode, double* grad_out) {
    alloc_adjoint();
    if (dfinal) for (int c = 0; c < 3; ++c) for (size_t q = 0; q < N; ++q) { lE[c][q] = (T)dfinal[c * N + q]; lH[c][q] = (T)dfinal[(3 + c) * N + q]; }
    std::vector<double> acc(has_design ? design.cells() : 0, 0.0);
    for (int m = nsteps; m >= 1; --m) {
      add_monitor_cotangent(m, dmon);
      if (mode == 1) {
        adjoint_H();
        const std::vector<T>& s = all_states[m - 1];
        for (int c = 0; c < 3; ++c) std::memcpy(H[c].data(), &s[(3 + c) * N], N * sizeof(T));
        grad_all_interior(acc);
        for (int c = 0; c < 3; ++c) std::memcpy(E[c].data(), &s[c * N], N * sizeof(T));
        adjoint_E();
        continue;
      }
      if (mode == 2) { inverse_H_all(); adjoint_H(); add_sources(m, (T)-1); inverse_E_all(); adjoint_E(); continue; }
      inverse_H();
      adjoint_H();
      inject(m - 1, true, interp);
      grad_inner(acc);
      add_sources(m, (T)-1);
      inverse_E();
      inject_E_with_grad(m - 1, interp, acc);
      adjoint_E();
    }
    if (grad_out && has_design) {
      size_t e = 0;
      for (int i = design.lo[0]; i < design.hi[0]; ++i) for (int j = design.lo[1]; j < design.hi[1]; ++j) for (int kk = design.lo[2]; kk < design.hi[2]; ++kk, ++e) {
        double ie = 1.0 / (double)eps[idx(i, j, kk)];
        grad_out[e] = -(ie * ie) * (double)S * acc[e];       // d(inv_eps)/d(eps) = -inv_eps^2
      }
    }
  }
  // plain-definition helper: gradient term on every design cell from the true H^{m-1/2} (design lies in the interior,
  // where step_E is the plain Yee formula)
  void grad_all_interior(std::vector<double>& acc) {
    if (!has_design) return;
    for (int i = design.lo[0]; i < design.hi[0]; ++i) for (int j = design.lo[1]; j < design.hi[1]; ++j) for (int kk = design.lo[2]; kk < design.hi[2]; ++kk) {
      const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);  double s = 0;
      for (int c = 0; c < 3; ++c) {
        const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
        T d1 = H[b1][q] - (cc[a1] > 0 ? H[b1][q - st[a1]] : (T)0);
        T d2 = H[b2][q] - (cc[a2] > 0 ? H[b2][q - st[a2]] : (T)0);
        s += (double)lE[c][q] * (double)(d1 - d2);
      }
      acc[box_index(design, cc)] += s;
    }
  }
  // whole-grid inverses for the P = 0 round-trip pin
  void inverse_H_all() {
    for (int c = 0; c < 3; ++c) {
      const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        T up1 = (cc[a1] + 1 < n[a1]) ? E[b1][q + st[a1]] : (T)0;
        T up2 = (cc[a2] + 1 < n[a2]) ? E[b2][q + st[a2]] : (T)0;
        H[c][q] = std::fma(S, (up1 - E[b1][q]) - (up2 - E[b2][q]), H[c][q]);
      }
    }
  }
  void inverse_E_all() {
    for (int c = 0; c < 3; ++c) {
      const int a1 = (c + 1) % 3, b1 = (c + 2) % 3, a2 = (c + 2) % 3, b2 = (c + 1) % 3;
      for (int i = 0; i < n[0]; ++i) for (int j = 0; j < n[1]; ++j) for (int kk = 0; kk < n[2]; ++kk) {
        const int cc[3] = {i, j, kk};  const size_t q = idx(i, j, kk);
        if (cc[a1] == 0 || cc[a2] == 0) continue;
        T d1 = H[b1][q] - H[b1][q - st[a1]];
        T d2 = H[b2][q] - H[b2][q - st[a2]];
        E[c][q] = std::fma(-ce[q], d1 - d2, E[c][q]);
      }
    }
  }
};

template <class T> void add_source_t(Sim<T>& s, int comp, const int* lo, const int* hi, const double* amp, const double* wave, int nwave) {
  Source<T> q;  q.comp = comp;  size_t cells = 1;
  for (int a = 0; a < 3; ++a) { q.lo[a] = lo[a]; q.hi[a] = hi[a]; cells *= (size_t)(hi[a] - lo[a]); }
  if (amp) { q.amp.resize(cells); for (size_t i = 0; i < cells; ++i) q.amp[i] = (T)amp[i]; }
  q.wave.resize(nwave);  for (int i = 0; i < nwave; ++i) q.wave[i] = (T)wave[i];
  s.src.push_back(std::move(q));
}
template <class T> void get_fields_t(Sim<T>& s, double* out) {
  for (int c = 0; c < 6; ++c) { const T* F = s.field(c); for (size_t q = 0; q < s.N; ++q) out[c * s.N + q] = (double)F[q]; }
}
template <class T> void set_fields_t(Sim<T>& s, const double* in) {
  for (int c = 0; c < 6; ++c) { T* F = s.field(c); for (size_t q = 0; q < s.N; ++q) F[q] = (T)in[c * s.N + q]; }
}
template <class T> void get_adjoint_t(Sim<T>& s, double* out) {
  for (int c = 0; c < 3; ++c) for (size_t q = 0; q < s.N; ++q) { out[c * s.N + q] = (double)s.lE[c][q]; out[(3 + c) * s.N + q] = (double)s.lH[c][q]; }
}
template <class T> void get_monitor_t(Sim<T>& s, double* out) { for (size_t i = 0; i < s.mon_record.size(); ++i) out[i] = (double)s.mon_record[i]; }

// One application of the forward step map and of its transpose on caller-supplied vectors, for the
// dot-product test  <A x, y> = <x, A^T y>.  Vector layout: [E(3N) | H(3N) | psiE(6N) | psiH(6N)].
template <class T> void load_state_t(Sim<T>& s, const double* v, bool adjoint) {
  const size_t N = s.N;
  if (adjoint) s.alloc_adjoint();
  for (int c = 0; c < 3; ++c) for (size_t q = 0; q < N; ++q) {
    (adjoint ? s.lE : s.E)[c][q] = (T)v[c * N + q];
    (adjoint ? s.lH : s.H)[c][q] = (T)v[(3 + c) * N + q];
    for (int t = 0; t < 2; ++t) {
      (adjoint ? s.lpsiE : s.psiE)[c][t][q] = (T)v[(6 + 2 * c + t) * N + q];
      (adjoint ? s.lpsiH : s.psiH)[c][t][q] = (T)v[(12 + 2 * c + t) * N + q];
    }
  }
}
template <class T> void save_state_t(Sim<T>& s, double* v, bool adjoint) {
  const size_t N = s.N;
  for (int c = 0; c < 3; ++c) for (size_t q = 0; q < N; ++q) {
    v[c * N + q] = (double)(adjoint ? s.lE : s.E)[c][q];
    v[(3 + c) * N + q] = (double)(adjoint ? s.lH : s.H)[c][q];
    for (int t = 0; t < 2; ++t) {
      v[(6 + 2 * c + t) * N + q] = (double)(adjoint ? s.lpsiE : s.psiE)[c][t][q];
      v[(12 + 2 * c + t) * N + q] = (double)(adjoint ? s.lpsiH : s.psiH)[c][t][q];
    }
  }
}

struct Handle { int prec; Sim<float>* f; Sim<double>* d; };

}  // namespace

#define DISPATCH(h, expr) do { Handle* H_ = (Handle*)(h); if (H_->prec == 32) { auto& s = *H_->f; expr; } else { auto& s = *H_->d; expr; } } while (0)

extern "C" {

void* orc_create(int prec, int nx, int ny, int nz, int P, double S, const double* eps,
                 double sigma_factor, double kappa_max, double alpha_max, double grade_m) {
  Handle* h = new Handle{prec, nullptr, nullptr};
  CpmlParams p{sigma_factor, kappa_max, alpha_max, grade_m};
  if (prec == 32) { h->f = new Sim<float>();  h->f->init(nx, ny, nz, P, S, eps, p); }
  else            { h->d = new Sim<double>(); h->d->init(nx, ny, nz, P, S, eps, p); }
  return h;
}
void orc_destroy(void* h) { Handle* H_ = (Handle*)h; delete H_->f; delete H_->d; delete H_; }
void orc_reset(void* h) { DISPATCH(h, s.reset()); }
void orc_set_design(void* h, const int* lo, const int* hi) {
  DISPATCH(h, { s.has_design = true; for (int a = 0; a < 3; ++a) { s.design.lo[a] = lo[a]; s.design.hi[a] = hi[a]; } });
}
// 0 = all six components on every face (reading R6), 1 = tangential only; before forward
void orc_set_store_mode(void* h, int mode) { DISPATCH(h, s.store_mode = mode); }
void orc_set_monitor(void* h, const int* lo, const int* hi, unsigned mask) {
  DISPATCH(h, { s.has_monitor = true; s.mon_mask = mask; for (int a = 0; a < 3; ++a) { s.monitor.lo[a] = lo[a]; s.monitor.hi[a] = hi[a]; } });
}
void orc_clear_sources(void* h) { DISPATCH(h, s.src.clear()); }
void orc_add_source(void* h, int comp, const int* lo, const int* hi, const double* amp, const double* wave, int nwave) {
  DISPATCH(h, add_source_t(s, comp, lo, hi, amp, wave, nwave));
}
void orc_set_keep_all(void* h, int on) { DISPATCH(h, s.keep_all = on != 0); }
void orc_forward(void* h, int nsteps, int dtype, int k) { DISPATCH(h, s.forward(nsteps, dtype, k)); }
// mode: 0 = the method, 1 = plain definition from store-all snapshots, 2 = pure time reversal (no store)
void orc_reverse(void* h, const double* dfinal, const double* dmon, int interp, int mode, double* grad_out) {
  DISPATCH(h, s.reverse(dfinal, dmon, interp, mode, grad_out));
}
void orc_get_fields(void* h, double* out) { DISPATCH(h, get_fields_t(s, out)); }
void orc_set_fields(void* h, const double* in) { DISPATCH(h, set_fields_t(s, in)); }
void orc_get_adjoint(void* h, double* out) { DISPATCH(h, get_adjoint_t(s, out)); }
void orc_get_monitor(void* h, double* out) { DISPATCH(h, get_monitor_t(s, out)); }
size_t orc_monitor_size(void* h) { size_t r = 0; DISPATCH(h, r = s.mon_record.size()); return r; }
size_t orc_store_bytes(void* h) { size_t r = 0; DISPATCH(h, r = s.store_bytes()); return r; }
int orc_num_slots(void* h) { int r = 0; DISPATCH(h, r = (int)s.slots.size()); return r; }
size_t orc_slot_values(void* h) { size_t r = 0; DISPATCH(h, r = s.slot_values()); return r; }
int orc_slot_step(void* h, int j) { int r = 0; DISPATCH(h, r = s.slots[j].step); return r; }
void orc_get_slot(void* h, int j, uint8_t* data, float* scales) {
  DISPATCH(h, { std::memcpy(data, s.slots[j].data.data(), s.slots[j].data.size()); std::memcpy(scales, s.slots[j].scale, 36 * sizeof(float)); });
}
size_t orc_slot_bytes(void* h, int j) { size_t r = 0; DISPATCH(h, r = s.slots[j].data.size()); return r; }
size_t orc_block_offset(void* h, int face, int comp) { size_t r = 0; DISPATCH(h, r = s.block_offset(face, comp)); return r; }
size_t orc_slice_offset(void* h, int face, int comp) { size_t r = 0; DISPATCH(h, r = s.slice_offset(face, comp)); return r; }
size_t orc_face_size(void* h, int face) { size_t r = 0; DISPATCH(h, r = s.face_size(face)); return r; }
// value the reverse run would inject for (state, face, comp, element)
double orc_fetch(void* h, int nstate, int face, int comp, size_t e, int interp) { double r = 0; DISPATCH(h, r = (double)s.fetch(nstate, face, comp, e, interp)); return r; }
void orc_fetch_face(void* h, int nstate, int face, int comp, int interp, double* out) {
  DISPATCH(h, { size_t fs = s.face_size(face); for (size_t e = 0; e < fs; ++e) out[e] = (double)s.fetch(nstate, face, comp, e, interp); });
}
void orc_get_tables(void* h, int axis, double* out /* [6][n_axis]: bE cE kE bH cH kH */) {
  DISPATCH(h, { int Na = s.n[axis]; for (int i = 0; i < Na; ++i) { out[i] = s.bE[axis][i]; out[Na + i] = s.cE[axis][i]; out[2 * Na + i] = s.kE[axis][i];
                out[3 * Na + i] = s.bH[axis][i]; out[4 * Na + i] = s.cH[axis][i]; out[5 * Na + i] = s.kH[axis][i]; } });
}
// single-step operators for the dot-product test (vector layout: see load_state_t)
void orc_apply_step(void* h, const double* x, double* y) { DISPATCH(h, { load_state_t(s, x, false); s.step_E(); s.step_H(); save_state_t(s, y, false); }); }
void orc_apply_step_transpose(void* h, const double* y, double* x) { DISPATCH(h, { load_state_t(s, y, true); s.adjoint_H(); s.adjoint_E(); save_state_t(s, x, true); }); }

// OpenMP thread count used by the loops above (bench.py's cpu_baseline reports it)
void orc_set_threads(int n) { omp_set_num_threads(n); }
int orc_get_threads() { return omp_get_max_threads(); }

// ---- standalone codec entry points ----
int orc_elem_bytes(int dtype) { return elem_bytes(dtype, 4); }
void orc_encode(int dtype, const float* x, size_t n, uint8_t* out, float* scale) { encode_slice(dtype, x, n, out, scale); }
void orc_encode_mx(const float* x, size_t n, uint8_t* codes, uint8_t* bscale) { encode_slice_mx(x, n, codes, bscale); }
void orc_decode_mx(const uint8_t* codes, const uint8_t* bscale, size_t n, float* out) { for (size_t i = 0; i < n; ++i) out[i] = decode_value_mx(codes, bscale, i); }
void orc_decode(int dtype, const uint8_t* in, size_t n, float scale, float* out) { for (size_t i = 0; i < n; ++i) out[i] = decode_value(dtype, in, i, scale); }
double orc_decode_code(int dtype, unsigned code) { Fmt f; if (!fmt_of(dtype, &f)) return 0; return fmt_decode(f, code); }
unsigned orc_encode_value(int dtype, double x) { Fmt f; if (!fmt_of(dtype, &f)) return 0; return fmt_encode(f, x); }
double orc_format_max(int dtype) { Fmt f; if (!fmt_of(dtype, &f)) return 0; return fmt_max(f); }
float orc_lerp(float a, float b, int num, int den) { return lerp_value<float>(a, b, num, den); }
float orc_cubic(float vm1, float v0, float v1, float v2, int num, int den) { return cubic_value<float>(vm1, v0, v1, v2, num, den); }
double orc_lerp64(double a, double b, int num, int den) { return lerp_value<double>(a, b, num, den); }
double orc_cubic64(double vm1, double v0, double v1, double v2, int num, int den) { return cubic_value<double>(vm1, v0, v1, v2, num, den); }

}  // extern "C"
