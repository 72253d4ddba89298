// fdtd_api.cu — host side of libfdtd_b200: the C ABI declared in include/fdtd.h.
// Argument validation, workspace carving, CPML tables, launch sequencing (R2 forward order, R9 reverse
// order).  Every step of the path runs in the kernels of fdtd_stencil.cuh / fdtd_store.cuh; there is no CPU path.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/fdtd.h"
#include "../../include/fdtd_bench.h"
#include "fdtd_stencil.cuh"
#include "fdtd_store.cuh"
#include "fdtd_fused.cuh"

using namespace fdtd;

namespace {

constexpr int kMaxSources = 128;
constexpr size_t kAmpStageFloats = 1u << 20;
constexpr double kC0 = 299792458.0;

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Layout {
  size_t ce, E[3], H[3], E2[3], H2[3], pHz2[2], psiE[3][2], psiH[3][2], tab, step, scratch, srcdesc, waves, store, scales, amax;
  size_t lE[3], lH[3], lE2[3], lH2[3], lpsiE[2][3][2], lpsiH[2][3][2], acc;
  size_t eps_own, mon_stage, grad_stage, amp_stage;
  size_t store_cap;
  int slots_cap;
  size_t total;
  std::vector<std::pair<size_t, size_t>> guards;   // FDTD_WS_GUARD: (offset, bytes) of the guard band behind every sub-array
};
constexpr size_t kGuardBytes = 4096;
constexpr unsigned kWsGuard = 4u;   // FDTD_WS_GUARD (include/fdtd_bench.h)

}  // namespace

namespace {
struct Split {          // one half-step over an x range: lean region + complement boxes
  Region reg{};
  bool has_lean = false;
  bool rows = false;    // the lean launch is a ROW kernel that also covers the z-slab cells of its rows (no class-Z boxes)
  int nlo = 0, nhi = 0; // its z-slab groups per row below / above the lean z range
  BoxList boxes{};
  int x0 = 0, x1 = 0;
};
}  // namespace

struct fdtd_sim {
  int n[3] = {0, 0, 0};
  int P = 0;
  double dx = 0, dt = 0, Sd = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t cur = nullptr;          // stream the next LAUNCH goes to (fork / on / join)
  cudaStream_t aux[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaStream_t cap = nullptr;          // origin stream of graph captures (the caller's stream may be the legacy default)
  cudaEvent_t ev_fork = nullptr, ev_mid = nullptr, ev_join[4] = {nullptr, nullptr, nullptr, nullptr};
  bool parallel = false;               // auxiliary streams available
  std::vector<cudaGraphExec_t> dead_graphs;
  cudaGraphExec_t graph_cache[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // forward, fused forward, reverse, fused reverse, fully fused reverse
  mutable std::string err;
  const float* eps_dev = nullptr;
  bool eps_owned = false;              // eps_dev points into the workspace (fdtd_set_eps_host)
  double cpml[4] = {0.8, 1.0, 0.01, 3.0};
  bool has_design = false;
  int dlo[3] = {0, 0, 0}, dhi[3] = {0, 0, 0};
  bool has_mon = false;
  BoxDev mon{};
  float* mon_rec = nullptr;
  // workspace
  char* ws = nullptr;
  size_t ws_bytes = 0;
  int max_nsteps = 0, max_k = 1, max_dtype = 0;
  unsigned flags = 0;
  Layout L{};
  Dev d{};
  StoreDev st{};
  std::vector<float> tables_host;
  std::vector<SrcDev> src_host;
  bool src_overlap = false;         // two sources add to one cell of one component: applied one launch per source, in index order
  std::vector<float> waves_host;
  int nsrc = 0;
  // E/H buffer pair(s): fb[b][0..2] = E, fb[b][3..5] = H of buffer b; d.E / d.H always point at the current one (cb)
  float* fb[2][6] = {{nullptr}};
  int cb = 0;
  float* lb[2][6] = {{nullptr}};   // lambda_E / lambda_H buffer pair(s), as fb; d.lE / d.lH point at the current one (acb)
  int acb = 0;
  bool fa_debug = false;           // DEBUG: fused adjoint path without its marching kernel (slab kernels on the whole grid)
  int fuse_adj_mode = -1;          // fused adjoint (adjoint of H + adjoint of E in one marching pass): -1 auto, 0 never, 1 whenever possible
  float* pz[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // psi_H of the z axis per buffer: [b][0] H_x term, [b][1] H_y term
  bool fuse_za = false;    // ... and the adjoint marching kernel (k_fused_ap) applies too
  bool fuse_z = false;     // the fused forward path uses the whole-row marching kernel (k_fused_fp): no class-Z slab boxes
  bool can_fuse = false;   // second buffer present (V == 4, P >= 4)
  int fuse_mode = -1;      // -1 auto (by size), 0 never, 1 whenever possible
  int fuse_rev_mode = -1;  // the same for the reverse primal (inverse-H + inverse-E)
  int xseg = 0;            // planes per block of the fused marching kernels (0: chosen by fused_xseg)
  int xseg_rev = 0;        // ... of the reverse-run marching kernels (primal and adjoint), if it is to differ
  int sm_count = 148;      // multiprocessors of the device (fdtd_create)
  bool rows_auto = true;   // what fdtd_set_rows(-1) selects (by grid size, see fdtd_create)
  bool use_iz = true;      // fused reverse primal: k_fused_ip instead of k_fused_he<true>
  bool use_fz = true;      // fused forward path: whole-row marching kernel (k_fused_fp) instead of k_fused_he + class-Z slab boxes
  bool use_zf = true;      // vector path: the inverse kernels inject the interior cells of the two z faces (fdtd_stencil.cuh, ZF)
  bool use_rows = true;    // vector path: row kernels (lean cells + the z-slab cells of the same rows in one launch)
  int zalign = 0;          // z alignment (cells) of the lean regions, chosen at create: 32 (128-byte lines) on grids that stream
                           // from HBM, 16 on grids that live in L2 (more cells for the slower general kernels otherwise)
  int store_mode = 0;      // 0: six components per face (R6); 1: tangential only (fdtd_set_store_mode)
  int V = 1;    // z cells per thread of the lean kernels (4 when nz % 4 == 0 and P % 4 == 0, else 1)
  int VG = 1;   // ... of the general kernels (2 in vector mode)
  // lean regions and complement box lists of the four split half-steps: 0 fwd E, 1 fwd H, 2 adj H, 3 adj E
  Split split[8]{};   // + 4, 5: the slab kernels' E / H box lists of the fused forward path; 6, 7: adjoint-of-H / adjoint-of-E box
                      // lists of the fused adjoint path

  // run state
  int nsteps = 0, k = 1, dtype = 0;
  bool forward_done = false, state_final = false;
  bool use_graphs = true;
  unsigned long long launches = 0;
};

namespace {

fdtd_status fail(const fdtd_sim* s, fdtd_status code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (s) s->err = buf;
  return code;
}
#define CUDA_TRY(s, call)                                                                          \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(s, FDTD_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

long long face_size(const fdtd_sim* s, int f) {
  const int a = f / 2;
  return (long long)(s->n[(a + 1) % 3] - 2 * s->P) * (s->n[(a + 2) % 3] - 2 * s->P);
}
int face_comps(const fdtd_sim* s) { return s->store_mode == 1 ? 2 : 6; }      // stored components per face
int store_slices(const fdtd_sim* s) { return 6 * face_comps(s); }
long long slot_values(const fdtd_sim* s) {
  long long v = 0;
  for (int f = 0; f < 6; ++f) v += face_comps(s) * face_size(s, f);
  return v;
}
int elem_bytes_host(int dt) { return dt == DT_F32 ? 4 : ((dt == DT_F16 || dt == DT_BF16) ? 2 : 1); }
bool dtype_ok(int dt) { return (dt >= 0 && dt <= 3) || dt == DT_MX32 || (dt >= DT_E4M3B11FNUZ && dt <= DT_E3M4); }
// micro-scaled store (DT_MX32): one scale byte per block of 32 values of a slice, kept behind the slot's codes
long long face_blocks(const fdtd_sim* s, int f) { return (face_size(s, f) + 31) / 32; }
long long slot_blocks(const fdtd_sim* s) {
  long long b = 0;
  for (int f = 0; f < 6; ++f) b += face_comps(s) * face_blocks(s, f);
  return b;
}
size_t slot_bytes_host(const fdtd_sim* s, int dt) {
  return (size_t)slot_values(s) * elem_bytes_host(dt) + (dt == DT_MX32 ? (size_t)slot_blocks(s) : 0);
}
// run STMT with DT bound to the compile-time store dtype
#define FDTD_DT_SWITCH(dt, STMT)                                                   \
  switch (dt) {                                                                    \
    case DT_F32: { constexpr int DT = DT_F32; STMT; } break;                       \
    case DT_F16: { constexpr int DT = DT_F16; STMT; } break;                       \
    case DT_BF16: { constexpr int DT = DT_BF16; STMT; } break;                     \
    case DT_E4M3S: { constexpr int DT = DT_E4M3S; STMT; } break;                   \
    case DT_MX32: { constexpr int DT = DT_MX32; STMT; } break;                     \
    case DT_E4M3B11FNUZ: { constexpr int DT = DT_E4M3B11FNUZ; STMT; } break;       \
    case DT_E5M2FNUZ: { constexpr int DT = DT_E5M2FNUZ; STMT; } break;             \
    case DT_E4M3FNUZ: { constexpr int DT = DT_E4M3FNUZ; STMT; } break;             \
    case DT_E4M3: { constexpr int DT = DT_E4M3; STMT; } break;                     \
    default: { constexpr int DT = DT_E3M4; STMT; } break;                          \
  }
int num_slots(int nsteps, int k) { return nsteps / k + 1 + (nsteps % k ? 1 : 0); }
long long psi_elems(const fdtd_sim* s, int a) { return 2LL * s->P * s->n[(a + 1) % 3] * s->n[(a + 2) % 3]; }
long long design_cells(const fdtd_sim* s) {
  return s->has_design ? (long long)(s->dhi[0] - s->dlo[0]) * (s->dhi[1] - s->dlo[1]) * (s->dhi[2] - s->dlo[2]) : 0;
}
long long mon_floats_per_step(const fdtd_sim* s) {
  return s->has_mon ? (long long)s->mon.ncomp * (s->mon.hi[0] - s->mon.lo[0]) * (s->mon.hi[1] - s->mon.lo[1]) *
                          (s->mon.hi[2] - s->mon.lo[2])
                    : 0;
}

Layout make_layout(const fdtd_sim* s, int nsteps, int dtype, int k, unsigned flags) {
  Layout L{};
  size_t o = 0;
  const size_t N = (size_t)s->n[0] * s->n[1] * s->n[2];
  const bool guard = (flags & kWsGuard) != 0;
  auto take = [&](size_t bytes) {
    size_t r = o;
    o = align_up(o + std::max<size_t>(bytes, 4));
    if (guard) { L.guards.emplace_back(o, kGuardBytes); o += kGuardBytes; }
    return r;
  };
  L.ce = take(N * 4);
  for (int c = 0; c < 3; ++c) L.E[c] = take(N * 4);
  for (int c = 0; c < 3; ++c) L.H[c] = take(N * 4);
  if (s->V == 4 && s->P >= 4) {   // ping-pong partners of E and H for the fused marching kernels
    for (int c = 0; c < 3; ++c) L.E2[c] = take(N * 4);
    for (int c = 0; c < 3; ++c) L.H2[c] = take(N * 4);
    for (int t = 0; t < 2; ++t) L.pHz2[t] = take((size_t)psi_elems(s, 2) * 4);   // partners of psi_H of the z axis (k_fused_fp)
  }
  for (int c = 0; c < 3; ++c)
    for (int t = 0; t < 2; ++t) L.psiE[c][t] = take((size_t)psi_elems(s, (c + 1 + t) % 3) * 4);
  for (int c = 0; c < 3; ++c)
    for (int t = 0; t < 2; ++t) L.psiH[c][t] = take((size_t)psi_elems(s, (c + 1 + t) % 3) * 4);
  L.tab = take((size_t)6 * (s->n[0] + s->n[1] + s->n[2]) * 4);
  L.step = take(16);
  L.scratch = take(16);
  L.srcdesc = take(sizeof(SrcDev) * kMaxSources);
  L.waves = take((size_t)kMaxSources * nsteps * 4);
  const int slots = num_slots(nsteps, k);
  L.slots_cap = slots;
  L.store_cap = (size_t)slots * slot_bytes_host(s, dtype);
  L.store = take(L.store_cap);
  L.scales = take((size_t)slots * 36 * 4);
  L.amax = take((size_t)slots * 36 * 4);
  if (flags & FDTD_WS_REVERSE) {
    for (int c = 0; c < 3; ++c) L.lE[c] = take(N * 4);
    for (int c = 0; c < 3; ++c) L.lH[c] = take(N * 4);
    if (s->V == 4 && s->P >= 4) {   // ping-pong partners of lambda_E, lambda_H for the fused adjoint path
      for (int c = 0; c < 3; ++c) L.lE2[c] = take(N * 4);
      for (int c = 0; c < 3; ++c) L.lH2[c] = take(N * 4);
    }
    for (int b = 0; b < 2; ++b)
      for (int c = 0; c < 3; ++c)
        for (int t = 0; t < 2; ++t) {
          L.lpsiE[b][c][t] = take((size_t)psi_elems(s, (c + 1 + t) % 3) * 4);
          L.lpsiH[b][c][t] = take((size_t)psi_elems(s, (c + 1 + t) % 3) * 4);
        }
    L.acc = take((size_t)design_cells(s) * 8);
  }
  if (flags & FDTD_WS_HOST_IO) {
    L.eps_own = take(N * 4);
    L.mon_stage = take((size_t)mon_floats_per_step(s) * nsteps * 4);
    L.grad_stage = take((size_t)design_cells(s) * 4);
    L.amp_stage = take(kAmpStageFloats * 4);
  }
  L.total = o;
  return L;
}

// CPML coefficient tables (ref. 17; constants = DESIGN.md R5): per axis bE cE kE bH cH kH.
// E-type terms sit at integer depth, H-type terms at half-integer depth.  b = exp(-(sigma/kappa + alpha)),
// c = sigma/(sigma*kappa + kappa^2*alpha)*(b - 1), k = 1/kappa - 1; sigma, alpha per time step (dimensionless).
void build_tables(fdtd_sim* s) {
  const int tot = s->n[0] + s->n[1] + s->n[2];
  s->tables_host.assign((size_t)6 * tot, 0.0f);
  const int P = s->P;
  if (P == 0) return;
  const double sf = s->cpml[0], kmax = s->cpml[1], amax = s->cpml[2], gm = s->cpml[3];
  const double S = (double)(float)s->Sd;
  const double sigma_max = sf * (gm + 1.0) * S;
  size_t base = 0;
  for (int a = 0; a < 3; ++a) {
    const int Na = s->n[a];
    for (int i = 0; i < Na; ++i) {
      const double rhoE = std::max(std::max((double)(P - i) / P, (double)(i - (Na - P)) / P), 0.0);
      const double rhoH = std::max(std::max((P - i - 0.5) / P, (i + 0.5 - (Na - P)) / P), 0.0);
      for (int h = 0; h < 2; ++h) {
        const double rho = h ? rhoH : rhoE;
        double b = 0, c = 0, kk = 0;
        if (rho > 0) {
          const double g = std::pow(rho, gm);
          const double sig = sigma_max * g;
          const double kap = 1.0 + (kmax - 1.0) * g;
          const double alp = amax * (1.0 - rho);
          b = std::exp(-(sig / kap + alp));
          const double den = sig * kap + kap * kap * alp;
          c = den > 0 ? sig / den * (b - 1.0) : 0.0;
          kk = 1.0 / kap - 1.0;
        }
        s->tables_host[base + (size_t)(3 * h + 0) * Na + i] = (float)b;
        s->tables_host[base + (size_t)(3 * h + 1) * Na + i] = (float)c;
        s->tables_host[base + (size_t)(3 * h + 2) * Na + i] = (float)kk;
      }
    }
    base += (size_t)6 * Na;
  }
}

bool box_ok(const int lo[3], const int hi[3], const int inner_lo[3], const int inner_hi[3]) {
  for (int a = 0; a < 3; ++a)
    if (lo[a] < inner_lo[a] || hi[a] > inner_hi[a] || hi[a] <= lo[a]) return false;
  return true;
}
bool in_interior(const fdtd_sim* s, const int lo[3], const int hi[3]) {
  int ilo[3], ihi[3];
  for (int a = 0; a < 3; ++a) { ilo[a] = s->P; ihi[a] = s->n[a] - s->P; }
  return box_ok(lo, hi, ilo, ihi);
}
bool in_grid(const fdtd_sim* s, const int lo[3], const int hi[3]) {
  int ilo[3] = {0, 0, 0};
  return box_ok(lo, hi, ilo, s->n);
}

// x / d == __umulhi(x, mul) for all x <= xmax (checked here; d == 1 is handled in fast_div)
FastDiv make_fastdiv(unsigned d, unsigned xmax) {
  FastDiv f{0u, d};
  if (d <= 1) { f.d = 1; return f; }
  f.mul = (unsigned)((1ull << 32) / d) + 1u;
  for (unsigned x = 0; x <= xmax; ++x)
    if ((unsigned)(((unsigned long long)x * f.mul) >> 32) != x / d) { std::fprintf(stderr, "fdtd: fastdiv(%u) fails at %u\n", d, x); std::abort(); }
  return f;
}
unsigned make_ginv(int G) {
  const unsigned m = (65536u + (unsigned)G - 1u) / (unsigned)G;
  for (unsigned lane = 0; lane < 32; ++lane)
    if (((lane * m) >> 16) != lane / (unsigned)G) { std::fprintf(stderr, "fdtd: ginv(%d) fails\n", G); std::abort(); }
  return m;
}

// Lean region [lo, hi) of split half-step `which` and the disjoint boxes covering the rest of the grid.
Split make_split(const fdtd_sim* s, int which, int x0, int x1) {
  const int P = s->P, V = s->V, VG = s->VG;
  Split sp;
  sp.x0 = x0; sp.x1 = x1;
  Region full;
  for (int a = 0; a < 3; ++a) {
    const int n = s->n[a];
    int lo, hi;
    switch (which) {
      case 0: lo = std::max(P, 1); hi = n - P; break;                 // fwd E: needs the -1 neighbours, no PEC-masked node
      case 1: lo = P; hi = std::min(n - P, n - 1); break;             // fwd H: needs the +1 neighbours
      case 2: lo = P + 1; hi = n - P; break;                          // adj H: the -1 neighbour must not be a slab cell
      case 3: lo = P; hi = std::min(n - P - 1, n - 1); break;         // adj E: the +1 neighbour must not be a slab cell
      // fused forward path: the marching kernel stores [P+1, n-P); the slab kernels cover the rest plus the plain layers
      // whose values they hand to each other (fdtd_fused.cuh, forward_fused_step)
      case 4: lo = P + 1; hi = n - P; break;                          // fused-path E: layer P joins the slab boxes
      case 5: lo = P + 1; hi = n - P - 1; break;                      // fused-path H: layers P and n-P-1 join them
      // fused adjoint path: the marching kernel stores [P+1, n-P-1) in x and y (whole rows in z); the slab kernels cover the rest,
      // and their adjoint-of-H boxes also the layer P+1, whose new lambda_E their adjoint-of-E boxes read across the edge
      case 6: lo = P + 2; hi = n - P - 1; break;
      default: lo = P + 1; hi = n - P - 1; break;
    }
    if (a == 2 && which >= 4 && s->fuse_z) { lo = 0; hi = n; }   // whole-row marching kernel: z-slab cells ride on their rows
    if (which >= 6 && s->fa_debug) { lo = 0; hi = 0; }              // DEBUG: no marching kernel, the slab kernels take the whole grid
    else if (a == 2) {
      // z range of the lean region: whole groups of V cells, and (zalign > V) whole 128-byte lines, so that neither the lean
      // nor the z-slab kernels fetch half-used lines (a row of the lean region then starts and ends on a line boundary).
      // Row kernels stream whole rows anyway: groups of V cells only.
      const bool rows = which < 4 && V == 4 && s->use_rows;
      const int za = (which < 4 && !rows && s->zalign > V && n % s->zalign == 0) ? s->zalign : V;
      int lo2 = (lo + za - 1) / za * za, hi2 = hi / za * za;
      if (hi2 - lo2 < za) { lo2 = (lo + V - 1) / V * V; hi2 = hi / V * V; }
      lo = lo2; hi = hi2;
    }
    full.lo[a] = lo; full.hi[a] = hi;
  }
  const bool full_lean = full.hi[0] > full.lo[0] && full.hi[1] > full.lo[1] && full.hi[2] > full.lo[2];
  Region& r = sp.reg;
  r = full;
  r.lo[0] = std::max(full.lo[0], x0); r.hi[0] = std::min(full.hi[0], x1);
  sp.has_lean = full_lean && r.hi[0] > r.lo[0];
  BoxList& B = sp.boxes;
  B = BoxList{};
  auto add = [&](int cls, int bx0, int bx1, int y0, int y1, int z0, int z1) {
    bx0 = std::max(bx0, x0); bx1 = std::min(bx1, x1);
    if (bx1 <= bx0 || y1 <= y0 || z1 <= z0) return;
    const int b = B.nb++;
    B.lo[b][0] = bx0; B.hi[b][0] = bx1; B.lo[b][1] = y0; B.hi[b][1] = y1; B.lo[b][2] = z0; B.hi[b][2] = z1;
    B.cls[b] = cls;
    const int groups = (z1 - z0 + VG - 1) / VG;
    const int G = std::min(groups, 32), RW = 32 / G;
    B.G[b] = G; B.RW[b] = RW;
    B.ginv[b] = make_ginv(G);
    B.nbx[b] = (groups + G - 1) / G;
    B.rows[b] = (bx1 - bx0) * (y1 - y0);
    B.nby[b] = (B.rows[b] + TY * RW - 1) / (TY * RW);
    B.dnbx[b] = make_fastdiv((unsigned)B.nbx[b], (unsigned)B.nbx[b] * B.nby[b]);
    B.drow[b] = make_fastdiv((unsigned)(y1 - y0), (unsigned)(B.nby[b] * TY * RW));
    B.off[b + 1] = B.off[b] + B.nbx[b] * B.nby[b];
  };
  const int nx = s->n[0], ny = s->n[1], nz = s->n[2];
  // classes: the x range of the lean region holds no x-slab cell, no wall plane and (adjoint) no cell whose x
  // neighbour is a slab cell, so boxes confined to it need no x terms (CLS_Y); likewise y for CLS_Z
  if (!full_lean) { add(CLS_X, 0, nx, 0, ny, 0, nz); return sp; }
  add(CLS_X, 0, full.lo[0], 0, ny, 0, nz);
  add(CLS_X, full.hi[0], nx, 0, ny, 0, nz);
  add(CLS_Y, full.lo[0], full.hi[0], 0, full.lo[1], 0, nz);
  add(CLS_Y, full.lo[0], full.hi[0], full.hi[1], ny, 0, nz);
  if (which < 4 && V == 4 && s->use_rows && sp.has_lean && x0 <= full.lo[0] && x1 >= full.hi[0]) {
    // the row kernel takes the z-slab cells of the lean x-y range itself
    sp.rows = true;
    sp.nlo = full.lo[2] / 4;
    sp.nhi = (nz - full.hi[2]) / 4;
    return sp;
  }
  add(CLS_Z, full.lo[0], full.hi[0], full.lo[1], full.hi[1], 0, full.lo[2]);
  add(CLS_Z, full.lo[0], full.hi[0], full.lo[1], full.hi[1], full.hi[2], nz);
  return sp;
}
dim3 grid_lean(const fdtd_sim* s, const Region& r) {
  return dim3((unsigned)((r.hi[2] - r.lo[2] + 32 * s->V - 1) / (32 * s->V)), (unsigned)((r.hi[1] - r.lo[1] + TY - 1) / TY),
              (unsigned)(r.hi[0] - r.lo[0]));
}
bool grid_inner(const fdtd_sim* s, dim3* g) {
  const int P = s->P, V = s->V;
  const int klo = P + 1, khi = s->n[2] - P - 1, rows = s->n[1] - 2 * P - 2, planes = s->n[0] - 2 * P - 2;
  if (khi <= klo || rows <= 0 || planes <= 0) return false;
  const int kg0 = (klo / V) * V;
  const int groups = (khi - kg0 + V - 1) / V;
  *g = dim3((unsigned)((groups + 31) / 32), (unsigned)((rows + TY - 1) / TY), (unsigned)planes);
  return true;
}

void set_cur(fdtd_sim* s, int b) {
  s->cb = b;
  for (int c = 0; c < 3; ++c) { s->d.E[c] = s->fb[b][c]; s->d.H[c] = s->fb[b][3 + c]; }
  // psi_H of the z axis is ping-ponged with the fields only where the whole-row marching kernel runs (fuse_z); everywhere else the
  // slab kernels update it in place, in buffer 0's arrays
  const int pb = s->fuse_z ? b : 0;
  if (s->pz[pb][0]) { s->d.psiH[0][1] = s->pz[pb][0]; s->d.psiH[1][0] = s->pz[pb][1]; }
}

void set_cur_adj(fdtd_sim* s, int b) {
  s->acb = b;
  for (int c = 0; c < 3; ++c) { s->d.lE[c] = s->lb[b][c]; s->d.lH[c] = s->lb[b][3 + c]; }
}

#define LAUNCH(s, kern, grid, block, ...)            \
  do {                                               \
    kern<<<grid, block, 0, (s)->cur>>>(__VA_ARGS__); \
    ++(s)->launches;                                 \
  } while (0)

// ---- fork / join over the handle's auxiliary streams: kernels of one phase that touch disjoint data run side by
// side.  Under stream capture these become parallel branches of the CUDA graph; outside they are plain streams. ----
void fork(fdtd_sim* s, int branches) {
  s->cur = s->stream;
  if (!s->parallel) return;
  cudaEventRecord(s->ev_fork, s->stream);
  for (int b = 1; b < branches; ++b) cudaStreamWaitEvent(s->aux[b - 1], s->ev_fork, 0);
}
void on(fdtd_sim* s, int branch) { s->cur = (s->parallel && branch > 0) ? s->aux[branch - 1] : s->stream; }
void join(fdtd_sim* s, int branches) {
  s->cur = s->stream;
  if (!s->parallel) return;
  for (int b = 1; b < branches; ++b) {
    cudaEventRecord(s->ev_join[b - 1], s->aux[b - 1]);
    cudaStreamWaitEvent(s->stream, s->ev_join[b - 1], 0);
  }
}

void launch_lean(fdtd_sim* s, int which, const Split& sp, int pb = 0) {
  if (!sp.has_lean) return;
  const dim3 b(32, TY);
  const dim3 g = grid_lean(s, sp.reg);
  const Region& r = sp.reg;
  if (sp.rows) {
    RowArgs ra;
    ra.reg = r; ra.nlo = sp.nlo; ra.nhi = sp.nhi;
    ra.ztiles = (int)g.x;
    ra.ns = (ROW_RS * (sp.nlo + sp.nhi) + 32 * TY - 1) / (32 * TY);
    const dim3 gr((unsigned)((ROW_RS / TY) * ra.ztiles + ra.ns), (unsigned)((r.hi[1] - r.lo[1] + ROW_RS - 1) / ROW_RS), g.z);
    switch (which) {
      case 0: LAUNCH(s, k_row<0>, gr, b, s->d, ra, pb); break;
      case 1: LAUNCH(s, k_row<1>, gr, b, s->d, ra, pb); break;
      case 2: LAUNCH(s, k_row<2>, gr, b, s->d, ra, pb); break;
      default: LAUNCH(s, k_row<3>, gr, b, s->d, ra, pb);
    }
    return;
  }
  if (s->V == 4) {
    switch (which) {
      case 0: LAUNCH(s, (k_lean_curlm<4, false>), g, b, s->d, r); break;
      case 1: LAUNCH(s, k_lean_h<4>, g, b, s->d, r); break;
      case 2: LAUNCH(s, (k_lean_curlm<4, true>), g, b, s->d, r); break;
      default: LAUNCH(s, k_lean_adj_e<4>, g, b, s->d, r);
    }
  } else {
    switch (which) {
      case 0: LAUNCH(s, (k_lean_curlm<1, false>), g, b, s->d, r); break;
      case 1: LAUNCH(s, k_lean_h<1>, g, b, s->d, r); break;
      case 2: LAUNCH(s, (k_lean_curlm<1, true>), g, b, s->d, r); break;
      default: LAUNCH(s, k_lean_adj_e<1>, g, b, s->d, r);
    }
  }
}
FieldIO io_inplace(const fdtd_sim* s, int which) {   // which: 0 = E half-step, 1 = H half-step
  FieldIO io;
  for (int c = 0; c < 3; ++c) { io.E[c] = s->d.E[c]; io.H[c] = s->d.H[c]; io.out[c] = which == 0 ? s->d.E[c] : s->d.H[c]; }
  io_psi_inplace(io, s->d);
  return io;
}
AdjIO adj_inplace(const fdtd_sim* s) {
  AdjIO io;
  for (int c = 0; c < 3; ++c) { io.lEin[c] = s->d.lE[c]; io.lH[c] = s->d.lH[c]; io.lEout[c] = s->d.lE[c]; io.lHout[c] = s->d.lH[c]; }
  return io;
}
void launch_gen(fdtd_sim* s, int which, int pb, const Split& sp, const FieldIO* iop = nullptr, const AdjIO* aop = nullptr) {
  const dim3 b(32, TY);
  const BoxList& B = sp.boxes;
  const FieldIO io = iop ? *iop : io_inplace(s, which == 1 ? 1 : 0);
  const AdjIO ao = aop ? *aop : adj_inplace(s);
  const unsigned g = (unsigned)B.off[B.nb];
  if (g == 0) return;
  if (s->VG == 4) {
    switch (which) {
      case 0: LAUNCH(s, k_gen_e<4>, g, b, s->d, B, io); break;
      case 1: LAUNCH(s, k_gen_h<4>, g, b, s->d, B, io); break;
      case 2: LAUNCH(s, k_gen_adj_h<4>, g, b, s->d, B, pb, ao); break;
      default: LAUNCH(s, k_gen_adj_e<4>, g, b, s->d, B, pb, ao);
    }
  } else if (s->VG == 2) {
    switch (which) {
      case 0: LAUNCH(s, k_gen_e<2>, g, b, s->d, B, io); break;
      case 1: LAUNCH(s, k_gen_h<2>, g, b, s->d, B, io); break;
      case 2: LAUNCH(s, k_gen_adj_h<2>, g, b, s->d, B, pb, ao); break;
      default: LAUNCH(s, k_gen_adj_e<2>, g, b, s->d, B, pb, ao);
    }
  } else {
    switch (which) {
      case 0: LAUNCH(s, k_gen_e<1>, g, b, s->d, B, io); break;
      case 1: LAUNCH(s, k_gen_h<1>, g, b, s->d, B, io); break;
      case 2: LAUNCH(s, k_gen_adj_h<1>, g, b, s->d, B, pb, ao); break;
      default: LAUNCH(s, k_gen_adj_e<1>, g, b, s->d, B, pb, ao);
    }
  }
}
// The four split half-steps: lean kernel on the plain cells + general kernel on the rest (disjoint writes).
void launch_lean(fdtd_sim* s, int which, int pb = 0) { launch_lean(s, which, s->split[which], pb); }
void launch_gen(fdtd_sim* s, int which, int pb) { launch_gen(s, which, pb, s->split[which]); }
void launch_split(fdtd_sim* s, int which, int pb) {
  launch_lean(s, which, pb);
  launch_gen(s, which, pb);
}
// The inverse kernels of the vector path also inject the interior cells of the two z faces (fdtd_stencil.cuh, ZF)
bool zface_fused(const fdtd_sim* s) { return s->V == 4 && s->use_zf; }
void launch_inv_h(fdtd_sim* s, int m_base, const int* step_dev, int interp) {
  dim3 gi;
  if (!grid_inner(s, &gi)) return;
  const dim3 b(32, TY);
  ZInj z;
  z.st = s->st; z.m_base = m_base; z.step_dev = step_dev; z.interp = interp;
  if (zface_fused(s)) { FDTD_DT_SWITCH(s->dtype, LAUNCH(s, (k_inv_h<4, DT, true>), gi, b, s->d, z)) }
  else if (s->V == 4) LAUNCH(s, (k_inv_h<4, DT_F32, false>), gi, b, s->d, z);
  else LAUNCH(s, (k_inv_h<1, DT_F32, false>), gi, b, s->d, z);
}
void launch_inv_e(fdtd_sim* s, int m_base, const int* step_dev, int interp) {
  dim3 gi;
  if (!grid_inner(s, &gi)) return;
  const dim3 b(32, TY);
  ZInj z;
  z.st = s->st; z.m_base = m_base; z.step_dev = step_dev; z.interp = interp;
  if (zface_fused(s)) { FDTD_DT_SWITCH(s->dtype, LAUNCH(s, (k_inv_e<4, DT, true>), gi, b, s->d, z)) }
  else if (s->V == 4) LAUNCH(s, (k_inv_e<4, DT_F32, false>), gi, b, s->d, z);
  else LAUNCH(s, (k_inv_e<1, DT_F32, false>), gi, b, s->d, z);
}
// design ∩ inner interior extents; false if empty
bool grad_extents(const fdtd_sim* s, int ext[3]) {
  if (!s->has_design) return false;
  for (int a = 0; a < 3; ++a) {
    ext[a] = std::min(s->dhi[a], s->n[a] - s->P - 1) - std::max(s->dlo[a], s->P + 1);
    if (ext[a] <= 0) return false;
  }
  return true;
}
void launch_grad(fdtd_sim* s) {
  int ext[3];
  if (!grad_extents(s, ext)) return;
  const long long cells = (long long)ext[0] * ext[1] * ext[2];
  LAUNCH(s, k_grad, (unsigned)((cells + 255) / 256), 256, s->d);
}
void launch_sources(fdtd_sim* s, int m_base, const int* step_dev, float sign, int x0 = 0, int x1 = 1 << 30, int buffer = -1) {
  if (s->nsrc == 0) return;
  bool any = false;
  for (int i = 0; i < s->nsrc; ++i) any = any || (s->src_host[i].lo[0] < x1 && s->src_host[i].hi[0] > x0);
  if (!any) return;
  long long maxc = 1;
  for (int i = 0; i < s->nsrc; ++i) {
    const SrcDev& q = s->src_host[i];
    maxc = std::max(maxc, (long long)(q.hi[0] - q.lo[0]) * (q.hi[1] - q.lo[1]) * (q.hi[2] - q.lo[2]));
  }
  const int threads = maxc >= 128 ? 128 : 32;
  const unsigned gx = (unsigned)std::min<long long>((maxc + threads - 1) / threads, 1024);
  Dev dd = s->d;
  if (buffer >= 0)
    for (int c = 0; c < 3; ++c) dd.E[c] = s->fb[buffer][c];
  const SrcDev* desc = reinterpret_cast<const SrcDev*>(s->ws + s->L.srcdesc);
  const float* waves = reinterpret_cast<const float*>(s->ws + s->L.waves);
  if (!s->src_overlap) {
    LAUNCH(s, k_sources, dim3(gx, (unsigned)s->nsrc), threads, dd, desc, waves, m_base, step_dev, sign, x0, x1);
    return;
  }
  // overlapping sources: float addition does not commute with itself twice over ((E + a) + b != (E + b) + a), and the order of
  // atomicAdd from concurrent blocks is not defined.  One launch per source, in index order — the order of the sum in R8.
  for (int i = 0; i < s->nsrc; ++i)
    if (s->src_host[i].lo[0] < x1 && s->src_host[i].hi[0] > x0)
      LAUNCH(s, k_sources, dim3(gx, 1), threads, dd, desc + i, waves, m_base, step_dev, sign, x0, x1);
}
void launch_box(fdtd_sim* s, const BoxDev& b, float* rec, int m_base, const int* step_dev, int mode, int half = 2) {
  if ((half == 0 && !(b.mask & 7u)) || (half == 1 && !(b.mask & 56u))) return;
  const long long tot = (long long)b.ncomp * (b.hi[0] - b.lo[0]) * (b.hi[1] - b.lo[1]) * (b.hi[2] - b.lo[2]);
  if (tot <= 0) return;
  LAUNCH(s, k_box, (unsigned)((tot + 255) / 256), 256, s->d, b, rec, m_base, step_dev, mode, half);
}
// half: 0 = E components, 1 = H components, 2 = all six
void launch_record(fdtd_sim* s, int m_base, const int* step_dev, int half) {
  const long long items = s->store_mode == 1 ? s->st.cell_off[6] * (half == 2 ? 2 : 1)   // 2 components on 3 of the 6 faces
                                             : s->st.cell_off[6] * (half == 2 ? 6 : 3);
  if (s->dtype == DT_MX32) {   // one warp per block of 32 values; the slices in the half are 'items / face cells' many
    const long long warps = s->st.blkc_off[6] * (items / s->st.cell_off[6]);
    LAUNCH(s, k_record_mx, (unsigned)((warps * 32 + 255) / 256), 256, s->d, s->st, m_base, step_dev, half);
    return;
  }
  const unsigned g = (unsigned)((items + 255) / 256);
  if (s->dtype == DT_E4M3S) LAUNCH(s, k_record_amax, g, 256, s->d, s->st, m_base, step_dev, half);
  FDTD_DT_SWITCH(s->dtype, LAUNCH(s, k_record<DT>, g, 256, s->d, s->st, m_base, step_dev, half))
}
// from / to: buffer that holds the shell E of state m / buffer that receives the injected values (-1 = the current one)
void launch_inject(fdtd_sim* s, int m_base, const int* step_dev, int magnetic, int interp, int from = -1, int to = -1) {
  // beside the two-kernel reverse primal of the vector path the z faces are injected by the inverse kernels themselves
  const int nfaces = (from < 0 && to < 0 && zface_fused(s)) ? 4 : 6;
  const unsigned g = (unsigned)((s->st.cell_off[nfaces] + 255) / 256);
  if (g == 0) return;
  InjIO io;
  for (int c = 0; c < 3; ++c) {
    io.Eold[c] = from < 0 ? s->d.E[c] : s->fb[from][c];
    io.Eout[c] = to < 0 ? s->d.E[c] : s->fb[to][c];
    io.Hout[c] = to < 0 ? s->d.H[c] : s->fb[to][3 + c];
  }
  FDTD_DT_SWITCH(s->dtype, LAUNCH(s, k_inject<DT>, g, 256, s->d, s->st, m_base, step_dev, magnetic, interp, io, nfaces))
}

// One forward step m-1 -> m (R2): E half-step (+CPML), sources, H half-step (+CPML), monitor, record.
// Phase E: {lean E then sources, general E, H halves of state m-1: record (if pending) and monitor row (H is read-only here)}.
// Phase H: {lean H, general H, E halves of state m: record (if due) and monitor row (E is read-only here)}.
// pending_h carries "state m-1 still needs its H half recorded" in and "state m ..." out; the monitor row of state m-1
// always has its H half pending (k_box skips state 0, which has no row).  No small kernel sits alone between phases.
bool sources_in_lean(const fdtd_sim* s, const Split& sp) {
  if (!sp.has_lean) return s->nsrc == 0;
  for (int i = 0; i < s->nsrc; ++i)
    for (int a = 0; a < 3; ++a)
      if (s->src_host[i].lo[a] < sp.reg.lo[a] || s->src_host[i].hi[a] > sp.reg.hi[a]) return false;
  return true;
}
void forward_step(fdtd_sim* s, int m_base, const int* step_dev, bool record, bool* pending_h) {
  const bool mon = s->has_mon && s->mon_rec;
  const bool src_inline = sources_in_lean(s, s->split[0]);
  fork(s, 3);
  on(s, 0); launch_lean(s, 0);
  if (src_inline) launch_sources(s, m_base, step_dev, 1.0f);
  on(s, 1); launch_gen(s, 0, 0);
  on(s, 2);
  if (*pending_h) launch_record(s, m_base - 1, step_dev, 1);
  if (mon) launch_box(s, s->mon, s->mon_rec, m_base - 1, step_dev, 0, 1);
  join(s, 3);
  if (!src_inline) launch_sources(s, m_base, step_dev, 1.0f);
  fork(s, 3);
  on(s, 0); launch_lean(s, 1);
  on(s, 1); launch_gen(s, 1, 0);
  on(s, 2);
  if (record) launch_record(s, m_base, step_dev, 0);
  if (mon) launch_box(s, s->mon, s->mon_rec, m_base, step_dev, 0, 0);
  join(s, 3);
  *pending_h = record;
}
// H halves of the final state that forward_step left pending
void forward_flush(fdtd_sim* s, int m, bool pending_h) {
  if (pending_h) launch_record(s, m, nullptr, 1);
  if (s->has_mon && s->mon_rec) launch_box(s, s->mon, s->mon_rec, m, nullptr, 0, 1);
}

// One reverse step m -> m-1 (R9), as two phases of mutually independent kernels:
//  1: {monitor cotangent then adjoint-H lean, adjoint-H general (after the cotangent), inverse-H (inner interior) then the
//      sources, inject H (shell)}
//  2: {adjoint-E lean, adjoint-E general, gradient + inverse-E (inner interior), inject E + shell gradient}
void reverse_step(fdtd_sim* s, int m_base, const int* step_dev, const float* dmon, int interp, int pb) {
  const bool cot = dmon && s->has_mon;
  fork(s, 4);
  on(s, 1);   // the general kernel is the long one of the phase: it is enqueued first
  if (cot) {
    launch_box(s, s->mon, const_cast<float*>(dmon), m_base, step_dev, 1);
    if (s->parallel) { cudaEventRecord(s->ev_mid, s->aux[0]); cudaStreamWaitEvent(s->stream, s->ev_mid, 0); }
  }
  launch_gen(s, 2, pb);
  on(s, 0); launch_lean(s, 2, pb);
  on(s, 2); launch_inv_h(s, m_base, step_dev, interp); launch_sources(s, m_base, step_dev, -1.0f);
  on(s, 3); launch_inject(s, m_base, step_dev, 1, interp);
  join(s, 4);
  fork(s, 5);
  on(s, 0); launch_lean(s, 3, pb);
  on(s, 1); launch_gen(s, 3, pb);
  on(s, 2); launch_inv_e(s, m_base, step_dev, interp);
  on(s, 3); launch_inject(s, m_base, step_dev, 0, interp);
  on(s, 4); launch_grad(s);   // reads H^{m-1/2} and lambda_E (read-only in this phase), adds to inner design cells only
  join(s, 5);
}

// ---- fused path (fdtd_fused.cuh): H half-step of step m and E half-step of step m+1 in one marching kernel ----
long long fused_tiles(const fdtd_sim* s, int xseg) {
  long long tiles = s->fuse_z ? (s->n[2] / 4 + 31) / 32 : ((s->n[2] - 2 * s->P) / 4 + FUSED_ZG - 1) / FUSED_ZG;
  tiles *= (s->n[1] - 2 * s->P + FUSED_TR - 1) / FUSED_TR;
  tiles *= (s->n[0] - 2 * s->P + xseg - 1) / xseg;
  return tiles;
}
// planes per block of the reverse-run marching kernels (primal and adjoint; they run one after the other on one branch, two
// blocks per SM): the count that minimises waves x (planes + 1) — whole waves of tiles, little priming overhead.  Measured on
// B200 (round 2): C3 reverse per 2000 steps at 20 / 22 / 24 / 26 / 28 / 32 planes 495.8 / 408.0 / 407.8 / 414.9 / 420.3 / 443.4 ms
// (10 segments x 28 = 280 tiles for 296 slots; the rule takes 23 there: the same 10 segments, one plane step fewer); C4 per 400
// steps at 24 / 32 / 40 planes 1047.9 / 1055.0 / 1046.4 ms (the rule takes 30: 3840 tiles, 13 waves; 1053 ms).
int fused_xseg_rev_auto(const fdtd_sim* s) {
  const long long slots = 2LL * std::max(1, s->sm_count);
  int best = 32;
  long long best_cost = -1;
  for (int x = 16; x <= 64; ++x) {
    const long long t = fused_tiles(s, x), cost = (t + slots - 1) / slots * (x + 1);
    if (best_cost < 0 || cost < best_cost || (cost == best_cost && x > best)) { best = x; best_cost = cost; }
  }
  return best;
}
// planes a block of the marching kernels walks.  Whole-row kernel (two blocks per SM): 32 where that leaves at least one tile per
// SM, else 16.  Measured on B200 (round 2, k_fused_fp): C4 forward per 400 steps at 32 / 40 / 48 planes 548.4 / 548.5 / 551.0 ms;
// C3 per 2000 steps at 16 / 20 / 24 / 28 / 32 planes 223.2 / 225.7 / 217.2 / 208.5 / 208.6 ms (196 tiles at 32).
int fused_xseg(const fdtd_sim* s, bool rev = false) {
  if (rev && s->xseg_rev > 0) return s->xseg_rev;
  if (s->xseg > 0) return s->xseg;
  if (rev && s->fuse_z) return fused_xseg_rev_auto(s);
  if (s->fuse_z) return fused_tiles(s, 32) >= 148 ? 32 : 16;
  return fused_tiles(s, 32) >= 4 * 3 * 148 ? 32 : 16;
}
void launch_fused(fdtd_sim* s, bool inv, int from, int to) {
  FusedArgs a;
  for (int c = 0; c < 3; ++c) {
    a.Ein[c] = s->fb[from][c]; a.Hin[c] = s->fb[from][3 + c];
    a.Eout[c] = s->fb[to][c]; a.Hout[c] = s->fb[to][3 + c];
  }
  for (int ax = 0; ax < 3; ++ax) { a.lo[ax] = s->P + 1; a.hi[ax] = s->n[ax] - s->P - (inv ? 1 : 0); }
  // forward: start on a whole group of 4 z cells.  The slab kernels' box lists (split 4, 5) cover z < P + 4 anyway (their lean z
  // range is rounded to groups), and a first group with one cell masked out cost every warp of the first z tile 24 scalar stores
  // per plane beside its 6 vector stores
  if (!inv) a.lo[2] = (a.lo[2] + 3) / 4 * 4;
  if (a.hi[0] <= a.lo[0] || a.hi[1] <= a.lo[1] || a.hi[2] <= a.lo[2]) return;
  a.xseg = fused_xseg(s, inv);
  if (inv && s->use_iz && s->n[2] - 2 * s->P >= 8) {   // reverse twin in the structure of the whole-row kernel (k_fused_ip)
    FusedIArgs z;
    for (int c = 0; c < 3; ++c) { z.Ein[c] = a.Ein[c]; z.Hin[c] = a.Hin[c]; z.Eout[c] = a.Eout[c]; z.Hout[c] = a.Hout[c]; }
    for (int ax = 0; ax < 2; ++ax) { z.lo[ax] = a.lo[ax]; z.hi[ax] = a.hi[ax]; }
    z.zlo = s->P; z.zhi = s->n[2] - s->P;
    z.xseg = a.xseg;
    const dim3 gz((unsigned)((s->n[2] / 4 + 31) / 32), (unsigned)((z.hi[1] - z.lo[1] + FUSED_TR - 1) / FUSED_TR),
                  (unsigned)((z.hi[0] - z.lo[0] + z.xseg - 1) / z.xseg));
    k_fused_ip<<<gz, dim3(32, FUSED_TR + 1), sizeof(FusedQSmem), s->cur>>>(s->d, z);
    ++s->launches;
    return;
  }
  if (!inv && s->fuse_z) {   // whole rows, z CPML terms in the edge lanes (k_fused_fp)
    FusedZArgs z;
    for (int c = 0; c < 3; ++c) { z.Ein[c] = a.Ein[c]; z.Hin[c] = a.Hin[c]; z.Eout[c] = a.Eout[c]; z.Hout[c] = a.Hout[c]; }
    for (int t = 0; t < 2; ++t) { z.pHz_in[t] = s->pz[from][t]; z.pHz_out[t] = s->pz[to][t]; }
    z.pEz[0] = s->d.psiE[0][1]; z.pEz[1] = s->d.psiE[1][0];
    for (int ax = 0; ax < 2; ++ax) { z.lo[ax] = a.lo[ax]; z.hi[ax] = a.hi[ax]; }
    z.xseg = a.xseg;
    const dim3 gz((unsigned)((s->n[2] / 4 + 31) / 32), (unsigned)((z.hi[1] - z.lo[1] + FUSED_TR - 1) / FUSED_TR),
                  (unsigned)((z.hi[0] - z.lo[0] + z.xseg - 1) / z.xseg));
    k_fused_fp<<<gz, dim3(32, FUSED_TR + 1), sizeof(FusedPSmem), s->cur>>>(s->d, z);
    ++s->launches;
    return;
  }
  const int zbase = a.lo[2] / 4 * 4, zlast = (a.hi[2] - 1) / 4 * 4, groups = (zlast - zbase) / 4 + 1;
  const dim3 g((unsigned)((groups + FUSED_ZG - 1) / FUSED_ZG), (unsigned)((a.hi[1] - a.lo[1] + FUSED_TR - 1) / FUSED_TR),
               (unsigned)((a.hi[0] - a.lo[0] + a.xseg - 1) / a.xseg));
  const dim3 b(32, FUSED_TR + 1);
  if (inv) LAUNCH(s, k_fused_he<true>, g, b, s->d, a);
  else LAUNCH(s, k_fused_he<false>, g, b, s->d, a);
}
// inverse-E update of the source cells redone in the canonical order after the reverse marching kernel (k_inv_e_sources)
void launch_inv_e_sources(fdtd_sim* s, int m_base, const int* step_dev, int from, int to) {
  if (s->nsrc == 0) return;
  long long maxc = 1;
  for (int i = 0; i < s->nsrc; ++i) {
    const SrcDev& q = s->src_host[i];
    maxc = std::max(maxc, (long long)(q.hi[0] - q.lo[0]) * (q.hi[1] - q.lo[1]) * (q.hi[2] - q.lo[2]));
  }
  InvFixArgs a;
  for (int c = 0; c < 3; ++c) { a.Eold[c] = s->fb[from][c]; a.Hnew[c] = s->fb[to][3 + c]; a.Eout[c] = s->fb[to][c]; }
  a.src = reinterpret_cast<const SrcDev*>(s->ws + s->L.srcdesc);
  a.waves = reinterpret_cast<const float*>(s->ws + s->L.waves);
  a.nsrc = s->nsrc; a.m_base = m_base; a.step_dev = step_dev;
  const int threads = maxc >= 128 ? 128 : 32;
  const dim3 g((unsigned)std::min<long long>((maxc + threads - 1) / threads, 1024), (unsigned)s->nsrc);
  LAUNCH(s, k_inv_e_sources, g, threads, s->d, a);
}
FieldIO io_of(const fdtd_sim* s, int eb, int hb, int ob, int out_is_h) {
  FieldIO io;
  for (int c = 0; c < 3; ++c) { io.E[c] = s->fb[eb][c]; io.H[c] = s->fb[hb][3 + c]; io.out[c] = s->fb[ob][out_is_h ? 3 + c : c]; }
  // psi_H of the z axis: in place, except in the whole-row fused path, where the H half-step (out_is_h) goes from the current
  // buffer's psi to the other buffer's (pz[b][0..1], ping-ponged with the fields)
  if (s->fuse_z && out_is_h) {
    for (int t = 0; t < 2; ++t) { io.pHz_in[t] = s->pz[hb][t]; io.pHz_out[t] = s->pz[ob][t]; }
  } else {
    io_psi_inplace(io, s->d);
  }
  return io;
}
// Fused forward step m (fdtd_fused.cuh): from (E^m incl. sources, H^{m-1/2}) in the current buffer to (E^{m+1}, H^{m+1/2}) in
// the other one.  Three branches that only READ the current buffer and the slab kernels' own output:
//   1: slab kernels  H half-step of step m (cur -> other H, boxes of split 5), then E half-step of step m+1
//      (E cur, H other -> other E, boxes of split 4).  Every H value the second one reads was written by the first one.
//   0: marching kernel on [P+1, n-P)^3 (cur -> other); its halo cells (index P) are plain cells recomputed from cur.
//      Where it overlaps the slab boxes (plain layers next to the slabs) both write the same bits.
//   2: E half of state m (record if due, monitor row) and the pending H half of state m-1, all from the current buffer.
// Then the buffers swap and the sources of step m+1 are added.
void forward_fused_step(fdtd_sim* s, int m_base, const int* step_dev, bool rec, bool* pending_h) {
  const int cur = s->cb, oth = cur ^ 1;
  const bool mon = s->has_mon && s->mon_rec;
  fork(s, 3);
  on(s, 1);
  { const FieldIO io = io_of(s, cur, cur, oth, 1); launch_gen(s, 1, 0, s->split[5], &io); }
  { const FieldIO io = io_of(s, cur, oth, oth, 0); launch_gen(s, 0, 0, s->split[4], &io); }
  on(s, 0); launch_fused(s, false, cur, oth);
  on(s, 2);
  if (rec) launch_record(s, m_base, step_dev, 0);
  if (*pending_h) launch_record(s, m_base - 1, step_dev, 1);
  if (mon) {
    launch_box(s, s->mon, s->mon_rec, m_base, step_dev, 0, 0);
    launch_box(s, s->mon, s->mon_rec, m_base - 1, step_dev, 0, 1);
  }
  join(s, 3);
  set_cur(s, oth);
  launch_sources(s, m_base + 1, step_dev, 1.0f);
  *pending_h = rec;
}

// Reverse step with the fused inverse kernel (fdtd_fused.cuh, INV): the primal goes from the current buffer (E^m, H^{m+1/2})
// to the other one (E^{m-1}, H^{m-1/2}) in one marching pass over the inner interior.
//  1: {monitor cotangent then adjoint-H general, adjoint-H lean, [inject H into the other buffer, then the marching kernel,
//      which subtracts the sources of step m itself between its two half-steps]}
//  2: {adjoint-E lean, adjoint-E general, gradient (new H), [sources subtracted from the OLD shell E, then inject E: old shell
//      E for the gradient term, new values into the other buffer]}
void reverse_fused_step(fdtd_sim* s, int m_base, const int* step_dev, const float* dmon, int interp, int pb) {
  const bool cot = dmon && s->has_mon;
  const int cur = s->cb, oth = cur ^ 1;
  const bool alone = s->fuse_rev_mode == 2;   // the marching kernel gets a phase of its own
  fork(s, 3);
  on(s, 1);
  if (cot) {
    launch_box(s, s->mon, const_cast<float*>(dmon), m_base, step_dev, 1);
    if (s->parallel) { cudaEventRecord(s->ev_mid, s->aux[0]); cudaStreamWaitEvent(s->stream, s->ev_mid, 0); }
  }
  launch_gen(s, 2, pb);
  on(s, 0); launch_lean(s, 2, pb);
  on(s, 2);
  launch_inject(s, m_base, step_dev, 1, interp, cur, oth);
  if (alone) join(s, 3);
  launch_fused(s, true, cur, oth);
  launch_inv_e_sources(s, m_base, step_dev, cur, oth);
  if (!alone) join(s, 3);
  set_cur(s, oth);
  fork(s, 4);
  on(s, 0); launch_lean(s, 3, pb);
  on(s, 1); launch_gen(s, 3, pb);
  on(s, 2); launch_grad(s);
  on(s, 3);
  launch_sources(s, m_base, step_dev, -1.0f, 0, 1 << 30, cur);
  launch_inject(s, m_base, step_dev, 0, interp, cur, oth);
  join(s, 4);
}

// ---- fully fused reverse step: fused primal (k_fused_ip) AND fused adjoint (adjoint of H + adjoint of E in one marching pass) ----
AdjIO adj_io(const fdtd_sim* s, int from, int to, bool phase_b) {
  AdjIO io;
  for (int c = 0; c < 3; ++c) {
    io.lEin[c] = phase_b ? s->lb[to][c] : s->lb[from][c];   // adjoint of E reads the NEW lambda_E
    io.lH[c] = s->lb[from][3 + c];
    io.lEout[c] = s->lb[to][c];
    io.lHout[c] = s->lb[to][3 + c];
  }
  return io;
}
void launch_fused_adj(fdtd_sim* s, int from, int to, int pb);   // the adjoint marching kernel (below)
// Phase 1: the monitor cotangent first (it changes the current lambda buffers, which everything below reads), then
//   branch 1: slab kernels, adjoint of H on the boxes of split 6 (current -> other lambda_E), then adjoint of E on those of split 7
//             (lambda_E other, lambda_H current -> other lambda_H); every lambda_E value the second one reads was written by the first;
//   branch 0: inject H, the primal marching kernel, its source cells, then the adjoint marching kernel on [P+1, n-P-1)^2 x whole rows
//             (one after the other: two marching kernels side by side starve each other, profiles/r02c_marching.md).
// Then both buffer pairs swap.  Phase 2: gradient (new lambda_E, new H) beside inject E (shell gradient term with the new lambda_E).
void reverse_fullfused_step(fdtd_sim* s, int m_base, const int* step_dev, const float* dmon, int interp, int pb) {
  const bool cot = dmon && s->has_mon;
  const int cur = s->cb, oth = cur ^ 1, acur = s->acb, aoth = acur ^ 1;
  if (cot) launch_box(s, s->mon, const_cast<float*>(dmon), m_base, step_dev, 1);
  fork(s, 2);
  on(s, 1);
  { const AdjIO io = adj_io(s, acur, aoth, false); launch_gen(s, 2, pb, s->split[6], nullptr, &io); }
  { const AdjIO io = adj_io(s, acur, aoth, true); launch_gen(s, 3, pb, s->split[7], nullptr, &io); }
  on(s, 0);
  launch_inject(s, m_base, step_dev, 1, interp, cur, oth);
  launch_fused(s, true, cur, oth);
  launch_inv_e_sources(s, m_base, step_dev, cur, oth);
  if (!s->fa_debug) launch_fused_adj(s, acur, aoth, pb);
  join(s, 2);
  set_cur(s, oth);
  set_cur_adj(s, aoth);
  fork(s, 2);
  on(s, 0); launch_grad(s);
  on(s, 1);
  launch_sources(s, m_base, step_dev, -1.0f, 0, 1 << 30, cur);
  launch_inject(s, m_base, step_dev, 0, interp, cur, oth);
  join(s, 2);
}
void launch_fused_adj(fdtd_sim* s, int from, int to, int pb) {
  FusedAArgs a;
  for (int c = 0; c < 3; ++c) {
    a.lEin[c] = s->lb[from][c]; a.lHin[c] = s->lb[from][3 + c];
    a.lEout[c] = s->lb[to][c]; a.lHout[c] = s->lb[to][3 + c];
  }
  const int nb = pb ^ 1;
  a.pH_in[0] = s->d.lpsiH[pb][0][1]; a.pH_in[1] = s->d.lpsiH[pb][1][0];
  a.pH_out[0] = s->d.lpsiH[nb][0][1]; a.pH_out[1] = s->d.lpsiH[nb][1][0];
  a.pE_in[0] = s->d.lpsiE[pb][0][1]; a.pE_in[1] = s->d.lpsiE[pb][1][0];
  a.pE_out[0] = s->d.lpsiE[nb][0][1]; a.pE_out[1] = s->d.lpsiE[nb][1][0];
  for (int ax = 0; ax < 2; ++ax) { a.lo[ax] = s->P + 1; a.hi[ax] = s->n[ax] - s->P - 1; }
  if (a.hi[0] <= a.lo[0] || a.hi[1] <= a.lo[1]) return;
  a.xseg = fused_xseg(s, true);
  const dim3 g((unsigned)((s->n[2] / 4 + 31) / 32), (unsigned)((a.hi[1] - a.lo[1] + FUSED_TR - 1) / FUSED_TR),
               (unsigned)((a.hi[0] - a.lo[0] + a.xseg - 1) / a.xseg));
  k_fused_ap<<<g, dim3(32, FUSED_TR + 1), sizeof(FusedASmem), s->cur>>>(s->d, a);
  ++s->launches;
}

// Capture `body` (which enqueues on s->stream and its auxiliaries) into a graph and launch it `times` times.  The
// instantiated graph of each kind (slot 0 forward, 1 fused forward, 2 reverse) is kept in the handle: the next run
// re-captures (pointers such as the monitor record may have changed) and patches the kept executable with
// cudaGraphExecUpdate, which costs far less host time than a new instantiation; only a change of topology (another k,
// another set of kernels) instantiates anew.
template <class F>
fdtd_status run_graph(fdtd_sim* s, int slot, int times, F body) {
  if (times <= 0) return FDTD_OK;
  cudaGraph_t graph = nullptr;
  const unsigned long long before = s->launches;
  cudaStream_t user = s->stream;
  CUDA_TRY(s, cudaStreamBeginCapture(s->cap, cudaStreamCaptureModeThreadLocal));
  s->stream = s->cur = s->cap;
  body();
  s->stream = s->cur = user;
  cudaError_t e = cudaStreamEndCapture(s->cap, &graph);
  if (e != cudaSuccess || !graph) return fail(s, FDTD_ERR_CUDA, "graph capture failed: %s", cudaGetErrorString(e));
  const unsigned long long per = s->launches - before;
  cudaGraphExec_t& exec = s->graph_cache[slot];
  if (exec) {
    cudaGraphExecUpdateResultInfo info;
    if (cudaGraphExecUpdate(exec, graph, &info) != cudaSuccess) {
      cudaGetLastError();
      s->dead_graphs.push_back(exec);   // may still be in flight: destroyed at the next sync point
      exec = nullptr;
    }
  }
  if (!exec) {
    e = cudaGraphInstantiate(&exec, graph, 0);
    if (e != cudaSuccess) { exec = nullptr; cudaGraphDestroy(graph); return fail(s, FDTD_ERR_CUDA, "graph instantiate failed: %s", cudaGetErrorString(e)); }
  }
  cudaGraphDestroy(graph);
  for (int r = 0; r < times; ++r) {
    e = cudaGraphLaunch(exec, s->stream);
    if (e != cudaSuccess) break;
  }
  s->launches = before + per * (unsigned long long)times;
  if (e != cudaSuccess) return fail(s, FDTD_ERR_CUDA, "graph launch failed: %s", cudaGetErrorString(e));
  return FDTD_OK;
}
void reap_graphs(fdtd_sim* s) {
  for (cudaGraphExec_t g : s->dead_graphs) cudaGraphExecDestroy(g);
  s->dead_graphs.clear();
}

fdtd_status zero_state(fdtd_sim* s) {
  const size_t N = (size_t)s->d.N;
  set_cur(s, 0);
  for (int c = 0; c < 6; ++c)
    if (s->fb[1][c]) CUDA_TRY(s, cudaMemsetAsync(s->fb[1][c], 0, N * 4, s->stream));
  for (int t = 0; t < 2; ++t)
    if (s->pz[1][t] && psi_elems(s, 2)) CUDA_TRY(s, cudaMemsetAsync(s->pz[1][t], 0, (size_t)psi_elems(s, 2) * 4, s->stream));
  for (int c = 0; c < 3; ++c) {
    CUDA_TRY(s, cudaMemsetAsync(s->d.E[c], 0, N * 4, s->stream));
    CUDA_TRY(s, cudaMemsetAsync(s->d.H[c], 0, N * 4, s->stream));
    for (int t = 0; t < 2; ++t) {
      const size_t pe = (size_t)psi_elems(s, (c + 1 + t) % 3) * 4;
      if (pe) {
        CUDA_TRY(s, cudaMemsetAsync(s->d.psiE[c][t], 0, pe, s->stream));
        CUDA_TRY(s, cudaMemsetAsync(s->d.psiH[c][t], 0, pe, s->stream));
      }
    }
  }
  s->forward_done = s->state_final = false;
  return FDTD_OK;
}

fdtd_status make_ce(fdtd_sim* s) {
  unsigned* scratch = reinterpret_cast<unsigned*>(s->ws + s->L.scratch);
  const unsigned init = 0x7f7fffffu;
  CUDA_TRY(s, cudaMemcpyAsync(scratch, &init, 4, cudaMemcpyHostToDevice, s->stream));
  LAUNCH(s, k_min_eps, 592, 256, s->eps_dev, s->d.N, scratch);
  LAUNCH(s, k_make_ce, 1184, 256, s->eps_dev, const_cast<float*>(s->d.ce), s->d.N, s->d.S);
  unsigned bits = 0;
  CUDA_TRY(s, cudaMemcpyAsync(&bits, scratch, 4, cudaMemcpyDeviceToHost, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  float mn;
  std::memcpy(&mn, &bits, 4);
  if (!(mn >= 1.0f)) return fail(s, FDTD_ERR_INVALID_ARG, "eps must be >= 1 everywhere (min %g)", (double)mn);
  return FDTD_OK;
}

fdtd_status upload_sources(fdtd_sim* s, int nsteps, const fdtd_source* src, int nsrc, bool amp_is_host) {
  if (nsrc < 0 || nsrc > kMaxSources) return fail(s, FDTD_ERR_INVALID_ARG, "nsrc must be in [0, %d]", kMaxSources);
  if (nsrc > 0 && !src) return fail(s, FDTD_ERR_INVALID_ARG, "src is NULL");
  s->src_host.assign(std::max(nsrc, 1), SrcDev{});
  s->waves_host.assign((size_t)std::max(nsrc, 1) * nsteps, 0.0f);
  size_t amp_used = 0;
  float* amp_stage = (s->flags & FDTD_WS_HOST_IO) ? reinterpret_cast<float*>(s->ws + s->L.amp_stage) : nullptr;
  for (int i = 0; i < nsrc; ++i) {
    const fdtd_source& q = src[i];
    if (q.comp < 0 || q.comp > 2) return fail(s, FDTD_ERR_INVALID_ARG, "source %d: comp must be 0..2", i);
    if (!in_interior(s, q.lo, q.hi)) return fail(s, FDTD_ERR_INVALID_ARG, "source %d: box outside the interior", i);
    if (!q.wave) return fail(s, FDTD_ERR_INVALID_ARG, "source %d: wave is NULL", i);
    SrcDev& o = s->src_host[i];
    o.comp = q.comp;
    for (int a = 0; a < 3; ++a) { o.lo[a] = q.lo[a]; o.hi[a] = q.hi[a]; }
    o.wave_off = (long long)i * nsteps;
    std::memcpy(&s->waves_host[(size_t)i * nsteps], q.wave, (size_t)nsteps * 4);
    o.amp = q.amp;
    if (q.amp && amp_is_host) {
      const size_t cells = (size_t)(q.hi[0] - q.lo[0]) * (q.hi[1] - q.lo[1]) * (q.hi[2] - q.lo[2]);
      if (!amp_stage || amp_used + cells > kAmpStageFloats)
        return fail(s, FDTD_ERR_OOM, "source amplitudes exceed the host-io staging area");
      CUDA_TRY(s, cudaMemcpyAsync(amp_stage + amp_used, q.amp, cells * 4, cudaMemcpyHostToDevice, s->stream));
      o.amp = amp_stage + amp_used;
      amp_used += cells;
    }
  }
  s->nsrc = nsrc;
  s->src_overlap = false;
  for (int i = 0; i < nsrc; ++i)
    for (int j = i + 1; j < nsrc; ++j) {
      const SrcDev &a = s->src_host[i], &b = s->src_host[j];
      bool meet = a.comp == b.comp;
      for (int c = 0; c < 3; ++c) meet = meet && std::max(a.lo[c], b.lo[c]) < std::min(a.hi[c], b.hi[c]);
      s->src_overlap = s->src_overlap || meet;
    }
  if (nsrc > 0) {
    CUDA_TRY(s, cudaMemcpyAsync(s->ws + s->L.srcdesc, s->src_host.data(), sizeof(SrcDev) * nsrc, cudaMemcpyHostToDevice,
                                s->stream));
    CUDA_TRY(s, cudaMemcpyAsync(s->ws + s->L.waves, s->waves_host.data(), (size_t)nsrc * nsteps * 4,
                                cudaMemcpyHostToDevice, s->stream));
    // the host vectors are pageable: the copies above have been staged when the calls return
  }
  return FDTD_OK;
}

// Fused forward run (fdtd_fused.cuh).  Step 1's E half-step runs alone, then nsteps-1 fused steps (H half-step of step m +
// E half-step of step m+1), then the H half-step of the last step.  States are recorded / monitored exactly as in
// forward_step: state m = (E^m, H^{m+1/2}).
// the marching kernels treat the first and the last interior group of a row differently (interface cells, z CPML hand-over): a row
// needs both (found by random-grid testing: nz - 2P = 4 gave wrong fields in forced mode)
bool fuse_grid_ok(const fdtd_sim* s) { return s->can_fuse && s->n[2] - 2 * s->P >= 8; }
bool use_fused(const fdtd_sim* s, int nsteps) {
  if (!fuse_grid_ok(s) || nsteps < 2 || s->fuse_mode == 0) return false;
  if (s->fuse_mode == 1) return true;
  // mode -1 (auto): where the marching kernel fills most of one wave of tiles (3 blocks per SM = 444 slots).  Round 1 (k_fused_he
  // beside class-Z slab boxes) paid only with several waves: C4 (7200 tiles) forward 1910 -> 1727 us per step, C3 (392 tiles)
  // 159 -> 161, C2 35 -> 44.  With the whole-row kernel (k_fused_fp, round 2): C4 1631 -> 1466 us per step against the split
  // path with row kernels, C3 (392 tiles) 129.8 -> 111.8; C2 (91 tiles) 29.1 -> 67.3: stays split.
  if (!s->fuse_z) return fused_tiles(s, fused_xseg(s)) >= 4 * 3 * 148;
  return fused_tiles(s, 16) >= 2 * 148;
}
bool fused_adjoint_possible(const fdtd_sim* s) { return s->fuse_adj_mode != 0 && s->fuse_za && s->lb[1][0] != nullptr; }
bool use_fused_reverse(const fdtd_sim* s) {
  if (s->fuse_rev_mode == 0 || !fuse_grid_ok(s)) return false;
  if (s->fuse_rev_mode >= 1) return true;
  if (!s->use_iz) return false;
  // mode -1 (auto).  Bit-identical to the two-kernel reverse primal; 3.1 GB fewer bytes per step on C4.  History of the primal
  // alone on C4: round 1 (k_fused_he<true>, 1.23 ms per launch) 3406 vs 3395 us per step: off; round 2 with direct loads (1.20 ms)
  // 3148 vs 3094: off; with the cp.async-pipelined kernel (k_fused_ip, 0.98 ms against 0.63 + 0.67 ms for the two inverse kernels)
  // 2924 vs 3090: on; C3 (196 tiles) 234.8 vs 223.7: off.  TOGETHER with the adjoint marching kernel (fully fused reverse step) it
  // pays from one block per SM upwards: C3 at 24 planes per block 203.9 vs 226.4 us per step, C4 2616 vs 3090; C2 (lives in L2,
  // 65 tiles) stays on the split kernels.
  if (fused_adjoint_possible(s)) return fused_tiles(s, fused_xseg(s, true)) >= std::max(1, s->sm_count);
  return fused_tiles(s, 32) >= 4 * 2 * 148;
}
bool use_fused_adjoint(const fdtd_sim* s) {
  if (!fused_adjoint_possible(s) || !use_fused_reverse(s)) return false;
  if (s->fuse_adj_mode >= 1) return true;
  return fused_tiles(s, fused_xseg(s, true)) >= std::max(1, s->sm_count);
}
fdtd_status forward_fused(fdtd_sim* s, int nsteps, int k) {
  // state 0 is recorded whole, then step 1's E half-step runs alone (in place)
  launch_record(s, 0, nullptr, 2);
  launch_split(s, 0, 0);
  launch_sources(s, 1, nullptr, 1.0f);
  bool pend = false;
  int done = 0;   // fused steps m = 1 .. nsteps-1 carried out so far
  int L = k * std::max(1, (16 + k - 1) / k);
  if (L & 1) L *= 2;   // even: the ping-pong buffer is the same at the start of every period
  const int periods = (s->use_graphs && s->aux[0]) ? (nsteps - 1) / L : 0;
  if (periods > 0) {
    int* step_dev = reinterpret_cast<int*>(s->ws + s->L.step);
    LAUNCH(s, k_set_int, 1, 1, step_dev, 0);
    s->parallel = true;
    fdtd_status g = run_graph(s, 1, periods, [&]() {
      bool p = true;   // state 0 (first period: written again, same bytes) or the last state of the previous period
      for (int t = 1; t <= L; ++t) forward_fused_step(s, t, step_dev, t % k == 0, &p);
      LAUNCH(s, k_tick, 1, 1, step_dev, L);
    });
    s->parallel = false;
    s->cur = s->stream;
    if (g != FDTD_OK) return g;
    done = periods * L;
    pend = true;
  }
  for (int m = done + 1; m <= nsteps - 1; ++m) forward_fused_step(s, m, nullptr, m % k == 0, &pend);
  // H halves of state nsteps-1 still pending, then the last H half-step alone, then the final state whole
  forward_flush(s, nsteps - 1, pend);
  launch_split(s, 1, 0);
  if (s->has_mon && s->mon_rec) launch_box(s, s->mon, s->mon_rec, nsteps, nullptr, 0);
  launch_record(s, nsteps, nullptr, 2);
  return FDTD_OK;
}

fdtd_status forward_impl(fdtd_sim* s, int nsteps, const fdtd_source* src, int nsrc, fdtd_dtype dt, int k, bool amp_is_host) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!s->ws) return fail(s, FDTD_ERR_OOM, "no workspace: call fdtd_set_workspace first");
  if (nsteps < 1) return fail(s, FDTD_ERR_INVALID_ARG, "nsteps must be >= 1");
  if (k < 1) return fail(s, FDTD_ERR_INVALID_ARG, "k must be >= 1");
  if (!dtype_ok((int)dt)) return fail(s, FDTD_ERR_INVALID_ARG, "unknown store dtype %d", (int)dt);
  const int slots = num_slots(nsteps, k);
  const size_t need = (size_t)slots * slot_bytes_host(s, (int)dt);
  if (nsteps > s->max_nsteps || slots > s->L.slots_cap || need > s->L.store_cap)
    return fail(s, FDTD_ERR_OOM, "workspace too small: store needs %zu bytes in %d slots, has %zu in %d (nsteps %d, max %d)",
                need, slots, s->L.store_cap, s->L.slots_cap, nsteps, s->max_nsteps);
  s->forward_done = s->state_final = false;
  fdtd_status r = upload_sources(s, nsteps, src, nsrc, amp_is_host);
  if (r != FDTD_OK) return r;
  s->nsteps = nsteps; s->k = k; s->dtype = (int)dt;
  s->st.nslots = slots; s->st.nsteps = nsteps; s->st.k = k; s->st.dtype = (int)dt;
  s->st.slot_bytes = slot_bytes_host(s, (int)dt);
  if (dt == FDTD_F8E4M3_SCALED) CUDA_TRY(s, cudaMemsetAsync(s->st.amax, 0, (size_t)slots * 36 * 4, s->stream));
  s->cur = s->stream;
  if (s->dead_graphs.size() > 32) { CUDA_TRY(s, cudaStreamSynchronize(s->stream)); reap_graphs(s); }
  if (use_fused(s, nsteps)) {
    fdtd_status g = forward_fused(s, nsteps, k);
    if (g != FDTD_OK) return g;
  } else {
    // state 0 (R10): its E half now, its H half during the first E phase (H is untouched until then)
    launch_record(s, 0, nullptr, 0);
    bool pend = true;
    int done = 0;
    // steady-state period of L = k*r steps as one CUDA graph: every period starts and ends with a pending H half
    const int L = k * std::max(1, (16 + k - 1) / k);
    const int periods = (s->use_graphs && s->aux[0]) ? nsteps / L : 0;
    if (periods > 0) {
      int* step_dev = reinterpret_cast<int*>(s->ws + s->L.step);
      LAUNCH(s, k_set_int, 1, 1, step_dev, 0);
      s->parallel = true;
      fdtd_status g = run_graph(s, 0, periods, [&]() {
        bool p = true;
        for (int t = 1; t <= L; ++t) forward_step(s, t, step_dev, t % k == 0, &p);
        LAUNCH(s, k_tick, 1, 1, step_dev, L);
      });
      s->parallel = false;
      s->cur = s->stream;
      if (g != FDTD_OK) return g;
      done = periods * L;
    }
    for (int m = done + 1; m <= nsteps; ++m) forward_step(s, m, nullptr, m % k == 0 || m == nsteps, &pend);
    forward_flush(s, nsteps, pend);
  }
  CUDA_TRY(s, cudaGetLastError());
  s->forward_done = s->state_final = true;
  return FDTD_OK;
}

fdtd_status reverse_impl(fdtd_sim* s, const fdtd_cotangent* fin, const float* dmon, fdtd_interp interp, float* grad_dev) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!s->forward_done || !s->state_final) return fail(s, FDTD_ERR_STATE, "fdtd_reverse needs a completed fdtd_forward");
  if (!(s->flags & FDTD_WS_REVERSE)) return fail(s, FDTD_ERR_STATE, "workspace was sized without FDTD_WS_REVERSE");
  if ((int)interp < 0 || (int)interp > 1) return fail(s, FDTD_ERR_INVALID_ARG, "unknown interpolation %d", (int)interp);
  if (dmon && !s->has_mon) return fail(s, FDTD_ERR_INVALID_ARG, "dL_dmon given but no monitor is set");
  if (s->store_mode == 1 && s->has_design)
    for (int a = 0; a < 3; ++a)
      if (s->dlo[a] < s->P + 1 || s->dhi[a] > s->n[a] - s->P - 1)
        return fail(s, FDTD_ERR_INVALID_ARG, "tangential store: the design box must lie in the inner interior (the shell is not reconstructed)");
  const size_t N = (size_t)s->d.N;
  s->cur = s->stream;
  if (s->dead_graphs.size() > 32) { CUDA_TRY(s, cudaStreamSynchronize(s->stream)); reap_graphs(s); }
  set_cur_adj(s, 0);
  for (int c = 0; c < 6; ++c)
    if (s->lb[1][c]) CUDA_TRY(s, cudaMemsetAsync(s->lb[1][c], 0, N * 4, s->stream));
  for (int c = 0; c < 3; ++c) {
    CUDA_TRY(s, cudaMemsetAsync(s->d.lE[c], 0, N * 4, s->stream));
    CUDA_TRY(s, cudaMemsetAsync(s->d.lH[c], 0, N * 4, s->stream));
    for (int t = 0; t < 2; ++t) {
      const size_t pe = (size_t)psi_elems(s, (c + 1 + t) % 3) * 4;
      for (int b = 0; b < 2 && pe; ++b) {
        CUDA_TRY(s, cudaMemsetAsync(s->d.lpsiE[b][c][t], 0, pe, s->stream));
        CUDA_TRY(s, cudaMemsetAsync(s->d.lpsiH[b][c][t], 0, pe, s->stream));
      }
    }
  }
  if (s->has_design) CUDA_TRY(s, cudaMemsetAsync(s->d.acc, 0, (size_t)design_cells(s) * 8, s->stream));
  if (fin) {
    if (!in_grid(s, fin->lo, fin->hi) || !(fin->comp_mask & 63u) || !fin->g_dev)
      return fail(s, FDTD_ERR_INVALID_ARG, "dL_dfinal: bad box, mask or pointer");
    BoxDev b{};
    for (int a = 0; a < 3; ++a) { b.lo[a] = fin->lo[a]; b.hi[a] = fin->hi[a]; }
    b.mask = fin->comp_mask & 63u;
    b.ncomp = __builtin_popcount(b.mask);
    launch_box(s, b, const_cast<float*>(fin->g_dev), 0, nullptr, 3);
  }
  s->state_final = false;
  int pb = 0;
  int top = s->nsteps;
  const bool rf = use_fused_reverse(s);   // inverse-H + inverse-E of the primal in one marching kernel (ping-pong buffers)
  const bool fa = use_fused_adjoint(s);   // ... and adjoint of H + adjoint of E in one marching kernel (lambda ping-pong buffers)
  {
    const int L = 16;   // even, so the psi ping-pong parity is the same at the start of every period
    const int periods = (s->use_graphs && s->aux[0]) ? s->nsteps / L : 0;
    if (periods > 0) {
      int* step_dev = reinterpret_cast<int*>(s->ws + s->L.step);
      LAUNCH(s, k_set_int, 1, 1, step_dev, s->nsteps);
      s->parallel = true;
      fdtd_status g = run_graph(s, fa ? 4 : (rf ? 3 : 2), periods, [&]() {
        for (int t = 0; t < L; ++t) {
          if (fa) reverse_fullfused_step(s, -t, step_dev, dmon, (int)interp, t & 1);
          else if (rf) reverse_fused_step(s, -t, step_dev, dmon, (int)interp, t & 1);
          else reverse_step(s, -t, step_dev, dmon, (int)interp, t & 1);
        }
        LAUNCH(s, k_tick, 1, 1, step_dev, -L);
      });
      s->parallel = false;
      s->cur = s->stream;
      if (g != FDTD_OK) return g;
      top -= periods * L;
    }
  }
  for (int m = top; m >= 1; --m, pb ^= 1) {
    if (fa) reverse_fullfused_step(s, m, nullptr, dmon, (int)interp, pb);
    else if (rf) reverse_fused_step(s, m, nullptr, dmon, (int)interp, pb);
    else reverse_step(s, m, nullptr, dmon, (int)interp, pb);
  }
  if (grad_dev && s->has_design)
    LAUNCH(s, k_grad_finalize, (unsigned)((design_cells(s) + 255) / 256), 256, s->d, s->eps_dev, grad_dev);
  CUDA_TRY(s, cudaGetLastError());
  return FDTD_OK;
}

}  // namespace

extern "C" {

fdtd_status fdtd_create(fdtd_sim** out, int nx, int ny, int nz, double dx, double dt, int pml_width, const float* eps_dev,
                        void* cuda_stream) {
  if (!out) return FDTD_ERR_INVALID_ARG;
  *out = nullptr;
  if (nx < 3 || ny < 3 || nz < 3 || pml_width < 0 || !eps_dev || !(dx > 0) || !(dt > 0)) return FDTD_ERR_INVALID_ARG;
  if (nx - 2 * pml_width < 2 || ny - 2 * pml_width < 2 || nz - 2 * pml_width < 2) return FDTD_ERR_INVALID_ARG;
  if ((long long)nx * ny * nz >= (1LL << 32)) return FDTD_ERR_INVALID_ARG;   // 32-bit element offsets in the kernels
  const double S = kC0 * dt / dx;
  if (S > (1.0 / std::sqrt(3.0)) * (1.0 + 1e-9)) return FDTD_ERR_INVALID_ARG;   // PAPER.md:37-39 CFL limit
  fdtd_sim* s = new (std::nothrow) fdtd_sim();
  if (!s) return FDTD_ERR_OOM;
  s->n[0] = nx; s->n[1] = ny; s->n[2] = nz; s->P = pml_width; s->dx = dx; s->dt = dt; s->Sd = S;
  s->eps_dev = eps_dev;
  s->V = (nz % 4 == 0 && pml_width % 4 == 0) ? 4 : 1;
  s->VG = s->V;
  s->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  s->cur = s->stream;
  if (const char* e = std::getenv("FDTD_FUSE")) { const int v = atoi(e); if (v >= -1 && v <= 1) s->fuse_mode = v; }
  if (const char* e = std::getenv("FDTD_FUSE_REV")) { const int v = atoi(e); if (v >= -1 && v <= 2) s->fuse_rev_mode = v; }
  {
    // DRAM is fetched in whole 128-byte lines: a lean region that starts 64 bytes into a row (P = 16) costs the lean AND the
    // z-slab kernel a half-used line per row end (measured on C3: reads 33 % above the arrays' size, profiles/r01d_c3.md)
    int dev = 0, l2 = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev);
    { int sms = 0; if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) s->sm_count = sms; }
    cudaGetLastError();
    const double fwd_bytes = 7.0 * 4.0 * (double)nx * ny * nz;
    s->zalign = (l2 > 0 && fwd_bytes > 1.5 * (double)l2) ? 32 : 16;
    // Row kernels (fdtd_stencil.cuh: lean cells and the z-slab cells of the same rows in one launch) pay where the arrays stream
    // from HBM (whole DRAM pages while they are open).  On a grid that lives in L2 (C2) the split with its own z-slab boxes is
    // as fast or faster: forward H 13.4 us against 14.6, adjoint of E 17.9 against 18.2 (round 2, B200).
    s->use_rows = s->rows_auto = l2 <= 0 || fwd_bytes > 1.5 * (double)l2;
  }
  if (const char* e = std::getenv("FDTD_ZALIGN")) {   // debug knob: only multiples of 4 that are >= V keep the float4 accesses aligned
    const int v = atoi(e);
    if (v >= s->V && v % 4 == 0) s->zalign = v;
  }
  if (const char* e = std::getenv("FDTD_ROWS")) s->use_rows = atoi(e) != 0;
  // z-face injection inside the inverse kernels: the two threads per row that do it make their whole warp walk the fetch path, so
  // it pays where a row is several warps long.  Measured (round 2, B200): C4 (4 warps per row) reverse 3176 -> 3106 us per step;
  // C3 (1 warp per row) 226.6 -> 238.4, C2 57.2 -> 63.1: off there.
  s->use_zf = nz - 2 * pml_width > 256;
  if (const char* e = std::getenv("FDTD_ZF")) s->use_zf = atoi(e) != 0;
  if (const char* e = std::getenv("FDTD_FZ")) s->use_fz = atoi(e) != 0;
  if (const char* e = std::getenv("FDTD_IZ")) s->use_iz = atoi(e) != 0;
  if (const char* e = std::getenv("FDTD_FUSE_ADJ")) { const int v = atoi(e); if (v >= -1 && v <= 1) s->fuse_adj_mode = v; }
  if (const char* e = std::getenv("FDTD_FA_DEBUG")) s->fa_debug = atoi(e) != 0;
  if (const char* e = std::getenv("FDTD_XSEG")) { const int v = atoi(e); if (v >= 1) s->xseg = v; }
  if (const char* e = std::getenv("FDTD_XSEG_REV")) { const int v = atoi(e); if (v >= 1) s->xseg_rev = v; }
  bool ok = cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&s->ev_mid, cudaEventDisableTiming) == cudaSuccess;
  for (int b = 0; b < 4 && ok; ++b)
    ok = cudaStreamCreateWithFlags(&s->aux[b], cudaStreamNonBlocking) == cudaSuccess &&
         cudaEventCreateWithFlags(&s->ev_join[b], cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&s->cap, cudaStreamNonBlocking) == cudaSuccess;
  if (!ok) { for (int b = 0; b < 4; ++b) s->aux[b] = nullptr; cudaGetLastError(); }   // graphs off, serial launches
  *out = s;
  return FDTD_OK;
}

fdtd_status fdtd_set_cpml(fdtd_sim* s, double sigma_factor, double kappa_max, double alpha_max, double grade_m) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (s->ws) return fail(s, FDTD_ERR_STATE, "fdtd_set_cpml must precede fdtd_set_workspace");
  if (sigma_factor < 0 || kappa_max < 1 || alpha_max < 0 || grade_m <= 0) return fail(s, FDTD_ERR_INVALID_ARG, "bad CPML constants");
  s->cpml[0] = sigma_factor; s->cpml[1] = kappa_max; s->cpml[2] = alpha_max; s->cpml[3] = grade_m;
  return FDTD_OK;
}

fdtd_status fdtd_set_design(fdtd_sim* s, const int lo[3], const int hi[3]) {
  if (!s || !lo || !hi) return FDTD_ERR_INVALID_ARG;
  if (s->ws) return fail(s, FDTD_ERR_STATE, "fdtd_set_design must precede fdtd_set_workspace");
  if (!in_interior(s, lo, hi)) return fail(s, FDTD_ERR_INVALID_ARG, "design box must lie inside the interior");
  for (int a = 0; a < 3; ++a) { s->dlo[a] = lo[a]; s->dhi[a] = hi[a]; }
  s->has_design = true;
  return FDTD_OK;
}

fdtd_status fdtd_set_monitor(fdtd_sim* s, const int lo[3], const int hi[3], unsigned comp_mask, float* record_dev) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!lo || !hi) { s->has_mon = false; s->mon_rec = nullptr; return FDTD_OK; }
  if (!in_grid(s, lo, hi) || !(comp_mask & 63u)) return fail(s, FDTD_ERR_INVALID_ARG, "monitor: bad box or mask");
  BoxDev b{};
  for (int a = 0; a < 3; ++a) { b.lo[a] = lo[a]; b.hi[a] = hi[a]; }
  b.mask = comp_mask & 63u;
  b.ncomp = __builtin_popcount(b.mask);
  if (s->ws && (s->flags & FDTD_WS_HOST_IO) && s->has_mon &&
      (long long)b.ncomp * (hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2]) > mon_floats_per_step(s))
    return fail(s, FDTD_ERR_STATE, "monitor grew after the host-io workspace was sized");
  s->mon = b;
  s->has_mon = true;
  s->mon_rec = record_dev;
  return FDTD_OK;
}

size_t fdtd_workspace_bytes(const fdtd_sim* s, int nsteps, fdtd_dtype dt, int k, unsigned flags) {
  if (!s || nsteps < 1 || k < 1 || !dtype_ok((int)dt)) return 0;
  return make_layout(s, nsteps, (int)dt, k, flags).total;
}

fdtd_status fdtd_set_workspace(fdtd_sim* s, void* ws_dev, size_t bytes, int nsteps, fdtd_dtype dt, int k, unsigned flags) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!ws_dev || nsteps < 1 || k < 1 || !dtype_ok((int)dt)) return fail(s, FDTD_ERR_INVALID_ARG, "bad workspace arguments");
  if (reinterpret_cast<uintptr_t>(ws_dev) % 256) return fail(s, FDTD_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
  const Layout L = make_layout(s, nsteps, (int)dt, k, flags);
  if (bytes < L.total) return fail(s, FDTD_ERR_OOM, "workspace too small: need %zu bytes, got %zu", L.total, bytes);
  if (s->eps_owned) {
    // eps came through fdtd_set_eps_host and lives in the PREVIOUS workspace, at an offset the new layout moves (or in a
    // buffer the caller may already have freed): it cannot be carried over.
    s->eps_owned = false;
    s->eps_dev = nullptr;
  }
  if (!s->eps_dev) {
    s->ws = nullptr;
    return fail(s, FDTD_ERR_STATE, "eps was set through fdtd_set_eps_host into the previous workspace: call fdtd_set_eps first");
  }
  s->ws = static_cast<char*>(ws_dev);
  s->ws_bytes = bytes; s->L = L; s->flags = flags;
  // debugging aid (fdtd_bench.h): every byte of the workspace starts as 0xFF — guard bands keep that pattern unless a kernel writes
  // out of bounds, and a float read from a guard band or from a sub-array nobody initialised is a NaN that reaches the results
  if (flags & kWsGuard) CUDA_TRY(s, cudaMemsetAsync(ws_dev, 0xFF, L.total, s->stream));
  s->max_nsteps = nsteps; s->max_k = k; s->max_dtype = (int)dt;
  Dev& d = s->d;
  d = Dev{};
  for (int a = 0; a < 3; ++a) d.n[a] = s->n[a];
  d.P = s->P;
  d.sy = s->n[2];
  d.sx = (idx_t)s->n[1] * (idx_t)s->n[2];
  d.N = (long long)s->n[0] * s->n[1] * s->n[2];
  d.S = (float)s->Sd;
  char* w = s->ws;
  d.ce = reinterpret_cast<float*>(w + L.ce);
  s->can_fuse = s->V == 4 && s->P >= 4;
  {
    // whole-row marching kernel: every tile boundary (a multiple of 128 cells) must have a plain cell right below it, because an
    // edge lane recomputes the new H of that cell without CPML terms
    bool ok = s->can_fuse && s->use_fz && 2 * s->P <= 4 * FUSED_ZSL;   // the staging area of the slab lanes
    for (int kb = 128; ok && kb < s->n[2]; kb += 128) ok = kb - 1 >= s->P && kb - 1 < s->n[2] - s->P;
    s->fuse_z = ok;
    // the adjoint marching kernel recomputes the cell ABOVE a tile boundary: that one has to be plain as well
    for (int kb = 128; ok && kb < s->n[2]; kb += 128) ok = kb < s->n[2] - s->P;
    s->fuse_za = ok;
    if (s->can_fuse) {   // the whole-row marching kernels use more than 48 KB of shared memory per block: opt in (not during a capture)
      CUDA_TRY(s, cudaFuncSetAttribute(k_fused_fp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedPSmem)));
      CUDA_TRY(s, cudaFuncSetAttribute(k_fused_ip, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedQSmem)));
      CUDA_TRY(s, cudaFuncSetAttribute(k_fused_ap, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedASmem)));
    }
  }
  for (int c = 0; c < 3; ++c) {
    d.E[c] = reinterpret_cast<float*>(w + L.E[c]);
    d.H[c] = reinterpret_cast<float*>(w + L.H[c]);
    s->fb[0][c] = d.E[c]; s->fb[0][3 + c] = d.H[c];
    s->fb[1][c] = s->can_fuse ? reinterpret_cast<float*>(w + L.E2[c]) : nullptr;
    s->fb[1][3 + c] = s->can_fuse ? reinterpret_cast<float*>(w + L.H2[c]) : nullptr;
    for (int t = 0; t < 2; ++t) {
      d.psiE[c][t] = reinterpret_cast<float*>(w + L.psiE[c][t]);
      d.psiH[c][t] = reinterpret_cast<float*>(w + L.psiH[c][t]);
    }
  }
  s->pz[0][0] = d.psiH[0][1]; s->pz[0][1] = d.psiH[1][0];
  for (int t = 0; t < 2; ++t) s->pz[1][t] = s->can_fuse ? reinterpret_cast<float*>(w + L.pHz2[t]) : nullptr;
  size_t base = 0;
  for (int a = 0; a < 3; ++a) {
    for (int t = 0; t < 6; ++t) d.tab[a][t] = reinterpret_cast<float*>(w + L.tab) + base + (size_t)t * s->n[a];
    base += (size_t)6 * s->n[a];
  }
  if (flags & FDTD_WS_REVERSE) {
    for (int c = 0; c < 3; ++c) {
      d.lE[c] = reinterpret_cast<float*>(w + L.lE[c]);
      d.lH[c] = reinterpret_cast<float*>(w + L.lH[c]);
      for (int b = 0; b < 2; ++b)
        for (int t = 0; t < 2; ++t) {
          d.lpsiE[b][c][t] = reinterpret_cast<float*>(w + L.lpsiE[b][c][t]);
          d.lpsiH[b][c][t] = reinterpret_cast<float*>(w + L.lpsiH[b][c][t]);
        }
    }
    d.acc = reinterpret_cast<double*>(w + L.acc);
    for (int c = 0; c < 3; ++c) {
      s->lb[0][c] = d.lE[c]; s->lb[0][3 + c] = d.lH[c];
      s->lb[1][c] = s->can_fuse ? reinterpret_cast<float*>(w + L.lE2[c]) : nullptr;
      s->lb[1][3 + c] = s->can_fuse ? reinterpret_cast<float*>(w + L.lH2[c]) : nullptr;
    }
    s->acb = 0;
  }
  d.has_design = s->has_design ? 1 : 0;
  {   // ce resident in L2 during the reverse run where it fits a third of it (fdtd_dev.cuh, ldv_ce)
    int dev = 0, l2 = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) != cudaSuccess) l2 = 0;
    d.ce_keep = ((long long)d.N * 4 <= (long long)l2 / 3) ? 1 : 0;
    if (const char* e = std::getenv("FDTD_CE_KEEP")) d.ce_keep = atoi(e) ? 1 : 0;
  }
  for (int a = 0; a < 3; ++a) { d.dlo[a] = s->dlo[a]; d.dhi[a] = s->dhi[a]; }
  // store geometry
  StoreDev& st = s->st;
  st = StoreDev{};
  st.base = w + L.store;
  st.scales = reinterpret_cast<float*>(w + L.scales);
  st.amax = reinterpret_cast<unsigned*>(w + L.amax);
  st.slot_values = slot_values(s);
  st.mode = s->store_mode;
  st.val_off[0] = st.cell_off[0] = 0;
  for (int f = 0; f < 6; ++f) {
    const int a = f / 2;
    const int b0 = a == 0 ? 1 : 0, b1 = a == 2 ? 1 : 2;
    st.du[f] = s->n[b0] - 2 * s->P;
    st.dv[f] = s->n[b1] - 2 * s->P;
    st.val_off[f + 1] = st.val_off[f] + face_comps(s) * face_size(s, f);
    st.blk_off[f + 1] = st.blk_off[f] + face_comps(s) * face_blocks(s, f);
    st.blkc_off[f + 1] = st.blkc_off[f] + face_blocks(s, f);
    st.cell_off[f + 1] = st.cell_off[f] + face_size(s, f);
  }
  s->VG = s->V;
  if (const char* e = std::getenv("FDTD_VG")) { const int v = atoi(e); if ((v == 1 || v == 2 || v == 4) && s->V == 4) s->VG = v; }
  for (int which = 0; which < 8; ++which) s->split[which] = make_split(s, which, 0, s->n[0]);
  build_tables(s);
  CUDA_TRY(s, cudaMemcpyAsync(w + L.tab, s->tables_host.data(), s->tables_host.size() * 4, cudaMemcpyHostToDevice, s->stream));
  CUDA_TRY(s, cudaMemsetAsync(w + L.step, 0, 16, s->stream));
  fdtd_status r = make_ce(s);
  if (r != FDTD_OK) { s->ws = nullptr; return r; }
  return zero_state(s);
}

fdtd_status fdtd_set_eps(fdtd_sim* s, const float* eps_dev) {
  if (!s || !eps_dev) return FDTD_ERR_INVALID_ARG;
  s->eps_dev = eps_dev;
  s->eps_owned = false;
  if (!s->ws) return FDTD_OK;
  fdtd_status r = make_ce(s);
  if (r != FDTD_OK) return r;
  return zero_state(s);
}

fdtd_status fdtd_reset(fdtd_sim* s) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!s->ws) return fail(s, FDTD_ERR_OOM, "no workspace");
  return zero_state(s);
}

fdtd_status fdtd_set_graphs(fdtd_sim* s, int enabled) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  s->use_graphs = enabled != 0;
  return FDTD_OK;
}

fdtd_status fdtd_set_fused(fdtd_sim* s, int mode, int xseg) {
  if (!s || mode < -1 || mode > 1 || xseg < 0) return FDTD_ERR_INVALID_ARG;
  s->fuse_mode = s->fuse_rev_mode = s->fuse_adj_mode = mode;
  if (xseg > 0) s->xseg = xseg;
  return FDTD_OK;
}

fdtd_status fdtd_set_store_mode(fdtd_sim* s, int mode) {
  if (!s || mode < 0 || mode > 1) return FDTD_ERR_INVALID_ARG;
  if (s->ws) return fail(s, FDTD_ERR_STATE, "fdtd_set_store_mode must precede fdtd_set_workspace");
  s->store_mode = mode;
  return FDTD_OK;
}

fdtd_status fdtd_set_rows(fdtd_sim* s, int mode) {
  if (!s || mode < -1 || mode > 1) return FDTD_ERR_INVALID_ARG;
  if (s->ws) return fail(s, FDTD_ERR_STATE, "fdtd_set_rows must precede fdtd_set_workspace");
  s->use_rows = mode < 0 ? s->rows_auto : mode == 1;
  return FDTD_OK;
}

int fdtd_uses_fused_adjoint(const fdtd_sim* s) { return (s && s->ws && use_fused_adjoint(s)) ? 1 : 0; }
int fdtd_uses_fused_reverse(const fdtd_sim* s) { return (s && s->ws && use_fused_reverse(s)) ? 1 : 0; }
int fdtd_uses_fused(const fdtd_sim* s, int nsteps) { return (s && s->ws && use_fused(s, nsteps)) ? 1 : 0; }

fdtd_status fdtd_forward(fdtd_sim* s, int nsteps, const fdtd_source* src, int nsrc, fdtd_dtype dt, int k) {
  return forward_impl(s, nsteps, src, nsrc, dt, k, false);
}

fdtd_status fdtd_reverse(fdtd_sim* s, const fdtd_cotangent* fin, const float* dmon, fdtd_interp interp, float* grad_dev) {
  return reverse_impl(s, fin, dmon, interp, grad_dev);
}

size_t fdtd_store_bytes(const fdtd_sim* s) {
  if (!s || !s->forward_done) return 0;
  return (size_t)s->st.nslots * (s->st.slot_bytes + (s->dtype == DT_E4M3S ? (size_t)store_slices(s) * 4 : 0));
}

fdtd_status fdtd_get_fields(fdtd_sim* s, float* out_dev) {
  if (!s || !out_dev) return FDTD_ERR_INVALID_ARG;
  if (!s->ws) return fail(s, FDTD_ERR_OOM, "no workspace");
  const size_t N = (size_t)s->d.N;
  for (int c = 0; c < 3; ++c) {
    CUDA_TRY(s, cudaMemcpyAsync(out_dev + c * N, s->d.E[c], N * 4, cudaMemcpyDeviceToDevice, s->stream));
    CUDA_TRY(s, cudaMemcpyAsync(out_dev + (3 + c) * N, s->d.H[c], N * 4, cudaMemcpyDeviceToDevice, s->stream));
  }
  return FDTD_OK;
}

fdtd_status fdtd_get_adjoint(fdtd_sim* s, float* out_dev) {
  if (!s || !out_dev) return FDTD_ERR_INVALID_ARG;
  if (!s->ws || !(s->flags & FDTD_WS_REVERSE)) return fail(s, FDTD_ERR_STATE, "no reverse workspace");
  const size_t N = (size_t)s->d.N;
  for (int c = 0; c < 3; ++c) {
    CUDA_TRY(s, cudaMemcpyAsync(out_dev + c * N, s->d.lE[c], N * 4, cudaMemcpyDeviceToDevice, s->stream));
    CUDA_TRY(s, cudaMemcpyAsync(out_dev + (3 + c) * N, s->d.lH[c], N * 4, cudaMemcpyDeviceToDevice, s->stream));
  }
  return FDTD_OK;
}

fdtd_status fdtd_get_box(fdtd_sim* s, const int lo[3], const int hi[3], unsigned comp_mask, float* out_dev) {
  if (!s || !lo || !hi || !out_dev) return FDTD_ERR_INVALID_ARG;
  if (!s->ws) return fail(s, FDTD_ERR_OOM, "no workspace");
  if (!in_grid(s, lo, hi) || !(comp_mask & 63u)) return fail(s, FDTD_ERR_INVALID_ARG, "get_box: bad box or mask");
  BoxDev b{};
  for (int a = 0; a < 3; ++a) { b.lo[a] = lo[a]; b.hi[a] = hi[a]; }
  b.mask = comp_mask & 63u;
  b.ncomp = __builtin_popcount(b.mask);
  launch_box(s, b, out_dev, 0, nullptr, 2);
  CUDA_TRY(s, cudaGetLastError());
  return FDTD_OK;
}

int fdtd_num_slots(const fdtd_sim* s) { return (s && s->forward_done) ? s->st.nslots : 0; }
size_t fdtd_slot_values(const fdtd_sim* s) { return s ? (size_t)slot_values(s) : 0; }
fdtd_status fdtd_slot_ptr(const fdtd_sim* s, int j, const void** data_dev, const float** scales_dev) {
  if (!s || !s->forward_done || j < 0 || j >= s->st.nslots) return FDTD_ERR_INVALID_ARG;
  if (data_dev) *data_dev = s->st.base + (size_t)j * s->st.slot_bytes;
  if (scales_dev) *scales_dev = s->st.scales + (size_t)j * 36;
  return FDTD_OK;
}
size_t fdtd_slot_bytes(const fdtd_sim* s, fdtd_dtype dt) { return (s && dtype_ok((int)dt)) ? slot_bytes_host(s, (int)dt) : 0; }

// ---- host-buffer variants ----
fdtd_status fdtd_set_eps_host(fdtd_sim* s, const float* eps_host) {
  if (!s || !eps_host) return FDTD_ERR_INVALID_ARG;
  if (!s->ws || !(s->flags & FDTD_WS_HOST_IO)) return fail(s, FDTD_ERR_STATE, "needs a workspace with FDTD_WS_HOST_IO");
  float* own = reinterpret_cast<float*>(s->ws + s->L.eps_own);
  CUDA_TRY(s, cudaMemcpyAsync(own, eps_host, (size_t)s->d.N * 4, cudaMemcpyHostToDevice, s->stream));
  const fdtd_status r = fdtd_set_eps(s, own);
  s->eps_owned = r == FDTD_OK;   // eps now lives inside the workspace: fdtd_set_workspace must not keep this pointer
  return r;
}

fdtd_status fdtd_forward_host(fdtd_sim* s, int nsteps, const fdtd_source* src, int nsrc, fdtd_dtype dt, int k, float* mon_host) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!s->ws || !(s->flags & FDTD_WS_HOST_IO)) return fail(s, FDTD_ERR_STATE, "needs a workspace with FDTD_WS_HOST_IO");
  float* saved = s->mon_rec;
  if (s->has_mon) s->mon_rec = reinterpret_cast<float*>(s->ws + s->L.mon_stage);
  fdtd_status r = forward_impl(s, nsteps, src, nsrc, dt, k, true);
  if (r == FDTD_OK && s->has_mon && mon_host)
    r = cudaMemcpyAsync(mon_host, s->mon_rec, (size_t)mon_floats_per_step(s) * nsteps * 4, cudaMemcpyDeviceToHost, s->stream) == cudaSuccess
            ? FDTD_OK : fail(s, FDTD_ERR_CUDA, "monitor download failed");
  s->mon_rec = saved;
  if (r != FDTD_OK) return r;
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  return FDTD_OK;
}

fdtd_status fdtd_reverse_host(fdtd_sim* s, const float* dmon_host, fdtd_interp interp, float* grad_host) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  if (!s->ws || !(s->flags & FDTD_WS_HOST_IO)) return fail(s, FDTD_ERR_STATE, "needs a workspace with FDTD_WS_HOST_IO");
  float* stage = reinterpret_cast<float*>(s->ws + s->L.mon_stage);
  if (dmon_host) {
    if (!s->has_mon) return fail(s, FDTD_ERR_INVALID_ARG, "dmon given but no monitor is set");
    CUDA_TRY(s, cudaMemcpyAsync(stage, dmon_host, (size_t)mon_floats_per_step(s) * s->nsteps * 4, cudaMemcpyHostToDevice, s->stream));
  }
  float* gstage = reinterpret_cast<float*>(s->ws + s->L.grad_stage);
  fdtd_status r = reverse_impl(s, nullptr, dmon_host ? stage : nullptr, interp, grad_host ? gstage : nullptr);
  if (r != FDTD_OK) return r;
  if (grad_host && s->has_design)
    CUDA_TRY(s, cudaMemcpyAsync(grad_host, gstage, (size_t)design_cells(s) * 4, cudaMemcpyDeviceToHost, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  return FDTD_OK;
}

// ---- stand-alone codec ----
fdtd_status fdtd_codec_encode(fdtd_dtype dt, const float* x_dev, size_t n, void* codes_dev, float* scale_dev,
                              unsigned* scratch_dev, void* cuda_stream) {
  if (!x_dev || !codes_dev || !scale_dev || !dtype_ok((int)dt)) return FDTD_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const unsigned g = (unsigned)std::min<size_t>(std::max<size_t>((n + 255) / 256, 1), 1184);
  if ((int)dt == DT_MX32) {   // codes_dev holds n codes followed by ceil(n/32) scale bytes
    const unsigned gm = (unsigned)std::min<size_t>(std::max<size_t>((n + 255) / 256, 1), 148 * 8);
    k_codec_encode_mx<<<gm, 256, 0, (cudaStream_t)cuda_stream>>>(x_dev, n, reinterpret_cast<unsigned char*>(codes_dev));
    const float one = 1.0f;
    if (cudaMemcpyAsync(scale_dev, &one, 4, cudaMemcpyHostToDevice, (cudaStream_t)cuda_stream) != cudaSuccess) return FDTD_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? FDTD_OK : FDTD_ERR_CUDA;
  }
  if ((int)dt == DT_E4M3S) {
    if (!scratch_dev) return FDTD_ERR_INVALID_ARG;
    if (cudaMemsetAsync(scratch_dev, 0, 4, st) != cudaSuccess) return FDTD_ERR_CUDA;
    k_codec_amax<<<g, 256, 0, st>>>(x_dev, n, scratch_dev);
  }
  FDTD_DT_SWITCH((int)dt, (k_codec_encode<DT><<<g, 256, 0, st>>>(x_dev, n, codes_dev, scale_dev, (int)dt == DT_E4M3S ? scratch_dev : nullptr)))
  return cudaGetLastError() == cudaSuccess ? FDTD_OK : FDTD_ERR_CUDA;
}

fdtd_status fdtd_codec_fetch(fdtd_dtype dt, fdtd_interp interp, const void* const codes_dev[4], const float scales[4],
                             int num, int den, size_t n, float* out_dev, void* cuda_stream) {
  if (!codes_dev || !scales || !out_dev || den < 1 || num < 0 || num >= den || !dtype_ok((int)dt)) return FDTD_ERR_INVALID_ARG;
  const int mode = num == 0 ? 0 : ((int)interp == 1 ? 2 : 1);
  if (!codes_dev[1] || (mode >= 1 && !codes_dev[2]) || (mode == 2 && (!codes_dev[0] || !codes_dev[3]))) return FDTD_ERR_INVALID_ARG;
  FetchArgs a;
  for (int j = 0; j < 4; ++j) { a.codes[j] = codes_dev[j]; a.scales[j] = scales[j]; }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const unsigned g = (unsigned)std::min<size_t>(std::max<size_t>((n + 255) / 256, 1), 1184);
  FDTD_DT_SWITCH((int)dt, (k_codec_fetch<DT><<<g, 256, 0, st>>>(a, mode, num, den, n, out_dev)))
  return cudaGetLastError() == cudaSuccess ? FDTD_OK : FDTD_ERR_CUDA;
}

// ---- allocation-free slice encoder (include/fdtd.h: fdtd_codec_encode_slices_noalloc) ----
// The absmax words of the per-slice reduction live in this file-scope device array instead of caller memory.  In HOST code the
// name below is a host-side stand-in, not a device address: its address is looked up once per device with cudaGetSymbolAddress
// (that device current) and passed to the kernels.  Shared by every call on a device; a call clears the words it uses first.
}  // extern "C"
static __device__ __align__(256) unsigned g_noalloc_amax[FDTD_NOALLOC_MAX_SLICES];
namespace {
constexpr int kMaxDevices = 64;
unsigned* g_noalloc_ptr[kMaxDevices] = {nullptr};
std::mutex g_noalloc_mutex;
thread_local std::string g_noalloc_err;

fdtd_status noalloc_fail(fdtd_status code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_noalloc_err = buf;
  return code;
}

// grid: x = blocks along a slice, y = slice.  Bit pattern of max|x| per slice, warp-reduced, one atomicMax per warp.
__global__ void __launch_bounds__(256) k_noalloc_amax(const float* __restrict__ x, size_t slice_len, unsigned* __restrict__ amax) {
  const float* xs = x + (size_t)blockIdx.y * slice_len;
  unsigned m = 0;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < slice_len; t += (size_t)gridDim.x * blockDim.x)
    m = max(m, __float_as_uint(fabsf(xs[t])));
  m = __reduce_max_sync(0xffffffffu, m);
  if ((threadIdx.x & 31) == 0) atomicMax(&amax[blockIdx.y], m);
}
template <int DT>
__global__ void __launch_bounds__(256) k_noalloc_encode(const float* __restrict__ x, size_t slice_len, void* codes, float* scales,
                                                        const unsigned* __restrict__ amax) {
  typedef typename Codec<DT>::code_t code_t;
  const size_t base = (size_t)blockIdx.y * slice_len;
  float inv = 1.0f, sc = 1.0f;
  if (DT == DT_E4M3S) {   // the arithmetic of k_codec_encode (R13)
    const float a = __uint_as_float(amax[blockIdx.y]);
    inv = a > 0.0f ? 448.0f / a : 0.0f;
    sc = a > 0.0f ? a / 448.0f : 0.0f;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) scales[blockIdx.y] = sc;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < slice_len; t += (size_t)gridDim.x * blockDim.x)
    reinterpret_cast<code_t*>(codes)[base + t] = Codec<DT>::enc(x[base + t], inv);
}
}  // namespace
extern "C" {

const char* fdtd_noalloc_last_error(void) { return g_noalloc_err.c_str(); }

fdtd_status fdtd_codec_encode_slices_noalloc(fdtd_dtype dt, const float* x_dev, int nslices, size_t slice_len, void* codes_dev,
                                             float* scales_dev, void* cuda_stream) {
  g_noalloc_err.clear();
  if (!x_dev || !codes_dev || !scales_dev) return noalloc_fail(FDTD_ERR_INVALID_ARG, "fdtd_codec_encode_slices_noalloc: NULL pointer");
  if (!dtype_ok((int)dt)) return noalloc_fail(FDTD_ERR_INVALID_ARG, "fdtd_codec_encode_slices_noalloc: unknown store dtype %d", (int)dt);
  if ((int)dt == DT_MX32)
    return noalloc_fail(FDTD_ERR_UNSUPPORTED, "fdtd_codec_encode_slices_noalloc: FDTD_F8E4M3_MX32 keeps its scale bytes behind the codes; use fdtd_codec_encode");
  if (nslices < 1 || slice_len < 1) return noalloc_fail(FDTD_ERR_INVALID_ARG, "fdtd_codec_encode_slices_noalloc: nslices and slice_len must be >= 1");
  if (nslices > FDTD_NOALLOC_MAX_SLICES)
    return noalloc_fail(FDTD_ERR_INVALID_ARG, "fdtd_codec_encode_slices_noalloc: %d slices exceed the static scratch array (FDTD_NOALLOC_MAX_SLICES = %d)",
                        nslices, FDTD_NOALLOC_MAX_SLICES);
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices)
    return noalloc_fail(FDTD_ERR_CUDA, "fdtd_codec_encode_slices_noalloc: cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
  unsigned* amax = nullptr;
  {
    // set-up, once per device, with that device current: the device address of the static array
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, g_noalloc_amax);
      if (e != cudaSuccess || !ptr)
        return noalloc_fail(FDTD_ERR_CUDA, "fdtd_codec_encode_slices_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
      g_noalloc_ptr[dev] = static_cast<unsigned*>(ptr);
    }
    amax = g_noalloc_ptr[dev];
  }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const unsigned bx = (unsigned)std::min<size_t>(std::max<size_t>((slice_len + 255) / 256, 1), 64);
  const dim3 g(bx, (unsigned)nslices);
  if ((int)dt == DT_E4M3S) {
    // the array keeps the last call's maxima: the words this call reduces into start at zero
    e = cudaMemsetAsync(amax, 0, (size_t)nslices * sizeof(unsigned), st);
    if (e != cudaSuccess) return noalloc_fail(FDTD_ERR_CUDA, "fdtd_codec_encode_slices_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
    k_noalloc_amax<<<g, 256, 0, st>>>(x_dev, slice_len, amax);
  }
  FDTD_DT_SWITCH((int)dt, (k_noalloc_encode<DT><<<g, 256, 0, st>>>(x_dev, slice_len, codes_dev, scales_dev, amax)))
  e = cudaGetLastError();
  if (e != cudaSuccess) return noalloc_fail(FDTD_ERR_CUDA, "fdtd_codec_encode_slices_noalloc: launch: %s", cudaGetErrorString(e));
  return FDTD_OK;
}

fdtd_status fdtd_profile_kernel(fdtd_sim* s, int id, int warm, int reps, double* ms_out, double* bytes_out) {
  if (!s || id < 0 || id > 22 || reps < 1 || warm < 0 || !ms_out) return FDTD_ERR_INVALID_ARG;
  if (!s->ws) return fail(s, FDTD_ERR_OOM, "no workspace");
  if (id >= 2 && !(s->flags & FDTD_WS_REVERSE)) return fail(s, FDTD_ERR_STATE, "needs a reverse workspace");
  if (((id >= 6 && id <= 8) || id == 2 || id == 4) && !s->forward_done) return fail(s, FDTD_ERR_STATE, "needs a completed forward run");
  if ((id == 21 || id == 22) && !(s->fuse_za && s->lb[1][0])) return fail(s, FDTD_ERR_UNSUPPORTED, "the fused adjoint path does not apply to this grid");
  if ((id == 9 || id == 10 || id == 19) && !s->can_fuse) return fail(s, FDTD_ERR_UNSUPPORTED, "the fused path needs nz % 4 == 0, pml_width % 4 == 0, pml_width >= 4");
  s->cur = s->stream;
  const int mrev = std::min(s->nsteps, s->nsteps / 2 + 2);   // nstate = mrev-1 falls between two slots
  // a split half-step is timed in the launch configuration of the real step: lean and general kernel side by side
  auto split_pair = [&](int which) {
    const bool was = s->parallel;
    s->parallel = s->aux[0] != nullptr;
    fork(s, 2);
    on(s, 1); launch_gen(s, which, 0);
    on(s, 0); launch_lean(s, which);
    join(s, 2);
    s->parallel = was;
  };
  auto once = [&]() {
    switch (id) {
      case 0: split_pair(0); break;
      case 1: split_pair(1); break;
      case 2: launch_inv_h(s, mrev, nullptr, 0); break;
      case 3: split_pair(2); break;
      case 4: {   // inverse-E and gradient side by side, as in the step
        const bool was = s->parallel;
        s->parallel = s->aux[0] != nullptr;
        fork(s, 2);
        on(s, 1); launch_grad(s);
        on(s, 0); launch_inv_e(s, mrev, nullptr, 0);
        join(s, 2);
        s->parallel = was;
        break;
      }
      case 5: split_pair(3); break;
      case 6: launch_record(s, s->nsteps, nullptr, 2); break;
      case 7: case 8:   // as the active reverse path launches it: in place (4 or 6 faces) or between the two buffers (6 faces)
        if (use_fused_reverse(s)) launch_inject(s, mrev, nullptr, id == 7 ? 1 : 0, 0, s->cb, s->cb ^ 1);
        else launch_inject(s, mrev, nullptr, id == 7 ? 1 : 0, 0);
        break;
      case 20: launch_grad(s); break;
      case 21: launch_fused_adj(s, s->acb, s->acb ^ 1, 0); break;   // adjoint marching kernel, alone
      case 22: {   // slab kernels of the fused adjoint path: adjoint of H, then adjoint of E on their boxes
        const AdjIO ia = adj_io(s, s->acb, s->acb ^ 1, false), ib = adj_io(s, s->acb, s->acb ^ 1, true);
        launch_gen(s, 2, 0, s->split[6], nullptr, &ia);
        launch_gen(s, 3, 0, s->split[7], nullptr, &ib);
        break;
      }
      case 9: launch_fused(s, false, s->cb, s->cb ^ 1); break;
      case 19: launch_fused(s, true, s->cb, s->cb ^ 1); break;   // reverse marching kernel (inverse-H + inverse-E), alone
      case 11: case 12: case 13: case 14: launch_lean(s, id - 11); break;     // lean kernel of split half-step id - 11, alone
      case 15: case 16: case 17: case 18: launch_gen(s, id - 15, 0); break;   // general kernel of split half-step id - 15, alone
      default: {
        const int cur = s->cb, oth = cur ^ 1;
        { const FieldIO io = io_of(s, cur, cur, oth, 1); launch_gen(s, 1, 0, s->split[5], &io); }
        { const FieldIO io = io_of(s, cur, oth, oth, 0); launch_gen(s, 0, 0, s->split[4], &io); }
      }
    }
  };
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  float ms = 0;
  cudaError_t ce = cudaEventCreate(&e0);
  if (ce == cudaSuccess) ce = cudaEventCreate(&e1);
  if (ce == cudaSuccess) {
    for (int r = 0; r < warm; ++r) once();
    ce = cudaEventRecord(e0, s->stream);
  }
  if (ce == cudaSuccess) {
    for (int r = 0; r < reps; ++r) once();
    ce = cudaEventRecord(e1, s->stream);
  }
  if (ce == cudaSuccess) ce = cudaEventSynchronize(e1);
  if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (ce != cudaSuccess) return fail(s, FDTD_ERR_CUDA, "fdtd_profile_kernel: %s", cudaGetErrorString(ce));
  CUDA_TRY(s, cudaGetLastError());
  *ms_out = (double)ms / reps;
  s->state_final = false;   // the fields are garbage now; the store of the last forward run stays readable (ids 6-8)
  if (bytes_out) {
    // algorithmic bytes per launch: f32 arrays read / written once, psi read+written in the slabs
    const double N = (double)s->d.N;
    double slab = 0;
    for (int a = 0; a < 3; ++a) slab += (double)psi_elems(s, a);
    double Ninner = 1;
    for (int a = 0; a < 3; ++a) Ninner *= std::max(0, s->n[a] - 2 * s->P - 2);
    double dcells = 0;
    if (s->has_design) {
      dcells = 1;
      for (int a = 0; a < 3; ++a) dcells *= std::max(0, std::min(s->dhi[a], s->n[a] - s->P - 1) - std::max(s->dlo[a], s->P + 1));
    }
    const double eb = elem_bytes_host(s->dtype);
    // shell cells k_inject handles, and those the inverse kernels inject themselves (interior cells of the two z faces)
    const double zin = (zface_fused(s) && !use_fused_reverse(s)) ? 2.0 * std::max(0, s->n[0] - 2 * s->P - 2) * std::max(0, s->n[1] - 2 * s->P - 2) : 0.0;
    const double shell = (double)s->st.cell_off[6] - zin;
    const double zbytes = (s->store_mode == 1 ? 1.0 : 3.0) * zin * (2 * eb + 4);
    double v = 0;
    switch (id) {
      case 0: v = 40 * N + 16 * slab; break;          // E rw (24) + H (12) + ce (4); 2 psi arrays rw per slab-cell-axis
      case 1: v = 36 * N + 16 * slab; break;          // H rw (24) + E (12)
      case 2: v = 36 * Ninner + zbytes; break;
      case 3: v = 36 * N + 16 * slab; break;          // lE rw + lH; lpsiH read (old) + written (new)
      case 4: v = 40 * Ninner + 28 * dcells + zbytes; break;   // E rw + H + ce; design: lE (12) + f64 acc rw (16)
      case 5: v = 40 * N + 16 * slab; break;          // lH rw + lE + ce
      case 6: v = (double)s->st.slot_values * 4 + (double)slot_bytes_host(s, s->dtype); break;   // f32 gathered, slot written (block scales included)
      case 7: case 8: v = (s->store_mode == 1 ? 1.0 : 3.0) * shell * (2 * eb + 4); break;   // two slots read, one f32 written per component
      case 20: v = 40 * dcells; break;   // lE (12) + f64 accumulator rw (16) + H of the design cells (12)
      case 21: {   // adjoint marching kernel: lambda_E, lambda_H read and written once, ce read; lambda_psi of the z axis rw
        const double rows = (double)std::max(0, s->n[0] - 2 * s->P - 2) * std::max(0, s->n[1] - 2 * s->P - 2);
        v = 52 * rows * s->n[2] + 32 * rows * 2 * s->P;
        break;
      }
      case 22: {   // its slab kernels: 36 B on the adjoint-of-H boxes, 40 B on the adjoint-of-E boxes, lambda_psi of the boxes' cells
        double in6 = 1, in7 = 1;
        for (int a = 0; a < 3; ++a) {
          in6 *= std::max(0, s->split[6].reg.hi[a] - s->split[6].reg.lo[a]);
          in7 *= std::max(0, s->split[7].reg.hi[a] - s->split[7].reg.lo[a]);
        }
        const double rows = (double)std::max(0, s->n[0] - 2 * s->P - 2) * std::max(0, s->n[1] - 2 * s->P - 2);
        v = 36 * (N - in6) + 40 * (N - in7) + 32 * (slab - rows * 2 * s->P);
        break;
      }
      case 19: {  // reverse marching kernel: 52 B per inner-interior cell
        v = 52 * Ninner;
        break;
      }
      case 9: {   // fused marching kernel: E, H read once and written once, ce read: 52 B per cell of [P+1, n-P)^3
        double c = 1;
        for (int a = 0; a < 3; ++a) c *= std::max(0, s->n[a] - 2 * s->P - 1);
        v = 52 * c;
        if (s->fuse_z) {
          // whole-row kernel (k_fused_fp): the rows of the lean x-y range over their full length, plus, on their z-slab cells,
          // psi_H of the z axis read and written (two arrays, ping-ponged) and psi_E read and written (two arrays): 32 B per cell
          const double rows = (double)std::max(0, s->n[0] - 2 * s->P - 1) * std::max(0, s->n[1] - 2 * s->P - 1);
          v = 52 * rows * s->n[2] + 32 * rows * 2 * s->P;
        }
        break;
      }
      case 11: case 12: case 13: case 14: case 15: case 16: case 17: case 18: {
        const int which = (id - 11) % 4;
        const Region& r = s->split[which].reg;
        double in = 1;
        for (int a = 0; a < 3; ++a) in *= std::max(0, r.hi[a] - r.lo[a]);
        if (!s->split[which].has_lean) in = 0;
        const double per = (which == 0 || which == 3) ? 40 : 36;
        v = id <= 14 ? per * in : per * (N - in) + 16 * slab;
        break;
      }
      default: {  // slab kernels of the fused path: H half-step on the complement of split 5, E half-step on that of split 4
        double in5 = 1, in4 = 1;
        for (int a = 0; a < 3; ++a) {
          in5 *= std::max(0, s->split[5].reg.hi[a] - s->split[5].reg.lo[a]);
          in4 *= std::max(0, s->split[4].reg.hi[a] - s->split[4].reg.lo[a]);
        }
        // psi of the boxes' cells only: the z-slab cells of the marching kernel's rows are counted with that kernel (id 9)
        const double zrows = s->fuse_z ? (double)std::max(0, s->n[0] - 2 * s->P - 1) * std::max(0, s->n[1] - 2 * s->P - 1) : 0.0;
        v = 36 * (N - in5) + 40 * (N - in4) + 32 * (slab - zrows * 2 * s->P);
      }
    }
    *bytes_out = v;
  }
  return FDTD_OK;
}

long long fdtd_debug_guard_check(fdtd_sim* s) {
  if (!s || !s->ws || !(s->flags & kWsGuard)) return -1;
  unsigned long long* cnt = reinterpret_cast<unsigned long long*>(s->ws + s->L.scratch);   // 16 bytes of scratch
  unsigned long long zero = 0, bad = 0;
  if (cudaStreamSynchronize(s->stream) != cudaSuccess) return -1;
  if (cudaMemcpy(cnt, &zero, 8, cudaMemcpyHostToDevice) != cudaSuccess) return -1;
  for (const auto& g : s->L.guards)
    k_guard_count<<<4, 256, 0, s->stream>>>(reinterpret_cast<const unsigned char*>(s->ws + g.first), g.second, cnt);
  if (cudaStreamSynchronize(s->stream) != cudaSuccess) return -1;
  if (cudaMemcpy(&bad, cnt, 8, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
  return (long long)bad;
}

fdtd_status fdtd_sync(fdtd_sim* s) {
  if (!s) return FDTD_ERR_INVALID_ARG;
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  CUDA_TRY(s, cudaGetLastError());
  reap_graphs(s);
  return FDTD_OK;
}

const char* fdtd_last_error(const fdtd_sim* s) { return s ? s->err.c_str() : "null handle"; }

void fdtd_destroy(fdtd_sim* s) {
  if (!s) return;
  cudaStreamSynchronize(s->stream);
  reap_graphs(s);
  for (int g = 0; g < 5; ++g)
    if (s->graph_cache[g]) cudaGraphExecDestroy(s->graph_cache[g]);
  for (int b = 0; b < 4; ++b) {
    if (s->aux[b]) cudaStreamDestroy(s->aux[b]);
    if (s->ev_join[b]) cudaEventDestroy(s->ev_join[b]);
  }
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  if (s->ev_mid) cudaEventDestroy(s->ev_mid);
  if (s->cap) cudaStreamDestroy(s->cap);
  delete s;
}

unsigned long long fdtd_launch_count(const fdtd_sim* s) { return s ? s->launches : 0; }

}  // extern "C"
