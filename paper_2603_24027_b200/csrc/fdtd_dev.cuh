// fdtd_dev.cuh — device-side data layout and small helpers shared by the kernels of libfdtd_b200.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdtd {

// Element offsets are 32-bit: fdtd_create rejects grids of 2^32 cells or more.
typedef unsigned idx_t;

// Everything a kernel needs to find its data.  Passed by value (__grid_constant__).
// Layout in HBM: six component-planar f32 arrays [nx][ny][nz], z fastest; ce = S/eps;
// CPML psi arrays stored compactly (slab cells only): psi?[c][t] belongs to component c and derivative axis
// a = (c+1+t)%3, its extent along a is 2P (low slab then high slab), the other two extents are the grid's.
struct Dev {
  int n[3];
  int P;
  idx_t sx, sy;      // strides of i and j (k stride = 1)
  long long N;
  float S;           // Courant number c*dt/dx (eq. 1)
  float* E[3];
  float* H[3];
  const float* ce;   // fl(S * fl(1/eps))
  float* psiE[3][2];
  float* psiH[3][2];
  const float* tab[3][6];  // per axis: bE cE kE bH cH kH (kE = 1/kappa - 1), length n[axis]
  // adjoint
  float* lE[3];
  float* lH[3];
  float* lpsiE[2][3][2];   // ping-pong buffers [buf][c][t]
  float* lpsiH[2][3][2];
  double* acc;             // dL/d(1/eps) / S accumulator over the design box
  int dlo[3], dhi[3];
  int has_design;
  int ce_keep;             // 1: the reverse kernels load ce with an L2 evict-last policy (grids whose ce fits a third of L2)
};

// Explicit input / output arrays of a forward general kernel: in place (out == the updated input) in the two-kernel
// path, other buffer in the fused path (ping-pong, fdtd_fused.cuh).
struct FieldIO {
  const float* E[3];
  const float* H[3];
  float* out[3];
  // psi_H of the z axis ([0]: the H_x term psiH[0][1], [1]: the H_y term psiH[1][0]): read from / written to.  The same arrays
  // except beside the whole-row marching kernel (k_fused_fz), whose halo workers need the old values while the owners write
  const float* pHz_in[2];
  float* pHz_out[2];
};
__device__ __host__ __forceinline__ void io_psi_inplace(FieldIO& io, const Dev& d) {
  io.pHz_in[0] = io.pHz_out[0] = d.psiH[0][1];
  io.pHz_in[1] = io.pHz_out[1] = d.psiH[1][0];
}

// Input / output arrays of an adjoint half-step: in place (out == in) in the two-kernel path, other buffer in the fused adjoint
// path (the adjoint marching kernel recomputes halo cells from OLD values, so lambda_E / lambda_H are ping-ponged there).
//  adjoint of H (A): reads lH, lEin; writes lEout.      adjoint of E (B): reads lEin (the NEW lambda_E), lH; writes lHout.
struct AdjIO {
  const float* lEin[3];
  const float* lH[3];
  float* lEout[3];
  float* lHout[3];
};
// A lean kernel's region (plain Yee cells) and the list of boxes that make up its complement (slab cells and the
// layers that touch them).  Each box has a class that says which CPML axes can occur in it (so the others compile
// out) and its own lane shape: G lanes along z (groups of V cells) x RW rows per warp, G*RW <= 32.
struct Region { int lo[3], hi[3]; };
struct FastDiv { unsigned mul, d; };   // x / d == __umulhi(x, mul) for the x range checked on the host (d == 1: x)
enum { CLS_X = 0, CLS_Y = 1, CLS_Z = 2 };   // X: any axis; Y: no x terms; Z: z terms only
struct BoxList {
  int nb;
  int lo[6][3], hi[6][3];
  int cls[6];
  int G[6], RW[6];
  unsigned ginv[6];        // (lane * ginv) >> 16 == lane / G for lane < 32
  int nbx[6], nby[6];      // blocks along z; blocks along the flattened (x plane, y row) index
  int rows[6];             // (x planes) * (y rows) of the box
  FastDiv dnbx[6], drow[6];   // division by nbx; by the number of y rows per plane
  int off[7];
};
__device__ __forceinline__ unsigned fast_div(unsigned x, const FastDiv f) { return f.d == 1u ? x : __umulhi(x, f.mul); }

__device__ __forceinline__ bool in_slab(int i, int n, int P) { return i < P || i >= n - P; }
__device__ __forceinline__ int slab_s(int i, int n, int P) { return i < P ? i : i - (n - 2 * P); }
__device__ __forceinline__ idx_t psi_index(const Dev& d, int a, int i, int j, int k) {
  const int P2 = 2 * d.P;
  if (a == 0) return ((idx_t)slab_s(i, d.n[0], d.P) * d.n[1] + j) * d.n[2] + k;
  if (a == 1) return ((idx_t)i * P2 + slab_s(j, d.n[1], d.P)) * d.n[2] + k;
  return ((idx_t)i * d.n[1] + j) * P2 + slab_s(k, d.n[2], d.P);
}

// V consecutive z cells held by one thread (V = 4: one 16-byte access; V = 1: scalar path for odd shapes).
template <int V> struct VF { float v[V]; };
template <int V> __device__ __forceinline__ VF<V> ldv(const float* p) {
  VF<V> r;
  if constexpr (V == 4) {
    const float4 t = *reinterpret_cast<const float4*>(p);
    r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
  } else if constexpr (V == 2) {
    const float2 t = *reinterpret_cast<const float2*>(p);
    r.v[0] = t.x; r.v[1] = t.y;
  } else {
    r.v[0] = *p;
  }
  return r;
}
// ce in the reverse run: read twice per step in the same phase (inverse-E and adjoint-of-E kernels, side by side) and never
// written.  Where the whole array fits a third of the L2 (d.ce_keep, set by the host) it is loaded with an evict-last policy so
// that the second reader — and the next step — find it there.  Measured A/B (FDTD_CE_KEEP=0/1, one box, forward + reverse runs back
// to back): C2 reverse 58.4 -> 55.9 us per step, C3 235.0 -> 232.9 and, with ce still resident, C3 forward 140.0 -> 137.8; in the
// default bench (L2 flushed between steps, 2000-step runs) C2 reverse 57.8 -> 57.2.  On 512^3 (ce = 537 MB) the hint costs 0.15 %,
// hence the switch.  The forward kernels keep the plain load: the same hint there measured 5 % slower on C3.
template <int V> __device__ __forceinline__ VF<V> ldv_ce(const Dev& d, const float* p) {
  VF<V> r;
  if constexpr (V == 4) {
    if (d.ce_keep) {
      unsigned long long pol;
      asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
      asm("ld.global.nc.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
          : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "l"(p), "l"(pol));
      return r;
    }
  }
  r = ldv<V>(p);
  return r;
}
template <int V> __device__ __forceinline__ void stv(float* p, const VF<V>& r) {
  if constexpr (V == 4) {
    *reinterpret_cast<float4*>(p) = make_float4(r.v[0], r.v[1], r.v[2], r.v[3]);
  } else if constexpr (V == 2) {
    *reinterpret_cast<float2*>(p) = make_float2(r.v[0], r.v[1]);
  } else {
    *p = r.v[0];
  }
}
template <int V> __device__ __forceinline__ VF<V> zerov() {
  VF<V> r;
#pragma unroll
  for (int v = 0; v < V; ++v) r.v[v] = 0.0f;
  return r;
}

// One Yee component update with its two CPML terms, in the canonical operation order (R3):
//   x = fma(coef, d1 - d2, x);  slab a1: psi1 = fma(b1, psi1, c1*d1), x = fma(coef, fma(k1, d1, psi1), x);
//   slab a2: psi2 = fma(b2, psi2, c2*d2), x = fma(-coef, fma(k2, d2, psi2), x).
// E half-step: coef = ce.  H half-step: coef = -S.  (Compiled with -fmad=false: every fma here is explicit.)
__device__ __forceinline__ float yee_update(float x, float coef, float d1, float d2, bool s1, float b1, float c1,
                                            float k1, float& psi1, bool s2, float b2, float c2, float k2,
                                            float& psi2) {
  x = fmaf(coef, d1 - d2, x);
  if (s1) {
    const float ps = fmaf(b1, psi1, c1 * d1);
    psi1 = ps;
    x = fmaf(coef, fmaf(k1, d1, ps), x);
  }
  if (s2) {
    const float ps = fmaf(b2, psi2, c2 * d2);
    psi2 = ps;
    x = fmaf(-coef, fmaf(k2, d2, ps), x);
  }
  return x;
}

// Transposed CPML term: g = cotangent reaching the (d/kappa + psi) sum; returns W = the cotangent of d beyond
// the plain Yee part, and the new lambda_psi (R9 step 1/5).
__device__ __forceinline__ float cpml_adjoint_term(float g, float lpsi_old, float bt, float ct, float kt,
                                                   float& lpsi_new) {
  const float phi = lpsi_old + g;
  lpsi_new = bt * phi;
  return fmaf(ct, phi, kt * g);
}

}  // namespace fdtd
