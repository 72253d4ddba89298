// fdtd_stencil.cuh — the bandwidth-bound stencil kernels: forward E / H half-steps with fused CPML, the
// inverse half-steps of the reverse run, the adjoint half-steps with the transposed CPML, gradient accumulation.
//
// Work split: every half-step is two launches that touch disjoint cells.
//  * a LEAN kernel over the box of plain Yee cells (no CPML term, no wall): few registers, high occupancy,
//    one thread = V = 4 consecutive z cells (16-byte accesses, a warp covers 512 contiguous bytes), TY rows per block,
//    one x plane per block; x/y/z neighbours come from L1/L2 (DRAM traffic measured = algorithmic bytes);
//  * a GENERAL kernel over the complement (the six slab boxes plus the layers that touch them): the same update
//    with the CPML psi recursion fused in, V = 2 to halve its register footprint, and a per-box lane shape so that
//    the thin z slabs still fill their warps.
#pragma once
#include "fdtd_dev.cuh"
#include "fdtd_store.cuh"

namespace fdtd {

#ifndef FDTD_TY
#define FDTD_TY 4
#endif
#ifndef FDTD_SWEEP_FLIP
#define FDTD_SWEEP_FLIP 1
#endif
constexpr bool SWEEP_FLIP = FDTD_SWEEP_FLIP != 0;
constexpr int TY = FDTD_TY;   // rows per block, one warp per row (4: measured best of 2 / 4 / 8 / 16 on C2, C3, C4)

// block / thread -> box b and (i, j, first k) inside the box list of a GENERAL kernel.  The (x plane, y row) pairs of a box
// are numbered consecutively and cut into blocks of TY * RW rows, so that thin boxes (a y slab has only P rows per plane,
// a z slab packs RW rows into a warp) leave no half-empty block per plane; a warp covers G z-groups x RW rows.
// FLIP: the kernel walks its blocks in the opposite order.  The H-type half-steps (forward H, adjoint of E, inverse E) sweep the
// grid downwards and the E-type ones upwards, so that each phase starts on the planes the previous phase touched last and
// finds them in L2 (an LRU cache swept cyclically by a working set larger than itself hits almost never).
template <int V, bool FLIP = false>
__device__ __forceinline__ bool box_decode(const BoxList& B, int& b, int& i, int& j, int& k0) {
  const unsigned blk = FLIP ? (unsigned)B.off[B.nb] - 1u - blockIdx.x : blockIdx.x;
  b = 0;
#pragma unroll
  for (int g = 1; g < 6; ++g) b += (g < B.nb && blk >= (unsigned)B.off[g]);
  const unsigned local = blk - B.off[b];
  const unsigned by = fast_div(local, B.dnbx[b]);          // block along the flattened rows
  const unsigned bx = local - by * B.nbx[b];               // block along z
  const int G = B.G[b], RW = B.RW[b];
  const int yl = (int)((threadIdx.x * B.ginv[b]) >> 16), zl = (int)threadIdx.x - yl * G;
  const unsigned row = (by * TY + threadIdx.y) * RW + yl;  // flattened (plane, row) index inside the box
  const unsigned pl = fast_div(row, B.drow[b]);
  i = B.lo[b][0] + (int)pl;
  j = B.lo[b][1] + (int)(row - pl * B.drow[b].d);
  k0 = B.lo[b][2] + ((int)bx * G + zl) * V;
  return yl < RW && row < (unsigned)B.rows[b] && k0 < B.hi[b][2];
}

// A general kernel body is instantiated per box class: HX / HY say whether CPML terms of the x / y axis (and, for
// the adjoint, neighbour terms across that axis) can occur in the box; z terms are always compiled in.
#define FDTD_CLASS_DISPATCH(BODY, ...)                                    \
  switch (B.cls[b]) {                                                     \
    case CLS_X: BODY<V, true, true>(__VA_ARGS__); break;                  \
    case CLS_Y: BODY<V, false, true>(__VA_ARGS__); break;                 \
    default: BODY<V, false, false>(__VA_ARGS__); break;                   \
  }

// ---------------------------------------------------------------------------------------------------------
// Forward half-steps on the slab boxes.  Layout of both bodies: all loads first; per component the plain update
// x = fma(coef, d1 - d2, x), then its CPML term of axis a1, then of axis a2 (canonical order, R3), each term
// one block under a thread-level condition (x: block-uniform, y: row-uniform, z: uniform over the thread's group,
// since P % V == 0); PEC-masked nodes are zeroed once at the end.
// ---------------------------------------------------------------------------------------------------------
// one CPML term over the thread's V cells: psi = fma(b, psi, c*d); x = fma(sgn*coef, fma(k, d, psi), x)
template <int V, bool ZAXIS>
__device__ __forceinline__ void cpml_term(VF<V>& x, VF<V>& psi, const VF<V>& coef, const float sgn, const float* dv,
                                          const float* b, const float* c, const float* k) {
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const int t = ZAXIS ? v : 0;                 // coefficients vary along z only
    const float ps = fmaf(b[t], psi.v[v], c[t] * dv[v]);
    psi.v[v] = ps;
    x.v[v] = fmaf(sgn * coef.v[v], fmaf(k[t], dv[v], ps), x.v[v]);
  }
}

// Forward E half-step (SURVEY 8(a) rows A1 + A3):  E_c += ce * (d_a1^- H_b1 - d_a2^- H_b2) + CPML terms,
// tangential E on the three low PEC walls held at zero.  DESIGN.md R1-R5.
template <int V, bool HX, bool HY>
__device__ __forceinline__ void gen_e_body(const Dev& d, const int i, const int j, const int k0, const FieldIO& io) {
  const int nx = d.n[0], ny = d.n[1], nz = d.n[2], P = d.P;
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * ny + j) * nz + k0;
  const bool xs = HX && P > 0 && in_slab(i, nx, P);
  const bool ys = HY && P > 0 && in_slab(j, ny, P);
  const bool zs = P > 0 && in_slab(k0, nz, P);

  const VF<V> hx = ldv<V>(io.H[0] + q), hy = ldv<V>(io.H[1] + q), hz = ldv<V>(io.H[2] + q);
  VF<V> hy_xm = zerov<V>(), hz_xm = zerov<V>(), hx_ym = zerov<V>(), hz_ym = zerov<V>();
  if (i > 0) {
    hy_xm = ldv<V>(io.H[1] + q - sx);
    hz_xm = ldv<V>(io.H[2] + q - sx);
  }
  if (j > 0) {
    hx_ym = ldv<V>(io.H[0] + q - sy);
    hz_ym = ldv<V>(io.H[2] + q - sy);
  }
  float hx_z0 = 0.0f, hy_z0 = 0.0f;
  if (k0 > 0) {
    hx_z0 = io.H[0][q - 1];
    hy_z0 = io.H[1][q - 1];
  }
  VF<V> ex = ldv<V>(io.E[0] + q), ey = ldv<V>(io.E[1] + q), ez = ldv<V>(io.E[2] + q);
  const VF<V> ce = ldv<V>(d.ce + q);
  // psi_E[c][t]: (0,0)=Ex/y (0,1)=Ex/z (1,0)=Ey/z (1,1)=Ey/x (2,0)=Ez/x (2,1)=Ez/y
  VF<V> p_ey_x, p_ez_x, p_ex_y, p_ez_y, p_ex_z, p_ey_z;
  idx_t qx = 0, qy = 0, qz = 0;
  float bx = 0, cx = 0, kx = 0, by = 0, cy = 0, ky = 0, bz[V], cz[V], kz[V];
  if (xs) {
    qx = psi_index(d, 0, i, j, k0);
    p_ey_x = ldv<V>(d.psiE[1][1] + qx);
    p_ez_x = ldv<V>(d.psiE[2][0] + qx);
    bx = __ldg(d.tab[0][0] + i); cx = __ldg(d.tab[0][1] + i); kx = __ldg(d.tab[0][2] + i);
  }
  if (ys) {
    qy = psi_index(d, 1, i, j, k0);
    p_ex_y = ldv<V>(d.psiE[0][0] + qy);
    p_ez_y = ldv<V>(d.psiE[2][1] + qy);
    by = __ldg(d.tab[1][0] + j); cy = __ldg(d.tab[1][1] + j); ky = __ldg(d.tab[1][2] + j);
  }
  if (zs) {
    qz = psi_index(d, 2, i, j, k0);
    p_ex_z = ldv<V>(d.psiE[0][1] + qz);
    p_ey_z = ldv<V>(d.psiE[1][0] + qz);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      bz[v] = __ldg(d.tab[2][0] + k0 + v); cz[v] = __ldg(d.tab[2][1] + k0 + v); kz[v] = __ldg(d.tab[2][2] + k0 + v);
    }
  }
  // the six one-sided differences
  float dy_hz[V], dz_hy[V], dz_hx[V], dx_hz[V], dx_hy[V], dy_hx[V];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
    const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
    dy_hz[v] = hz.v[v] - hz_ym.v[v];
    dz_hy[v] = hy.v[v] - hy_zm;
    dz_hx[v] = hx.v[v] - hx_zm;
    dx_hz[v] = hz.v[v] - hz_xm.v[v];
    dx_hy[v] = hy.v[v] - hy_xm.v[v];
    dy_hx[v] = hx.v[v] - hx_ym.v[v];
  }
  // Ex: a1 = y (d_y^- Hz), a2 = z (d_z^- Hy)
#pragma unroll
  for (int v = 0; v < V; ++v) ex.v[v] = fmaf(ce.v[v], dy_hz[v] - dz_hy[v], ex.v[v]);
  if (ys) cpml_term<V, false>(ex, p_ex_y, ce, 1.0f, dy_hz, &by, &cy, &ky);
  if (zs) cpml_term<V, true>(ex, p_ex_z, ce, -1.0f, dz_hy, bz, cz, kz);
  // Ey: a1 = z (d_z^- Hx), a2 = x (d_x^- Hz)
#pragma unroll
  for (int v = 0; v < V; ++v) ey.v[v] = fmaf(ce.v[v], dz_hx[v] - dx_hz[v], ey.v[v]);
  if (zs) cpml_term<V, true>(ey, p_ey_z, ce, 1.0f, dz_hx, bz, cz, kz);
  if (xs) cpml_term<V, false>(ey, p_ey_x, ce, -1.0f, dx_hz, &bx, &cx, &kx);
  // Ez: a1 = x (d_x^- Hy), a2 = y (d_y^- Hx)
#pragma unroll
  for (int v = 0; v < V; ++v) ez.v[v] = fmaf(ce.v[v], dx_hy[v] - dy_hx[v], ez.v[v]);
  if (xs) cpml_term<V, false>(ez, p_ez_x, ce, 1.0f, dx_hy, &bx, &cx, &kx);
  if (ys) cpml_term<V, false>(ez, p_ez_y, ce, -1.0f, dy_hx, &by, &cy, &ky);
  // PEC walls (rare): a masked node keeps E = 0 and its psi untouched, as if the update had skipped it
  if (i == 0 || j == 0 || k0 == 0) {
    auto keep = [&](VF<V>& psi, const float* arr, idx_t qq, bool active, bool ij_masked, bool k_masks) {
      if (!active) return;
      const VF<V> old = ldv<V>(arr + qq);
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (ij_masked || (k_masks && k0 + v == 0)) psi.v[v] = old.v[v];
    };
    keep(p_ex_y, d.psiE[0][0], qy, ys, j == 0, true);
    keep(p_ex_z, d.psiE[0][1], qz, zs, j == 0, true);
    keep(p_ey_z, d.psiE[1][0], qz, zs, i == 0, true);
    keep(p_ey_x, d.psiE[1][1], qx, xs, i == 0, true);
    keep(p_ez_x, d.psiE[2][0], qx, xs, i == 0 || j == 0, false);
    keep(p_ez_y, d.psiE[2][1], qy, ys, i == 0 || j == 0, false);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int k = k0 + v;
      if (j == 0 || k == 0) ex.v[v] = 0.0f;
      if (k == 0 || i == 0) ey.v[v] = 0.0f;
      if (i == 0 || j == 0) ez.v[v] = 0.0f;
    }
  }
  stv<V>(io.out[0] + q, ex);
  stv<V>(io.out[1] + q, ey);
  stv<V>(io.out[2] + q, ez);
  if (xs) {
    stv<V>(d.psiE[1][1] + qx, p_ey_x);
    stv<V>(d.psiE[2][0] + qx, p_ez_x);
  }
  if (ys) {
    stv<V>(d.psiE[0][0] + qy, p_ex_y);
    stv<V>(d.psiE[2][1] + qy, p_ez_y);
  }
  if (zs) {
    stv<V>(d.psiE[0][1] + qz, p_ex_z);
    stv<V>(d.psiE[1][0] + qz, p_ey_z);
  }
}

// Forward H half-step (rows A2 + A4):  H_c -= S * (d_a1^+ E_b1 - d_a2^+ E_b2) + CPML terms; ghost E[n] = 0.
template <int V, bool HX, bool HY>
__device__ __forceinline__ void gen_h_body(const Dev& d, const int i, const int j, const int k0, const FieldIO& io) {
  const int nx = d.n[0], ny = d.n[1], nz = d.n[2], P = d.P;
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * ny + j) * nz + k0;
  const bool xs = HX && P > 0 && in_slab(i, nx, P);
  const bool ys = HY && P > 0 && in_slab(j, ny, P);
  const bool zs = P > 0 && in_slab(k0, nz, P);

  const VF<V> ex = ldv<V>(io.E[0] + q), ey = ldv<V>(io.E[1] + q), ez = ldv<V>(io.E[2] + q);
  VF<V> ey_xp = zerov<V>(), ez_xp = zerov<V>(), ex_yp = zerov<V>(), ez_yp = zerov<V>();
  if (i + 1 < nx) {
    ey_xp = ldv<V>(io.E[1] + q + sx);
    ez_xp = ldv<V>(io.E[2] + q + sx);
  }
  if (j + 1 < ny) {
    ex_yp = ldv<V>(io.E[0] + q + sy);
    ez_yp = ldv<V>(io.E[2] + q + sy);
  }
  float ex_zp = 0.0f, ey_zp = 0.0f;
  if (k0 + V < nz) {
    ex_zp = io.E[0][q + V];
    ey_zp = io.E[1][q + V];
  }
  VF<V> hx = ldv<V>(io.H[0] + q), hy = ldv<V>(io.H[1] + q), hz = ldv<V>(io.H[2] + q);
  // psi_H[c][t]: (0,0)=Hx/y (0,1)=Hx/z (1,0)=Hy/z (1,1)=Hy/x (2,0)=Hz/x (2,1)=Hz/y
  VF<V> p_hy_x, p_hz_x, p_hx_y, p_hz_y, p_hx_z, p_hy_z;
  idx_t qx = 0, qy = 0, qz = 0;
  float bx = 0, cx = 0, kx = 0, by = 0, cy = 0, ky = 0, bz[V], cz[V], kz[V];
  if (xs) {
    qx = psi_index(d, 0, i, j, k0);
    p_hy_x = ldv<V>(d.psiH[1][1] + qx);
    p_hz_x = ldv<V>(d.psiH[2][0] + qx);
    bx = __ldg(d.tab[0][3] + i); cx = __ldg(d.tab[0][4] + i); kx = __ldg(d.tab[0][5] + i);
  }
  if (ys) {
    qy = psi_index(d, 1, i, j, k0);
    p_hx_y = ldv<V>(d.psiH[0][0] + qy);
    p_hz_y = ldv<V>(d.psiH[2][1] + qy);
    by = __ldg(d.tab[1][3] + j); cy = __ldg(d.tab[1][4] + j); ky = __ldg(d.tab[1][5] + j);
  }
  if (zs) {
    qz = psi_index(d, 2, i, j, k0);
    p_hx_z = ldv<V>(io.pHz_in[0] + qz);
    p_hy_z = ldv<V>(io.pHz_in[1] + qz);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      bz[v] = __ldg(d.tab[2][3] + k0 + v); cz[v] = __ldg(d.tab[2][4] + k0 + v); kz[v] = __ldg(d.tab[2][5] + k0 + v);
    }
  }
  float dy_ez[V], dz_ey[V], dz_ex[V], dx_ez[V], dx_ey[V], dy_ex[V];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float ey_zq = v == V - 1 ? ey_zp : ey.v[v < V - 1 ? v + 1 : v];
    const float ex_zq = v == V - 1 ? ex_zp : ex.v[v < V - 1 ? v + 1 : v];
    dy_ez[v] = ez_yp.v[v] - ez.v[v];
    dz_ey[v] = ey_zq - ey.v[v];
    dz_ex[v] = ex_zq - ex.v[v];
    dx_ez[v] = ez_xp.v[v] - ez.v[v];
    dx_ey[v] = ey_xp.v[v] - ey.v[v];
    dy_ex[v] = ex_yp.v[v] - ex.v[v];
  }
  VF<V> mS;
#pragma unroll
  for (int v = 0; v < V; ++v) mS.v[v] = -d.S;
  // Hx: a1 = y (d_y^+ Ez), a2 = z (d_z^+ Ey)
#pragma unroll
  for (int v = 0; v < V; ++v) hx.v[v] = fmaf(mS.v[v], dy_ez[v] - dz_ey[v], hx.v[v]);
  if (ys) cpml_term<V, false>(hx, p_hx_y, mS, 1.0f, dy_ez, &by, &cy, &ky);
  if (zs) cpml_term<V, true>(hx, p_hx_z, mS, -1.0f, dz_ey, bz, cz, kz);
  // Hy: a1 = z (d_z^+ Ex), a2 = x (d_x^+ Ez)
#pragma unroll
  for (int v = 0; v < V; ++v) hy.v[v] = fmaf(mS.v[v], dz_ex[v] - dx_ez[v], hy.v[v]);
  if (zs) cpml_term<V, true>(hy, p_hy_z, mS, 1.0f, dz_ex, bz, cz, kz);
  if (xs) cpml_term<V, false>(hy, p_hy_x, mS, -1.0f, dx_ez, &bx, &cx, &kx);
  // Hz: a1 = x (d_x^+ Ey), a2 = y (d_y^+ Ex)
#pragma unroll
  for (int v = 0; v < V; ++v) hz.v[v] = fmaf(mS.v[v], dx_ey[v] - dy_ex[v], hz.v[v]);
  if (xs) cpml_term<V, false>(hz, p_hz_x, mS, 1.0f, dx_ey, &bx, &cx, &kx);
  if (ys) cpml_term<V, false>(hz, p_hz_y, mS, -1.0f, dy_ex, &by, &cy, &ky);
  stv<V>(io.out[0] + q, hx);
  stv<V>(io.out[1] + q, hy);
  stv<V>(io.out[2] + q, hz);
  if (xs) {
    stv<V>(d.psiH[1][1] + qx, p_hy_x);
    stv<V>(d.psiH[2][0] + qx, p_hz_x);
  }
  if (ys) {
    stv<V>(d.psiH[0][0] + qy, p_hx_y);
    stv<V>(d.psiH[2][1] + qy, p_hz_y);
  }
  if (zs) {
    stv<V>(io.pHz_out[0] + qz, p_hx_z);
    stv<V>(io.pHz_out[1] + qz, p_hy_z);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Reverse run, primal reconstruction on the inner interior (row R2).  One thread = one (i, j, z-group);
// elements outside the inner interior are neither computed nor written.  Grid: x = z groups, y = rows from P+1, z = planes
// from P+1.
// ---------------------------------------------------------------------------------------------------------
// Z-face injection inside the inverse kernels (ZF, vector path): the interface cells of the two z faces, (i, j, P) and
// (i, j, n-P-1), are the elements just outside a row's inner-interior range — element 0 of its first group of 4 cells and
// element 3 of its last one.  The thread that owns such a group fetches the dequantised, interpolated shell values (row R1)
// itself and stores the group whole.  Done from k_inject, these cells are a scatter of 4-byte writes at a stride of one row
// (one 32-byte DRAM sector read, modified and written per value: 1.4 M of them per half-step on 512^3), which cost the reverse
// step 137 us of 3177 on C4 although inject moves 1 % of the step's bytes; here they ride on lines that are written anyway, and
// the inverse kernels lose their element-wise stores at the row ends.  Interior cells of a z face belong to no other face, so
// the ownership rule of DESIGN.md R9 is untouched; k_inject keeps the x and y faces (contiguous along z).
struct ZInj {
  StoreDev st;
  int m_base;
  const int* step_dev;
  int interp;
};
// values of the three components (magnetic: H, else E) of z-face `side` at (i, j); returns a bit mask of the components stored
template <int DT>
__device__ __forceinline__ unsigned zface_fetch(const Dev& d, const ZInj& z, const FetchPlan& p, int side, int i, int j, bool magnetic,
                                                float out[3]) {
  const StoreDev& s = z.st;
  const int f = 4 + side;
  const long long e = (long long)(i - d.P) * s.dv[f] + (j - d.P);
  const long long fs = (long long)s.du[f] * s.dv[f];
  const long long nb = s.blkc_off[f + 1] - s.blkc_off[f], b0 = s.blk_off[f] + (e >> 5);
  unsigned mask = 0;
  if (s.mode == 1) {   // tangential store: H (x, y) on the low face, E (x, y) on the high face
    if (side != (magnetic ? 0 : 1)) return 0;
#pragma unroll
    for (int cc = 0; cc < 2; ++cc) {
      out[cc] = fetch_value<DT>(s, p, f * 6 + (magnetic ? 3 + cc : cc), s.val_off[f] + cc * fs + e, b0 + cc * nb);
      mask |= 1u << cc;
    }
    return mask;
  }
#pragma unroll
  for (int cc = 0; cc < 3; ++cc) {
    const int comp = magnetic ? 3 + cc : cc;
    out[cc] = fetch_value<DT>(s, p, f * 6 + comp, s.val_off[f] + comp * fs + e, b0 + comp * nb);
  }
  return 7u;
}

// inverse of the H half-step:  H^{m-1/2} = H^{m+1/2} + S * curl^+(E^m)
template <int V, int DT, bool ZF>
__global__ void __launch_bounds__(32 * TY) k_inv_h(const __grid_constant__ Dev d, const __grid_constant__ ZInj z) {
  const int nx = d.n[0], ny = d.n[1], nz = d.n[2], P = d.P;
  const int klo = P + 1, khi = nz - P - 1;
  const int k0 = (klo / V) * V + (blockIdx.x * 32 + threadIdx.x) * V;
  const int j = P + 1 + blockIdx.y * TY + threadIdx.y;
  const int i = P + 1 + blockIdx.z;
  if (k0 >= khi || j >= ny - P - 1 || i >= nx - P - 1) return;
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * ny + j) * nz + k0;
  const float S = d.S;
  const bool part_lo = k0 < klo, part_hi = k0 + V > khi;
  float zlo[3], zhi[3];
  unsigned mlo = 0, mhi = 0;
  if (ZF && (part_lo || part_hi)) {   // shell values first: their loads overlap with everything below
    const FetchPlan p = make_plan(cur_step(z.m_base, z.step_dev) - 1, z.st.nsteps, z.st.k, z.st.nslots, z.interp);
    if (part_lo) mlo = zface_fetch<DT>(d, z, p, 0, i, j, true, zlo);
    if (part_hi) mhi = zface_fetch<DT>(d, z, p, 1, i, j, true, zhi);
  }
  const VF<V> ex = ldv<V>(d.E[0] + q), ey = ldv<V>(d.E[1] + q), ez = ldv<V>(d.E[2] + q);
  const VF<V> ey_xp = ldv<V>(d.E[1] + q + sx), ez_xp = ldv<V>(d.E[2] + q + sx);
  const VF<V> ex_yp = ldv<V>(d.E[0] + q + sy), ez_yp = ldv<V>(d.E[2] + q + sy);
  float ex_zp = 0.0f, ey_zp = 0.0f;
  if (k0 + V < nz) {
    ex_zp = d.E[0][q + V];
    ey_zp = d.E[1][q + V];
  }
  VF<V> hx = ldv<V>(d.H[0] + q), hy = ldv<V>(d.H[1] + q), hz = ldv<V>(d.H[2] + q);
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const int k = k0 + v;
    if (k < klo || k >= khi) continue;
    const float ey_zq = v == V - 1 ? ey_zp : ey.v[v < V - 1 ? v + 1 : v];
    const float ex_zq = v == V - 1 ? ex_zp : ex.v[v < V - 1 ? v + 1 : v];
    hx.v[v] = fmaf(S, (ez_yp.v[v] - ez.v[v]) - (ey_zq - ey.v[v]), hx.v[v]);
    hy.v[v] = fmaf(S, (ex_zq - ex.v[v]) - (ez_xp.v[v] - ez.v[v]), hy.v[v]);
    hz.v[v] = fmaf(S, (ey_xp.v[v] - ey.v[v]) - (ex_yp.v[v] - ex.v[v]), hz.v[v]);
  }
  if (ZF) {
    // the shell elements take the injected values (components the store does not hold keep what the arrays hold)
    if (part_lo) {
      if (mlo & 1u) hx.v[0] = zlo[0];
      if (mlo & 2u) hy.v[0] = zlo[1];
      if (mlo & 4u) hz.v[0] = zlo[2];
    }
    if (part_hi) {
      if (mhi & 1u) hx.v[V - 1] = zhi[0];
      if (mhi & 2u) hy.v[V - 1] = zhi[1];
      if (mhi & 4u) hz.v[V - 1] = zhi[2];
    }
    stv<V>(d.H[0] + q, hx);
    stv<V>(d.H[1] + q, hy);
    stv<V>(d.H[2] + q, hz);
    return;
  }
  // a group that straddles the shell must not touch the shell cells: inject H runs concurrently with this kernel
  if (!part_lo && !part_hi) {
    stv<V>(d.H[0] + q, hx);
    stv<V>(d.H[1] + q, hy);
    stv<V>(d.H[2] + q, hz);
  } else {
#pragma unroll
    for (int v = 0; v < V; ++v)
      if (k0 + v >= klo && k0 + v < khi) {
        d.H[0][q + v] = hx.v[v];
        d.H[1][q + v] = hy.v[v];
        d.H[2][q + v] = hz.v[v];
      }
  }
}

// shell-cell gradient term in its dE form (R9 step 4), shared with k_inject's arithmetic:
//   acc += sum_c lE_c * ((E_old - E_new)_c / ce)   on design ∩ shell
__device__ __forceinline__ void shell_grad(const Dev& d, int i, int j, int k, idx_t qc, const float eold[3], const float enew[3], float cev) {
  if (!(d.has_design && i >= d.dlo[0] && i < d.dhi[0] && j >= d.dlo[1] && j < d.dhi[1] && k >= d.dlo[2] && k < d.dhi[2])) return;
  const double ce = (double)cev;
  double sacc = 0.0;
#pragma unroll
  for (int cc = 0; cc < 3; ++cc) {
    const float dE = eold[cc] - enew[cc];
    sacc += (double)d.lE[cc][qc] * ((double)dE / ce);
  }
  const long long ei = ((long long)(i - d.dlo[0]) * (d.dhi[1] - d.dlo[1]) + (j - d.dlo[1])) * (d.dhi[2] - d.dlo[2]) + (k - d.dlo[2]);
  d.acc[ei] += sacc;
}

// inverse of the E half-step (row R2):  E^{m-1} = E^m - ce * curl^-(H^{m-1/2})   on the inner interior
template <int V, int DT, bool ZF>
__global__ void __launch_bounds__(32 * TY) k_inv_e(const __grid_constant__ Dev d, const __grid_constant__ ZInj z) {
  const int nx = d.n[0], ny = d.n[1], nz = d.n[2], P = d.P;
  const int klo = P + 1, khi = nz - P - 1;
  const int k0 = (klo / V) * V + (blockIdx.x * 32 + threadIdx.x) * V;
  const int j = P + 1 + blockIdx.y * TY + threadIdx.y;
  const int i = SWEEP_FLIP ? nx - P - 2 - (int)blockIdx.z : P + 1 + (int)blockIdx.z;
  if (k0 >= khi || j >= ny - P - 1 || i >= nx - P - 1) return;
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * ny + j) * nz + k0;
  const bool part_lo = k0 < klo, part_hi = k0 + V > khi;
  float zlo[3], zhi[3];
  unsigned mlo = 0, mhi = 0;
  if (ZF && (part_lo || part_hi)) {
    const FetchPlan p = make_plan(cur_step(z.m_base, z.step_dev) - 1, z.st.nsteps, z.st.k, z.st.nslots, z.interp);
    if (part_lo) mlo = zface_fetch<DT>(d, z, p, 0, i, j, false, zlo);
    if (part_hi) mhi = zface_fetch<DT>(d, z, p, 1, i, j, false, zhi);
  }
  const VF<V> hx = ldv<V>(d.H[0] + q), hy = ldv<V>(d.H[1] + q), hz = ldv<V>(d.H[2] + q);
  const VF<V> hy_xm = ldv<V>(d.H[1] + q - sx), hz_xm = ldv<V>(d.H[2] + q - sx);
  const VF<V> hx_ym = ldv<V>(d.H[0] + q - sy), hz_ym = ldv<V>(d.H[2] + q - sy);
  const float hx_z0 = d.H[0][q - 1], hy_z0 = d.H[1][q - 1];   // k0 >= 1: the inner interior starts at P + 1
  VF<V> ex = ldv<V>(d.E[0] + q), ey = ldv<V>(d.E[1] + q), ez = ldv<V>(d.E[2] + q);
  const VF<V> ce = ldv_ce<V>(d, d.ce + q);
  const float eold_lo[3] = {ex.v[0], ey.v[0], ez.v[0]}, eold_hi[3] = {ex.v[V - 1], ey.v[V - 1], ez.v[V - 1]};
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
    const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
    const float cx = (hz.v[v] - hz_ym.v[v]) - (hy.v[v] - hy_zm);
    const float cy = (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]);
    const float cz = (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym.v[v]);
    ex.v[v] = fmaf(-ce.v[v], cx, ex.v[v]);
    ey.v[v] = fmaf(-ce.v[v], cy, ey.v[v]);
    ez.v[v] = fmaf(-ce.v[v], cz, ez.v[v]);
  }
  if (ZF) {
    // Shell elements: E_new = the injected value (a component the store does not hold keeps E_old: tangential store, where the
    // design box cannot touch the shell); the gradient term of design ∩ shell uses E_old, exactly as k_inject does.
    if (part_lo) {
      float en[3] = {eold_lo[0], eold_lo[1], eold_lo[2]};
#pragma unroll
      for (int cc = 0; cc < 3; ++cc)
        if (mlo >> cc & 1u) en[cc] = zlo[cc];
      if (mlo == 7u) shell_grad(d, i, j, k0, q, eold_lo, en, ce.v[0]);
      ex.v[0] = en[0]; ey.v[0] = en[1]; ez.v[0] = en[2];
    }
    if (part_hi) {
      float en[3] = {eold_hi[0], eold_hi[1], eold_hi[2]};
#pragma unroll
      for (int cc = 0; cc < 3; ++cc)
        if (mhi >> cc & 1u) en[cc] = zhi[cc];
      if (mhi == 7u) shell_grad(d, i, j, k0 + V - 1, q + (V - 1), eold_hi, en, ce.v[V - 1]);
      ex.v[V - 1] = en[0]; ey.v[V - 1] = en[1]; ez.v[V - 1] = en[2];
    }
    stv<V>(d.E[0] + q, ex);
    stv<V>(d.E[1] + q, ey);
    stv<V>(d.E[2] + q, ez);
    return;
  }
  if (!part_lo && !part_hi) {   // see k_inv_h: inject E runs concurrently on the shell cells
    stv<V>(d.E[0] + q, ex);
    stv<V>(d.E[1] + q, ey);
    stv<V>(d.E[2] + q, ez);
  } else {
#pragma unroll
    for (int v = 0; v < V; ++v)
      if (k0 + v >= klo && k0 + v < khi) {
        d.E[0][q + v] = ex.v[v];
        d.E[1][q + v] = ey.v[v];
        d.E[2][q + v] = ez.v[v];
      }
  }
}

// gradient term (row R3) on design ∩ inner interior:  acc += sum_c lE_c * curl^-(H^{m-1/2})_c  (f64 accumulator).
// Its own kernel so that the inverse-E sweep above stays a lean f32 kernel; it reads H^{m-1/2} and lE, both
// read-only in this phase (it runs beside k_inv_e and the adjoint-E kernels).  One thread per design cell.
__global__ void __launch_bounds__(256) k_grad(const __grid_constant__ Dev d) {
  const int P = d.P;
  int lo[3], ext[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    lo[a] = max(d.dlo[a], P + 1);
    ext[a] = min(d.dhi[a], d.n[a] - P - 1) - lo[a];
  }
  const idx_t t = blockIdx.x * 256u + threadIdx.x;   // flat index over the clipped design box, z fastest
  if (t >= (idx_t)ext[0] * ext[1] * ext[2]) return;
  const idx_t row = t / (idx_t)ext[2];
  const int k = lo[2] + (int)(t - row * ext[2]);
  const int i = lo[0] + (int)(row / (idx_t)ext[1]), j = lo[1] + (int)(row % (idx_t)ext[1]);
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * d.n[1] + j) * d.n[2] + k;
  const float hx = d.H[0][q], hy = d.H[1][q], hz = d.H[2][q];
  const float cx = (hz - d.H[2][q - sy]) - (hy - d.H[1][q - 1]);
  const float cy = (hx - d.H[0][q - 1]) - (hz - d.H[2][q - sx]);
  const float cz = (hy - d.H[1][q - sx]) - (hx - d.H[0][q - sy]);
  double s = 0.0;
  s += (double)d.lE[0][q] * (double)cx;
  s += (double)d.lE[1][q] * (double)cy;
  s += (double)d.lE[2][q] * (double)cz;
  const idx_t e = ((idx_t)(i - d.dlo[0]) * (d.dhi[1] - d.dlo[1]) + (j - d.dlo[1])) * (d.dhi[2] - d.dlo[2]) + (k - d.dlo[2]);
  d.acc[e] += s;
}

// ---------------------------------------------------------------------------------------------------------
// Adjoint of the H half-step (row R4): lE_e += -S * curl^-(lH)_e on all cells (PEC-masked nodes -> 0), plus the
// transposed CPML: for the H term (c,t) with axis a and field b:  g = -S*s*lH_c, W = cH*(lpsiH + g) + kH*g,
// lpsiH <- bH*(lpsiH + g), lE_b -= d_a^-(W).   lpsiH is ping-ponged (pb = buffer read, pb^1 = written), because
// W at the low-side neighbour needs that neighbour's OLD lpsiH.
// Layout of the body: plain update of the three components, then one correction block per CPML axis in the
// order z, y, x — the canonical subtraction order of every component (lE_x: z,y; lE_y: z,x; lE_z: y,x).  A block is
// entered when this cell or its low-side neighbour along that axis is a slab cell (x, y: uniform over the warp's
// row).  Inside a block the arithmetic is unconditional: the coefficient tables are zero outside the slabs and a
// missing lpsi reads as zero, so absent terms evaluate to W = 0 exactly.
// ---------------------------------------------------------------------------------------------------------
template <int V, bool HX, bool HY>
__device__ __forceinline__ void gen_adj_h_body(const Dev& d, const int i, const int j, const int k0, int pb, const AdjIO& io) {
  const int nx = d.n[0], ny = d.n[1], nz = d.n[2], P = d.P;
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * ny + j) * nz + k0;
  const float S = d.S;
  const int nb = pb ^ 1;
  const VF<V> lhx = ldv<V>(io.lH[0] + q), lhy = ldv<V>(io.lH[1] + q), lhz = ldv<V>(io.lH[2] + q);
  VF<V> lhy_xm = zerov<V>(), lhz_xm = zerov<V>(), lhx_ym = zerov<V>(), lhz_ym = zerov<V>();
  if (i > 0) {
    lhy_xm = ldv<V>(io.lH[1] + q - sx);
    lhz_xm = ldv<V>(io.lH[2] + q - sx);
  }
  if (j > 0) {
    lhx_ym = ldv<V>(io.lH[0] + q - sy);
    lhz_ym = ldv<V>(io.lH[2] + q - sy);
  }
  float lhx_z0 = 0.0f, lhy_z0 = 0.0f;
  if (k0 > 0) {
    lhx_z0 = io.lH[0][q - 1];
    lhy_z0 = io.lH[1][q - 1];
  }
  VF<V> lex = ldv<V>(io.lEin[0] + q), ley = ldv<V>(io.lEin[1] + q), lez = ldv<V>(io.lEin[2] + q);

  const bool xs = HX && P > 0 && in_slab(i, nx, P), xsm = HX && P > 0 && i > 0 && in_slab(i - 1, nx, P);
  const bool ys = HY && P > 0 && in_slab(j, ny, P), ysm = HY && P > 0 && j > 0 && in_slab(j - 1, ny, P);
  const bool zs0 = P > 0 && in_slab(k0, nz, P);                 // V = 4: a group never straddles a slab edge
  const bool zsm0 = P > 0 && k0 > 0 && in_slab(k0 - 1, nz, P);
  const bool zany = zs0 || zsm0;                                // (P % V == 0, so only element 0 can have a slab neighbour alone)
  // issue the lpsi loads of every active block before any arithmetic
  VF<V> o01 = zerov<V>(), o10 = zerov<V>(), o00 = zerov<V>(), o21 = zerov<V>(), o11 = zerov<V>(), o20 = zerov<V>();
  VF<V> o00m = zerov<V>(), o21m = zerov<V>(), o11m = zerov<V>(), o20m = zerov<V>();
  float o01_z0 = 0.0f, o10_z0 = 0.0f;
  idx_t qx = 0, qy = 0, qz = 0;
  if (zs0) {
    qz = psi_index(d, 2, i, j, k0);
    o01 = ldv<V>(d.lpsiH[pb][0][1] + qz);
    o10 = ldv<V>(d.lpsiH[pb][1][0] + qz);
  }
  if (zsm0) {
    const idx_t qm = psi_index(d, 2, i, j, k0 - 1);
    o01_z0 = d.lpsiH[pb][0][1][qm];
    o10_z0 = d.lpsiH[pb][1][0][qm];
  }
  if (ys) {
    qy = psi_index(d, 1, i, j, k0);
    o00 = ldv<V>(d.lpsiH[pb][0][0] + qy);
    o21 = ldv<V>(d.lpsiH[pb][2][1] + qy);
  }
  if (ysm) {
    const idx_t qm = psi_index(d, 1, i, j - 1, k0);
    o00m = ldv<V>(d.lpsiH[pb][0][0] + qm);
    o21m = ldv<V>(d.lpsiH[pb][2][1] + qm);
  }
  if (xs) {
    qx = psi_index(d, 0, i, j, k0);
    o11 = ldv<V>(d.lpsiH[pb][1][1] + qx);
    o20 = ldv<V>(d.lpsiH[pb][2][0] + qx);
  }
  if (xsm) {
    const idx_t qm = psi_index(d, 0, i - 1, j, k0);
    o11m = ldv<V>(d.lpsiH[pb][1][1] + qm);
    o20m = ldv<V>(d.lpsiH[pb][2][0] + qm);
  }

  // --- plain part ---
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float lhy_zm = v == 0 ? lhy_z0 : lhy.v[v > 0 ? v - 1 : 0];
    const float lhx_zm = v == 0 ? lhx_z0 : lhx.v[v > 0 ? v - 1 : 0];
    lex.v[v] = fmaf(-S, (lhz.v[v] - lhz_ym.v[v]) - (lhy.v[v] - lhy_zm), lex.v[v]);
    ley.v[v] = fmaf(-S, (lhx.v[v] - lhx_zm) - (lhz.v[v] - lhz_xm.v[v]), ley.v[v]);
    lez.v[v] = fmaf(-S, (lhy.v[v] - lhy_xm.v[v]) - (lhx.v[v] - lhx_ym.v[v]), lez.v[v]);
  }
  float dummy;
  // --- z block: terms (c=0,t=1: g = +S*lH_x -> lE_y) and (c=1,t=0: g = -S*lH_y -> lE_x) ---
  if (zany) {
    VF<V> n01, n10;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int k = k0 + v;
      const float bz = __ldg(d.tab[2][3] + k), cz = __ldg(d.tab[2][4] + k), kz = __ldg(d.tab[2][5] + k);
      const float czm = k > 0 ? __ldg(d.tab[2][4] + k - 1) : 0.0f, kzm = k > 0 ? __ldg(d.tab[2][5] + k - 1) : 0.0f;
      const float lhy_zm = v == 0 ? lhy_z0 : lhy.v[v > 0 ? v - 1 : 0];
      const float lhx_zm = v == 0 ? lhx_z0 : lhx.v[v > 0 ? v - 1 : 0];
      const float p01 = v == 0 ? o01_z0 : o01.v[v > 0 ? v - 1 : 0];
      const float p10 = v == 0 ? o10_z0 : o10.v[v > 0 ? v - 1 : 0];
      const float w01 = cpml_adjoint_term(S * lhx.v[v], o01.v[v], bz, cz, kz, n01.v[v]);
      const float w10 = cpml_adjoint_term(-S * lhy.v[v], o10.v[v], bz, cz, kz, n10.v[v]);
      const float w01m = cpml_adjoint_term(S * lhx_zm, p01, 0.0f, czm, kzm, dummy);
      const float w10m = cpml_adjoint_term(-S * lhy_zm, p10, 0.0f, czm, kzm, dummy);
      lex.v[v] -= (w10 - w10m);
      ley.v[v] -= (w01 - w01m);
    }
    if (zs0) {
      stv<V>(d.lpsiH[nb][0][1] + qz, n01);
      stv<V>(d.lpsiH[nb][1][0] + qz, n10);
    }
  }
  // --- y block: terms (c=0,t=0: g = -S*lH_x -> lE_z) and (c=2,t=1: g = +S*lH_z -> lE_x) ---
  if (HY && (ys || ysm)) {
    const float by = __ldg(d.tab[1][3] + j), cy = __ldg(d.tab[1][4] + j), ky = __ldg(d.tab[1][5] + j);
    const float cym = j > 0 ? __ldg(d.tab[1][4] + j - 1) : 0.0f, kym = j > 0 ? __ldg(d.tab[1][5] + j - 1) : 0.0f;
    VF<V> n00, n21;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const float w00 = cpml_adjoint_term(-S * lhx.v[v], o00.v[v], by, cy, ky, n00.v[v]);
      const float w21 = cpml_adjoint_term(S * lhz.v[v], o21.v[v], by, cy, ky, n21.v[v]);
      const float w00m = cpml_adjoint_term(-S * lhx_ym.v[v], o00m.v[v], 0.0f, cym, kym, dummy);
      const float w21m = cpml_adjoint_term(S * lhz_ym.v[v], o21m.v[v], 0.0f, cym, kym, dummy);
      lex.v[v] -= (w21 - w21m);
      lez.v[v] -= (w00 - w00m);
    }
    if (ys) {
      stv<V>(d.lpsiH[nb][0][0] + qy, n00);
      stv<V>(d.lpsiH[nb][2][1] + qy, n21);
    }
  }
  // --- x block: terms (c=1,t=1: g = +S*lH_y -> lE_z) and (c=2,t=0: g = -S*lH_z -> lE_y) ---
  if (HX && (xs || xsm)) {
    const float bx = __ldg(d.tab[0][3] + i), cx = __ldg(d.tab[0][4] + i), kx = __ldg(d.tab[0][5] + i);
    const float cxm = i > 0 ? __ldg(d.tab[0][4] + i - 1) : 0.0f, kxm = i > 0 ? __ldg(d.tab[0][5] + i - 1) : 0.0f;
    VF<V> n11, n20;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const float w11 = cpml_adjoint_term(S * lhy.v[v], o11.v[v], bx, cx, kx, n11.v[v]);
      const float w20 = cpml_adjoint_term(-S * lhz.v[v], o20.v[v], bx, cx, kx, n20.v[v]);
      const float w11m = cpml_adjoint_term(S * lhy_xm.v[v], o11m.v[v], 0.0f, cxm, kxm, dummy);
      const float w20m = cpml_adjoint_term(-S * lhz_xm.v[v], o20m.v[v], 0.0f, cxm, kxm, dummy);
      ley.v[v] -= (w20 - w20m);
      lez.v[v] -= (w11 - w11m);
    }
    if (xs) {
      stv<V>(d.lpsiH[nb][1][1] + qx, n11);
      stv<V>(d.lpsiH[nb][2][0] + qx, n20);
    }
  }
  // --- PEC-masked nodes (low walls) ---
  if (i == 0 || j == 0 || k0 == 0) {
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int k = k0 + v;
      if (j == 0 || k == 0) lex.v[v] = 0.0f;
      if (k == 0 || i == 0) ley.v[v] = 0.0f;
      if (i == 0 || j == 0) lez.v[v] = 0.0f;
    }
  }
  stv<V>(io.lEout[0] + q, lex);
  stv<V>(io.lEout[1] + q, ley);
  stv<V>(io.lEout[2] + q, lez);
}

// ---------------------------------------------------------------------------------------------------------
// Adjoint of the E half-step (row R4): with G_c = ce*lE_c,  lH_h += curl^+(G)_h on all cells, plus the transposed
// CPML: for the E term (c,t) with axis a and field b: g = s*G_c, W = cE*(lpsiE + g) + kE*g, lpsiE <- bE*(lpsiE+g)
// (skipped on PEC-masked E_c nodes: W = 0, lpsiE kept), lH_b -= d_a^+(W).
// Same layout as gen_adj_h_body: plain part, then the z, y, x correction blocks (lH_x: z,y; lH_y: z,x; lH_z: y,x).
// ---------------------------------------------------------------------------------------------------------
template <int V, bool HX, bool HY>
__device__ __forceinline__ void gen_adj_e_body(const Dev& d, const int i, const int j, const int k0, int pb, const AdjIO& io) {
  const int nx = d.n[0], ny = d.n[1], nz = d.n[2], P = d.P;
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * ny + j) * nz + k0;
  const int nb = pb ^ 1;
  const VF<V> ce = ldv_ce<V>(d, d.ce + q);
  VF<V> gx = ldv<V>(io.lEin[0] + q), gy = ldv<V>(io.lEin[1] + q), gz = ldv<V>(io.lEin[2] + q);
  VF<V> gy_xp = zerov<V>(), gz_xp = zerov<V>(), gx_yp = zerov<V>(), gz_yp = zerov<V>();
  VF<V> ce_xp = zerov<V>(), ce_yp = zerov<V>();
  float gx_zp = 0.0f, gy_zp = 0.0f, ce_zp = 0.0f;
  if (i + 1 < nx) {
    ce_xp = ldv_ce<V>(d, d.ce + q + sx);
    gy_xp = ldv<V>(io.lEin[1] + q + sx);
    gz_xp = ldv<V>(io.lEin[2] + q + sx);
  }
  if (j + 1 < ny) {
    ce_yp = ldv_ce<V>(d, d.ce + q + sy);
    gx_yp = ldv<V>(io.lEin[0] + q + sy);
    gz_yp = ldv<V>(io.lEin[2] + q + sy);
  }
  if (k0 + V < nz) {
    ce_zp = d.ce[q + V];
    gx_zp = io.lEin[0][q + V];
    gy_zp = io.lEin[1][q + V];
  }
  VF<V> lhx = ldv<V>(io.lH[0] + q), lhy = ldv<V>(io.lH[1] + q), lhz = ldv<V>(io.lH[2] + q);

  const bool xs = HX && P > 0 && in_slab(i, nx, P), xsp = HX && P > 0 && i + 1 < nx && in_slab(i + 1, nx, P);
  const bool ys = HY && P > 0 && in_slab(j, ny, P), ysp = HY && P > 0 && j + 1 < ny && in_slab(j + 1, ny, P);
  const bool zs0 = P > 0 && in_slab(k0, nz, P);
  const bool zsp0 = P > 0 && k0 + V < nz && in_slab(k0 + V, nz, P);
  const bool zany = zs0 || zsp0;
  // old lambda_psi_E: axis x terms (c=1,t=1: Ey) (c=2,t=0: Ez); axis y (c=0,t=0: Ex) (c=2,t=1: Ez); axis z (c=0,t=1: Ex) (c=1,t=0: Ey)
  VF<V> o01 = zerov<V>(), o10 = zerov<V>(), o00 = zerov<V>(), o21 = zerov<V>(), o11 = zerov<V>(), o20 = zerov<V>();
  VF<V> o00p = zerov<V>(), o21p = zerov<V>(), o11p = zerov<V>(), o20p = zerov<V>();
  float o01_zp = 0.0f, o10_zp = 0.0f;
  idx_t qx = 0, qy = 0, qz = 0;
  if (zs0) {
    qz = psi_index(d, 2, i, j, k0);
    o01 = ldv<V>(d.lpsiE[pb][0][1] + qz);
    o10 = ldv<V>(d.lpsiE[pb][1][0] + qz);
  }
  if (zsp0) {
    const idx_t qp = psi_index(d, 2, i, j, k0 + V);
    o01_zp = d.lpsiE[pb][0][1][qp];
    o10_zp = d.lpsiE[pb][1][0][qp];
  }
  if (ys) {
    qy = psi_index(d, 1, i, j, k0);
    o00 = ldv<V>(d.lpsiE[pb][0][0] + qy);
    o21 = ldv<V>(d.lpsiE[pb][2][1] + qy);
  }
  if (ysp) {
    const idx_t qp = psi_index(d, 1, i, j + 1, k0);
    o00p = ldv<V>(d.lpsiE[pb][0][0] + qp);
    o21p = ldv<V>(d.lpsiE[pb][2][1] + qp);
  }
  if (xs) {
    qx = psi_index(d, 0, i, j, k0);
    o11 = ldv<V>(d.lpsiE[pb][1][1] + qx);
    o20 = ldv<V>(d.lpsiE[pb][2][0] + qx);
  }
  if (xsp) {
    const idx_t qp = psi_index(d, 0, i + 1, j, k0);
    o11p = ldv<V>(d.lpsiE[pb][1][1] + qp);
    o20p = ldv<V>(d.lpsiE[pb][2][0] + qp);
  }

  // --- G = ce * lE at the cell and its high-side neighbours; plain part ---
  gx_zp = ce_zp * gx_zp;
  gy_zp = ce_zp * gy_zp;
#pragma unroll
  for (int v = 0; v < V; ++v) {
    gx.v[v] = ce.v[v] * gx.v[v];
    gy.v[v] = ce.v[v] * gy.v[v];
    gz.v[v] = ce.v[v] * gz.v[v];
    gy_xp.v[v] = ce_xp.v[v] * gy_xp.v[v];
    gz_xp.v[v] = ce_xp.v[v] * gz_xp.v[v];
    gx_yp.v[v] = ce_yp.v[v] * gx_yp.v[v];
    gz_yp.v[v] = ce_yp.v[v] * gz_yp.v[v];
  }
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float gx_zq = v == V - 1 ? gx_zp : gx.v[v < V - 1 ? v + 1 : v];
    const float gy_zq = v == V - 1 ? gy_zp : gy.v[v < V - 1 ? v + 1 : v];
    lhx.v[v] = lhx.v[v] + ((gz_yp.v[v] - gz.v[v]) - (gy_zq - gy.v[v]));
    lhy.v[v] = lhy.v[v] + ((gx_zq - gx.v[v]) - (gz_xp.v[v] - gz.v[v]));
    lhz.v[v] = lhz.v[v] + ((gy_xp.v[v] - gy.v[v]) - (gx_yp.v[v] - gx.v[v]));
  }
  float dummy;
  // PEC masks of E_c at q: Ex: j==0||k==0, Ey: k==0||i==0, Ez: i==0||j==0; at the +a neighbour only the other axis counts
  // --- z block: terms (c=0,t=1: g = -G_x -> lH_y) and (c=1,t=0: g = +G_y -> lH_x) ---
  if (zany) {
    VF<V> n01 = o01, n10 = o10;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int k = k0 + v;
      const float bz = __ldg(d.tab[2][0] + k), cz = __ldg(d.tab[2][1] + k), kz = __ldg(d.tab[2][2] + k);
      const float czp = k + 1 < nz ? __ldg(d.tab[2][1] + k + 1) : 0.0f, kzp = k + 1 < nz ? __ldg(d.tab[2][2] + k + 1) : 0.0f;
      const float gx_zq = v == V - 1 ? gx_zp : gx.v[v < V - 1 ? v + 1 : v];
      const float gy_zq = v == V - 1 ? gy_zp : gy.v[v < V - 1 ? v + 1 : v];
      const float p01 = v == V - 1 ? o01_zp : o01.v[v < V - 1 ? v + 1 : v];
      const float p10 = v == V - 1 ? o10_zp : o10.v[v < V - 1 ? v + 1 : v];
      float w01 = 0.0f, w10 = 0.0f, w01p = 0.0f, w10p = 0.0f;
      if (!(j == 0 || k == 0)) w01 = cpml_adjoint_term(-gx.v[v], o01.v[v], bz, cz, kz, n01.v[v]);
      if (!(k == 0 || i == 0)) w10 = cpml_adjoint_term(gy.v[v], o10.v[v], bz, cz, kz, n10.v[v]);
      if (j != 0) w01p = cpml_adjoint_term(-gx_zq, p01, 0.0f, czp, kzp, dummy);
      if (i != 0) w10p = cpml_adjoint_term(gy_zq, p10, 0.0f, czp, kzp, dummy);
      lhx.v[v] -= (w10p - w10);
      lhy.v[v] -= (w01p - w01);
    }
    if (zs0) {
      stv<V>(d.lpsiE[nb][0][1] + qz, n01);
      stv<V>(d.lpsiE[nb][1][0] + qz, n10);
    }
  }
  // --- y block: terms (c=0,t=0: g = +G_x -> lH_z) and (c=2,t=1: g = -G_z -> lH_x) ---
  if (HY && (ys || ysp)) {
    const float by = __ldg(d.tab[1][0] + j), cy = __ldg(d.tab[1][1] + j), ky = __ldg(d.tab[1][2] + j);
    const float cyp = j + 1 < ny ? __ldg(d.tab[1][1] + j + 1) : 0.0f, kyp = j + 1 < ny ? __ldg(d.tab[1][2] + j + 1) : 0.0f;
    VF<V> n00 = o00, n21 = o21;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int k = k0 + v;
      float w00 = 0.0f, w21 = 0.0f, w00p = 0.0f, w21p = 0.0f;
      if (!(j == 0 || k == 0)) w00 = cpml_adjoint_term(gx.v[v], o00.v[v], by, cy, ky, n00.v[v]);
      if (!(i == 0 || j == 0)) w21 = cpml_adjoint_term(-gz.v[v], o21.v[v], by, cy, ky, n21.v[v]);
      if (k != 0) w00p = cpml_adjoint_term(gx_yp.v[v], o00p.v[v], 0.0f, cyp, kyp, dummy);
      if (i != 0) w21p = cpml_adjoint_term(-gz_yp.v[v], o21p.v[v], 0.0f, cyp, kyp, dummy);
      lhx.v[v] -= (w21p - w21);
      lhz.v[v] -= (w00p - w00);
    }
    if (ys) {
      stv<V>(d.lpsiE[nb][0][0] + qy, n00);
      stv<V>(d.lpsiE[nb][2][1] + qy, n21);
    }
  }
  // --- x block: terms (c=1,t=1: g = -G_y -> lH_z) and (c=2,t=0: g = +G_z -> lH_y) ---
  if (HX && (xs || xsp)) {
    const float bx = __ldg(d.tab[0][0] + i), cx = __ldg(d.tab[0][1] + i), kx = __ldg(d.tab[0][2] + i);
    const float cxp = i + 1 < nx ? __ldg(d.tab[0][1] + i + 1) : 0.0f, kxp = i + 1 < nx ? __ldg(d.tab[0][2] + i + 1) : 0.0f;
    VF<V> n11 = o11, n20 = o20;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int k = k0 + v;
      float w11 = 0.0f, w20 = 0.0f, w11p = 0.0f, w20p = 0.0f;
      if (!(k == 0 || i == 0)) w11 = cpml_adjoint_term(-gy.v[v], o11.v[v], bx, cx, kx, n11.v[v]);
      if (!(i == 0 || j == 0)) w20 = cpml_adjoint_term(gz.v[v], o20.v[v], bx, cx, kx, n20.v[v]);
      if (k != 0) w11p = cpml_adjoint_term(-gy_xp.v[v], o11p.v[v], 0.0f, cxp, kxp, dummy);
      if (j != 0) w20p = cpml_adjoint_term(gz_xp.v[v], o20p.v[v], 0.0f, cxp, kxp, dummy);
      lhy.v[v] -= (w20p - w20);
      lhz.v[v] -= (w11p - w11);
    }
    if (xs) {
      stv<V>(d.lpsiE[nb][1][1] + qx, n11);
      stv<V>(d.lpsiE[nb][2][0] + qx, n20);
    }
  }
  stv<V>(io.lHout[0] + q, lhx);
  stv<V>(io.lHout[1] + q, lhy);
  stv<V>(io.lHout[2] + q, lhz);
}

// ---------------------------------------------------------------------------------------------------------
// GENERAL kernels: one launch per half-step over the box list; each block runs the body of its box's class.
// ---------------------------------------------------------------------------------------------------------
template <int V>
__global__ void __launch_bounds__(32 * TY) k_gen_e(const __grid_constant__ Dev d, const __grid_constant__ BoxList B,
                                                   const __grid_constant__ FieldIO io) {
  int b, i, j, k0;
  if (!box_decode<V>(B, b, i, j, k0)) return;
  FDTD_CLASS_DISPATCH(gen_e_body, d, i, j, k0, io)
}
template <int V>
__global__ void __launch_bounds__(32 * TY) k_gen_h(const __grid_constant__ Dev d, const __grid_constant__ BoxList B,
                                                   const __grid_constant__ FieldIO io) {
  int b, i, j, k0;
  if (!box_decode<V, SWEEP_FLIP>(B, b, i, j, k0)) return;
  FDTD_CLASS_DISPATCH(gen_h_body, d, i, j, k0, io)
}
template <int V>
__global__ void __launch_bounds__(32 * TY) k_gen_adj_h(const __grid_constant__ Dev d, const __grid_constant__ BoxList B, int pb,
                                                       const __grid_constant__ AdjIO io) {
  int b, i, j, k0;
  if (!box_decode<V>(B, b, i, j, k0)) return;
  FDTD_CLASS_DISPATCH(gen_adj_h_body, d, i, j, k0, pb, io)
}
template <int V>
__global__ void __launch_bounds__(32 * TY) k_gen_adj_e(const __grid_constant__ Dev d, const __grid_constant__ BoxList B, int pb,
                                                       const __grid_constant__ AdjIO io) {
  int b, i, j, k0;
  if (!box_decode<V, SWEEP_FLIP>(B, b, i, j, k0)) return;
  FDTD_CLASS_DISPATCH(gen_adj_e_body, d, i, j, k0, pb, io)
}

// ---------------------------------------------------------------------------------------------------------
// LEAN kernels: plain Yee cells only (region chosen by the host so that no CPML term, no PEC mask and no ghost
// applies, and — for the adjoint — no neighbour W term either).  Grid: x = z groups, y = row tiles, z = planes.
// Same canonical arithmetic as the general kernels (R3), so results are bit-identical to them.
// ---------------------------------------------------------------------------------------------------------
template <int V, bool FLIP = false>
__device__ __forceinline__ bool lean_decode(const Region& r, int& i, int& j, int& k0) {
  k0 = r.lo[2] + (blockIdx.x * 32 + threadIdx.x) * V;
  j = r.lo[1] + blockIdx.y * TY + threadIdx.y;
  i = FLIP ? r.hi[0] - 1 - (int)blockIdx.z : r.lo[0] + (int)blockIdx.z;
  return k0 < r.hi[2] && j < r.hi[1];
}

// ADJ = false: forward E half-step   E_c  = fma(ce, curl^-(H)_c,  E_c)      (row A1)
// ADJ = true : adjoint of H half-step lE_c = fma(-S, curl^-(lH)_c, lE_c)     (row R4)
template <int V, bool ADJ>
__device__ __forceinline__ void lean_curlm_body(const Dev& d, const int i, const int j, const int k0) {
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * d.n[1] + j) * d.n[2] + k0;
  const float* const* in = ADJ ? d.lH : d.H;
  float* const* out = ADJ ? d.lE : d.E;
  const VF<V> hx = ldv<V>(in[0] + q), hy = ldv<V>(in[1] + q), hz = ldv<V>(in[2] + q);
  const VF<V> hy_xm = ldv<V>(in[1] + q - sx), hz_xm = ldv<V>(in[2] + q - sx);
  const VF<V> hx_ym = ldv<V>(in[0] + q - sy), hz_ym = ldv<V>(in[2] + q - sy);
  const float hx_z0 = in[0][q - 1], hy_z0 = in[1][q - 1];
  VF<V> ex = ldv<V>(out[0] + q), ey = ldv<V>(out[1] + q), ez = ldv<V>(out[2] + q);
  VF<V> ce;
  if (!ADJ) ce = ldv<V>(d.ce + q);
  const float mS = -d.S;
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
    const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
    const float c = ADJ ? mS : ce.v[v];
    ex.v[v] = fmaf(c, (hz.v[v] - hz_ym.v[v]) - (hy.v[v] - hy_zm), ex.v[v]);
    ey.v[v] = fmaf(c, (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]), ey.v[v]);
    ez.v[v] = fmaf(c, (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym.v[v]), ez.v[v]);
  }
  stv<V>(out[0] + q, ex);
  stv<V>(out[1] + q, ey);
  stv<V>(out[2] + q, ez);
}

// forward H half-step on plain cells:  H_c = fma(-S, curl^+(E)_c, H_c)   (row A2)
template <int V>
__device__ __forceinline__ void lean_h_body(const Dev& d, const int i, const int j, const int k0) {
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * d.n[1] + j) * d.n[2] + k0;
  const VF<V> ex = ldv<V>(d.E[0] + q), ey = ldv<V>(d.E[1] + q), ez = ldv<V>(d.E[2] + q);
  const VF<V> ey_xp = ldv<V>(d.E[1] + q + sx), ez_xp = ldv<V>(d.E[2] + q + sx);
  const VF<V> ex_yp = ldv<V>(d.E[0] + q + sy), ez_yp = ldv<V>(d.E[2] + q + sy);
  const float ex_zp = d.E[0][q + V], ey_zp = d.E[1][q + V];
  VF<V> hx = ldv<V>(d.H[0] + q), hy = ldv<V>(d.H[1] + q), hz = ldv<V>(d.H[2] + q);
  const float mS = -d.S;
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float ey_zq = v == V - 1 ? ey_zp : ey.v[v < V - 1 ? v + 1 : v];
    const float ex_zq = v == V - 1 ? ex_zp : ex.v[v < V - 1 ? v + 1 : v];
    hx.v[v] = fmaf(mS, (ez_yp.v[v] - ez.v[v]) - (ey_zq - ey.v[v]), hx.v[v]);
    hy.v[v] = fmaf(mS, (ex_zq - ex.v[v]) - (ez_xp.v[v] - ez.v[v]), hy.v[v]);
    hz.v[v] = fmaf(mS, (ey_xp.v[v] - ey.v[v]) - (ex_yp.v[v] - ex.v[v]), hz.v[v]);
  }
  stv<V>(d.H[0] + q, hx);
  stv<V>(d.H[1] + q, hy);
  stv<V>(d.H[2] + q, hz);
}

// adjoint of the E half-step on plain cells:  lH_h = lH_h + curl^+(ce*lE)_h   (row R4)
template <int V>
__device__ __forceinline__ void lean_adj_e_body(const Dev& d, const int i, const int j, const int k0) {
  const idx_t sx = d.sx, sy = d.sy;
  const idx_t q = ((idx_t)i * d.n[1] + j) * d.n[2] + k0;
  const VF<V> ce = ldv_ce<V>(d, d.ce + q), ce_xp = ldv_ce<V>(d, d.ce + q + sx), ce_yp = ldv_ce<V>(d, d.ce + q + sy);
  const float ce_zp = d.ce[q + V];
  VF<V> gx = ldv<V>(d.lE[0] + q), gy = ldv<V>(d.lE[1] + q), gz = ldv<V>(d.lE[2] + q);
  VF<V> gy_xp = ldv<V>(d.lE[1] + q + sx), gz_xp = ldv<V>(d.lE[2] + q + sx);
  VF<V> gx_yp = ldv<V>(d.lE[0] + q + sy), gz_yp = ldv<V>(d.lE[2] + q + sy);
  const float gx_zp = ce_zp * d.lE[0][q + V], gy_zp = ce_zp * d.lE[1][q + V];
  VF<V> lhx = ldv<V>(d.lH[0] + q), lhy = ldv<V>(d.lH[1] + q), lhz = ldv<V>(d.lH[2] + q);
#pragma unroll
  for (int v = 0; v < V; ++v) {
    gx.v[v] = ce.v[v] * gx.v[v];
    gy.v[v] = ce.v[v] * gy.v[v];
    gz.v[v] = ce.v[v] * gz.v[v];
    gy_xp.v[v] = ce_xp.v[v] * gy_xp.v[v];
    gz_xp.v[v] = ce_xp.v[v] * gz_xp.v[v];
    gx_yp.v[v] = ce_yp.v[v] * gx_yp.v[v];
    gz_yp.v[v] = ce_yp.v[v] * gz_yp.v[v];
  }
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float gx_zq = v == V - 1 ? gx_zp : gx.v[v < V - 1 ? v + 1 : v];
    const float gy_zq = v == V - 1 ? gy_zp : gy.v[v < V - 1 ? v + 1 : v];
    lhx.v[v] = lhx.v[v] + ((gz_yp.v[v] - gz.v[v]) - (gy_zq - gy.v[v]));
    lhy.v[v] = lhy.v[v] + ((gx_zq - gx.v[v]) - (gz_xp.v[v] - gz.v[v]));
    lhz.v[v] = lhz.v[v] + ((gy_xp.v[v] - gy.v[v]) - (gx_yp.v[v] - gx.v[v]));
  }
  stv<V>(d.lH[0] + q, lhx);
  stv<V>(d.lH[1] + q, lhy);
  stv<V>(d.lH[2] + q, lhz);
}

// the lean kernels proper (scalar path V = 1, and the per-kernel timings of fdtd_profile_kernel)
template <int V, bool ADJ>
__global__ void __launch_bounds__(32 * TY) k_lean_curlm(const __grid_constant__ Dev d, const __grid_constant__ Region r) {
  int i, j, k0;
  if (!lean_decode<V>(r, i, j, k0)) return;
  lean_curlm_body<V, ADJ>(d, i, j, k0);
}
template <int V>
__global__ void __launch_bounds__(32 * TY) k_lean_h(const __grid_constant__ Dev d, const __grid_constant__ Region r) {
  int i, j, k0;
  if (!lean_decode<V, SWEEP_FLIP>(r, i, j, k0)) return;
  lean_h_body<V>(d, i, j, k0);
}
template <int V>
__global__ void __launch_bounds__(32 * TY) k_lean_adj_e(const __grid_constant__ Dev d, const __grid_constant__ Region r) {
  int i, j, k0;
  if (!lean_decode<V, SWEEP_FLIP>(r, i, j, k0)) return;
  lean_adj_e_body<V>(d, i, j, k0);
}

// ---------------------------------------------------------------------------------------------------------
// ROW kernels (vector path): the lean cells and the z-slab cells of the same rows in ONE launch, so that every row of the
// lean x-y range is streamed whole and DRAM pages are used in full while they are open.  A lean region that covers 256 of a
// row's 512 bytes, next to a z-slab kernel that fetches the two 128-byte ends at a 512-byte stride somewhere else in the grid
// (C3), ran at 0.70-0.79 of the measured copy bandwidth; with whole rows the lean half-steps alone measured 0.94-1.0 (round 2,
// FDTD_DEBUG_FULLROW timing experiment: C3 forward E 76.3 -> 60.3 us, adjoint of E 82.6 -> 61.3 us; C4 forward E 927 -> 827 us).
// Grid: x = blocks of one SUPER-TILE of ROW_RS rows: first its lean blocks (row tile of TY rows x z tile of 128 cells, exactly
// the lean kernels' blocks), then `ns` SLAB blocks that pack the z-slab groups of those ROW_RS rows densely into their threads
// (item -> row, group) and run the class-Z general body on them (z CPML terms, low z wall, high z ghost); y = super-tile;
// z = plane.  Blocks are dispatched x-fastest, so the slab cells of a row are in flight together with its lean cells, and no
// lean block waits for the (3x longer) slab body of a neighbour warp.
// WHICH: 0 forward E, 1 forward H, 2 adjoint of H, 3 adjoint of E.  Same bodies as the split kernels: bit-identical results.
// ---------------------------------------------------------------------------------------------------------
// Resident blocks per SM the row kernels are compiled for (128 threads each): 6 (<= 85 registers, no spills) for the E-type and
// adjoint kernels, 8 (64 registers, a few spilled words in the slab blocks only) for the forward H kernel.  Measured on B200,
// group time in us, bounds 5 / 6 / 7 / 8: C4 forward E 834 / 834 / 849 / 872, forward H 847 / 847 / 815 / 799, adjoint of H
// 815 / 790 / 810 / 824, adjoint of E 918 / 862 / 912 / 890; C3 forward E 64.6 / 64.9 / 67.0 / 71.2, adjoint of E 77.1 / 71.4 / 73.2 / 72.9.
#ifndef FDTD_ROW_MINB
#define FDTD_ROW_MINB(WHICH) ((WHICH) == 1 ? 8 : 6)
#endif
constexpr int ROW_RS = 4 * TY;   // rows per super-tile
struct RowArgs {
  Region reg;     // lean region; z bounds are multiples of 4
  int nlo, nhi;   // z-slab groups (of 4 cells) per row below reg.lo[2] / from reg.hi[2] up to nz
  int ztiles;     // lean blocks along z
  int ns;         // slab blocks per super-tile
};
template <int WHICH>
__global__ void __launch_bounds__(32 * TY, FDTD_ROW_MINB(WHICH)) k_row(const __grid_constant__ Dev d, const __grid_constant__ RowArgs r, const int pb) {
  constexpr bool FLIP = SWEEP_FLIP && (WHICH == 1 || WHICH == 3);
  const int i = FLIP ? r.reg.hi[0] - 1 - (int)blockIdx.z : r.reg.lo[0] + (int)blockIdx.z;
  const int jsup = r.reg.lo[1] + (int)blockIdx.y * ROW_RS;
  const int nlean = (ROW_RS / TY) * r.ztiles;
  if ((int)blockIdx.x < nlean) {
    const int rt = (int)blockIdx.x / r.ztiles, zt = (int)blockIdx.x - rt * r.ztiles;
    const int k0 = r.reg.lo[2] + (zt * 32 + (int)threadIdx.x) * 4;
    const int j = jsup + rt * TY + (int)threadIdx.y;
    if (k0 >= r.reg.hi[2] || j >= r.reg.hi[1]) return;
    if (WHICH == 0) lean_curlm_body<4, false>(d, i, j, k0);
    else if (WHICH == 1) lean_h_body<4>(d, i, j, k0);
    else if (WHICH == 2) lean_curlm_body<4, true>(d, i, j, k0);
    else lean_adj_e_body<4>(d, i, j, k0);
    return;
  }
  const int ng = r.nlo + r.nhi;
  const int rows = min(ROW_RS, r.reg.hi[1] - jsup);
  const int it = ((int)blockIdx.x - nlean) * (32 * TY) + (int)threadIdx.y * 32 + (int)threadIdx.x;
  if (it >= rows * ng) return;
  // items are numbered group-major inside a row, rows consecutive: a warp covers whole rows' slab groups
  const int row = it / ng, g = it - row * ng;
  const int k0 = g < r.nlo ? 4 * g : r.reg.hi[2] + 4 * (g - r.nlo);
  const int j = jsup + row;
  if (WHICH == 0 || WHICH == 1) {
    FieldIO io;
#pragma unroll
    for (int c = 0; c < 3; ++c) { io.E[c] = d.E[c]; io.H[c] = d.H[c]; io.out[c] = WHICH == 0 ? d.E[c] : d.H[c]; }
    io_psi_inplace(io, d);
    if (WHICH == 0) gen_e_body<4, false, false>(d, i, j, k0, io);
    else gen_h_body<4, false, false>(d, i, j, k0, io);
  } else {
    AdjIO io;
#pragma unroll
    for (int c = 0; c < 3; ++c) { io.lEin[c] = d.lE[c]; io.lH[c] = d.lH[c]; io.lEout[c] = d.lE[c]; io.lHout[c] = d.lH[c]; }
    if (WHICH == 2) gen_adj_h_body<4, false, false>(d, i, j, k0, pb, io);
    else gen_adj_e_body<4, false, false>(d, i, j, k0, pb, io);
  }
}

}  // namespace fdtd
