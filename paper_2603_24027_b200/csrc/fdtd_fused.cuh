// fdtd_fused.cuh — fused marching kernels: two dependent half-steps in one pass over the plain cells, so that the
// intermediate field never makes a round trip through HBM (52 B per cell instead of 76).
//
//  k_fused_he<INV = false>  forward:  H^{m+1/2} = H^{m-1/2} - S curl^+(E^m)   then  E^{m+1} = E^m     + ce curl^-(H^{m+1/2})
//  k_fused_he<INV = true >  reverse:  H^{m-1/2} = H^{m+1/2} + S curl^+(E^m)   then  E^{m-1} = E^m     - ce curl^-(H^{m-1/2})
//
// A block owns a tile of TR rows x 31 z-groups (4 cells each) and marches along x through a segment of planes,
// keeping E of the next plane and the new H of the previous plane in registers.  The E update of a cell needs the NEW
// H of its three low-side neighbours: x from the previous march step, y from the warp below through shared memory,
// z from the lane below by shuffle.  Warp 0 and lane 0 of a block are halo workers: they recompute the new H of the
// row / z-group just below the tile and store nothing; the first march step of a segment does the same for the plane
// below the segment.  E of the row above (for the H update) also comes through shared memory, written one march step
// ahead.  Because neighbouring blocks recompute each other's cells from the OLD fields, input and output are different
// buffers (ping-pong).
//
// Forward: the region [lo, hi) starts one cell inside the interior (lo = P + 1), so every halo cell (index P) is a plain
// cell whose new H follows from the inputs alone: the kernel reads nothing that another kernel of the same step writes
// and runs beside the slab kernels.  Reverse (INV): the region is the inner interior and the halo cells are interface
// shell cells, whose H^{m-1/2} the inject kernel has already put into the OUTPUT buffer; they are read from there.  The
// sources of step m are ignored here and the (few) source cells redone afterwards by k_inv_e_sources.
// Arithmetic is that of the lean kernels (R3), so results are bit-identical to the two-kernel path.
#pragma once
#include "fdtd_dev.cuh"
#include "fdtd_store.cuh"

namespace fdtd {

constexpr int FUSED_TR = 8;              // rows stored per block (+1 halo warp)
constexpr int FUSED_ZG = 31;             // z-groups stored per warp (+1 halo lane)

struct FusedArgs {
  const float* Ein[3];
  const float* Hin[3];
  float* Eout[3];
  float* Hout[3];
  int lo[3], hi[3];      // region on which both half-steps are applied and stored
  int xseg;              // planes per block along x
};

template <bool INV>
__global__ void __launch_bounds__(32 * (FUSED_TR + 1), 3) k_fused_he(const __grid_constant__ Dev d, const __grid_constant__ FusedArgs a) {
  // [buffer][warp][component][lane]: a warp's 128-bit accesses are contiguous (lane-major, 16 bytes apart), hence free of bank
  // conflicts; with [lane][component] (32 bytes apart) ncu counted 8-way conflicts on every shared load and store
  __shared__ float4 shH[2][FUSED_TR + 1][2][32];   // new Hx, Hz of the current plane, double-buffered over the march
  __shared__ float4 shE[2][FUSED_TR + 1][2][32];   // Ex, Ez of the NEXT plane (read one march step later by the row below)
  const int lane = threadIdx.x, w = threadIdx.y;
  const int ny = d.n[1], nz = d.n[2];
  const int zbase = (a.lo[2] / 4) * 4;            // first stored group of tile 0
  const int k0raw = zbase + ((int)blockIdx.x * FUSED_ZG + lane - 1) * 4;
  const int jraw = a.lo[1] + (int)blockIdx.y * FUSED_TR + w - 1;
  const int xs = a.lo[0] + (int)blockIdx.z * a.xseg, xe = min(xs + a.xseg, a.hi[0]);
  // address clamps keep every load in bounds for the workers that overshoot the region; their results are never stored
  const int zlast = ((a.hi[2] - 1) / 4) * 4;
  const int k0 = min(k0raw, zlast), j = min(jraw, a.hi[1] - 1);
  const bool own_row = w >= 1 && jraw < a.hi[1];
  const bool own_grp = lane >= 1 && k0raw <= zlast;
  const bool own = own_row && own_grp;
  bool zv[4];                                     // element inside the region along z
#pragma unroll
  for (int v = 0; v < 4; ++v) zv[v] = k0 + v >= a.lo[2] && k0 + v < a.hi[2];
  const bool zfull = zv[0] && zv[1] && zv[2] && zv[3];
  const bool yp_smem = w < FUSED_TR && jraw + 1 < a.hi[1];   // the warp above holds row j + 1 (not a clamped copy)
  const idx_t sx = d.sx, sy = d.sy;
  const float cH = INV ? d.S : -d.S;
  idx_t q = ((idx_t)(xs - 1) * ny + j) * nz + k0; // the march starts one plane below the segment (priming)

  VF<4> ex = ldv<4>(a.Ein[0] + q), ey = ldv<4>(a.Ein[1] + q), ez = ldv<4>(a.Ein[2] + q);
  VF<4> hy_xm = zerov<4>(), hz_xm = zerov<4>();
  int buf = 0;
  for (int i = xs - 1; i < xe; ++i, q += sx, buf ^= 1) {
    // ---- loads: E of the next plane (kept for the next march step), H of this plane, y+1 / z+1 neighbours of E ----
    const VF<4> exn = ldv<4>(a.Ein[0] + q + sx), eyn = ldv<4>(a.Ein[1] + q + sx), ezn = ldv<4>(a.Ein[2] + q + sx);
    VF<4> hx = ldv<4>(a.Hin[0] + q), hy = ldv<4>(a.Hin[1] + q), hz = ldv<4>(a.Hin[2] + q);
    VF<4> ex_yp, ez_yp;
    if (yp_smem && i >= xs) {
      const float4 t0 = shE[buf][w + 1][0][lane], t1 = shE[buf][w + 1][1][lane];
      ex_yp.v[0] = t0.x; ex_yp.v[1] = t0.y; ex_yp.v[2] = t0.z; ex_yp.v[3] = t0.w;
      ez_yp.v[0] = t1.x; ez_yp.v[1] = t1.y; ez_yp.v[2] = t1.z; ez_yp.v[3] = t1.w;
    } else {
      ex_yp = ldv<4>(a.Ein[0] + q + sy);
      ez_yp = ldv<4>(a.Ein[2] + q + sy);
    }
    float ex_zp = __shfl_down_sync(0xffffffffu, ex.v[0], 1), ey_zp = __shfl_down_sync(0xffffffffu, ey.v[0], 1);
    if (lane == 31 || k0raw >= zlast) {           // no lane above holds the next group
      ex_zp = a.Ein[0][q + 4];
      ey_zp = a.Ein[1][q + 4];
    }
    VF<4> ce;
    const bool store_plane = own && i >= xs;
    if (store_plane) ce = ldv<4>(d.ce + q);

    // ---- H half-step ----
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float ey_zq = v == 3 ? ey_zp : ey.v[v < 3 ? v + 1 : v];
      const float ex_zq = v == 3 ? ex_zp : ex.v[v < 3 ? v + 1 : v];
      hx.v[v] = fmaf(cH, (ez_yp.v[v] - ez.v[v]) - (ey_zq - ey.v[v]), hx.v[v]);
      hy.v[v] = fmaf(cH, (ex_zq - ex.v[v]) - (ezn.v[v] - ez.v[v]), hy.v[v]);
      hz.v[v] = fmaf(cH, (eyn.v[v] - ey.v[v]) - (ex_yp.v[v] - ex.v[v]), hz.v[v]);
    }
    if (INV) {
      // Shell cells next to the region take their new H from the output buffer (inject has put H^{m-1/2} there).  Only
      // what an E update inside the region reads is needed: Hx, Hz of the row below (d_y^-), Hy, Hz of the plane below
      // (d_x^-), Hx, Hy of the cell below in z (d_z^-).  The shell cell above the last group is read by nobody.
      if (j < a.lo[1]) {
        hx = ldv<4>(a.Hout[0] + q);
        hz = ldv<4>(a.Hout[2] + q);
      } else if (i < a.lo[0]) {
        hy = ldv<4>(a.Hout[1] + q);
        hz = ldv<4>(a.Hout[2] + q);
      } else if (!zv[0]) {
        hx.v[0] = a.Hout[0][q];
        hy.v[0] = a.Hout[1][q];
      }
    }
    // ---- hand the new H to the row above (shared memory) and to the lane above (shuffle); E of the next plane to the
    //      row below for the next march step ----
    shH[buf][w][0][lane] = make_float4(hx.v[0], hx.v[1], hx.v[2], hx.v[3]);
    shH[buf][w][1][lane] = make_float4(hz.v[0], hz.v[1], hz.v[2], hz.v[3]);
    shE[buf ^ 1][w][0][lane] = make_float4(exn.v[0], exn.v[1], exn.v[2], exn.v[3]);
    shE[buf ^ 1][w][1][lane] = make_float4(ezn.v[0], ezn.v[1], ezn.v[2], ezn.v[3]);
    const float hx_z0 = __shfl_up_sync(0xffffffffu, hx.v[3], 1), hy_z0 = __shfl_up_sync(0xffffffffu, hy.v[3], 1);
    __syncthreads();
    if (store_plane) {
      const float4 t0 = shH[buf][w - 1][0][lane], t1 = shH[buf][w - 1][1][lane];
      const float hx_ym[4] = {t0.x, t0.y, t0.z, t0.w}, hz_ym[4] = {t1.x, t1.y, t1.z, t1.w};
      VF<4> eo;
      VF<4> e1, e2;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
        const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
        const float c = INV ? -ce.v[v] : ce.v[v];
        eo.v[v] = fmaf(c, (hz.v[v] - hz_ym[v]) - (hy.v[v] - hy_zm), ex.v[v]);
        e1.v[v] = fmaf(c, (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]), ey.v[v]);
        e2.v[v] = fmaf(c, (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym[v]), ez.v[v]);
      }
      if (zfull) {
        stv<4>(a.Hout[0] + q, hx); stv<4>(a.Hout[1] + q, hy); stv<4>(a.Hout[2] + q, hz);
        stv<4>(a.Eout[0] + q, eo); stv<4>(a.Eout[1] + q, e1); stv<4>(a.Eout[2] + q, e2);
      } else {
#pragma unroll
        for (int v = 0; v < 4; ++v)
          if (zv[v]) {
            a.Hout[0][q + v] = hx.v[v]; a.Hout[1][q + v] = hy.v[v]; a.Hout[2][q + v] = hz.v[v];
            a.Eout[0][q + v] = eo.v[v]; a.Eout[1][q + v] = e1.v[v]; a.Eout[2][q + v] = e2.v[v];
          }
      }
    }
    hy_xm = hy; hz_xm = hz;
    ex = exn; ey = eyn; ez = ezn;
  }
}

// ---------------------------------------------------------------------------------------------------------
// k_fused_fz — forward marching kernel over WHOLE rows: the plain cells of the lean x-y range and the z-slab cells at both ends of
// their rows, with the z terms of the CPML (psi_E, psi_H of the z axis), the z = 0 wall and the ghost above z = nz - 1 done in
// the edge lanes.  Why: beside k_fused_he the z-slab cells of those rows were slab-kernel boxes of 17 to 20 cells at each end of
// a 2 KB row (C4) — 1.5 GB of DRAM traffic per step for 0.83 GB of arrays, at 4.4 TB/s.  Here they ride on their rows.
//  * Every lane owns a group of 4 cells (no halo lane): a row of nz = 512 cells is exactly 4 tiles of 32 groups.  The new H just
//    below a tile, which the E update of the tile's first cell needs, is one cell: lane 0 recomputes H_x, H_y there from the old
//    fields with a handful of scalar loads (the host makes sure that cell is not a slab cell).
//  * Halo rows (warp 0) and the priming plane recompute the new H of cells that other blocks own, z-slab cells included, from the
//    OLD psi_H: psi_H of the z axis is therefore ping-ponged like E and H (pHz_in / pHz_out); psi_E is only ever touched by the
//    owner of its cell and stays in place.
//  * Arithmetic and its order are those of gen_h_body / gen_e_body for a class-Z box (R3): plain update, then the z term;
//    masked nodes (E_x, E_y at z = 0) become 0 and keep their psi.  Bit-identical to the two-kernel path (tests).
// ---------------------------------------------------------------------------------------------------------
constexpr int FUSED_ZSL = 8;    // slab groups per row the staging area holds: 2 * pml_width / 4 <= 8 (static shared memory <= 48 KB)
__device__ __forceinline__ void fused_cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
struct FusedZArgs {
  const float* Ein[3];
  const float* Hin[3];
  float* Eout[3];
  float* Hout[3];
  const float* pHz_in[2];   // old psi_H of the z axis: [0] the H_x term (psiH[0][1]), [1] the H_y term (psiH[1][0])
  float* pHz_out[2];
  float* pEz[2];            // psi_E of the z axis, in place: [0] the E_x term (psiE[0][1]), [1] the E_y term (psiE[1][0])
  int lo[2], hi[2];         // x and y range on which both half-steps are applied and stored; z is the whole row
  int xseg;
};

struct FusedZSmem {
  float4 H[2][FUSED_TR + 1][3][32];    // new H_x, H_y, H_z of the plane, double-buffered over the march
  float4 E[2][FUSED_TR + 1][3][32];    // E_x, E_y, E_z of the NEXT plane
  float4 P[2][4][FUSED_TR + 1][FUSED_ZSL];   // psi of the z axis, staged a plane ahead: psiHx, psiHy, psiEx, psiEy
  float C[6][FUSED_ZSL * 4];           // CPML coefficients of the z axis for the slab cells: bH cH kH bE cE kE
};
__global__ void __launch_bounds__(32 * (FUSED_TR + 1), 3) k_fused_fz(const __grid_constant__ Dev d, const __grid_constant__ FusedZArgs a) {
  // Shared memory doubles as the register file's overflow: whatever a thread carries from one plane to the next (E of the next
  // plane, its new H of the plane below) lives in the thread's OWN slots of the arrays through which the neighbouring rows read
  // it anyway, and is read back where it is needed.  With those 24 values in registers the kernel spilled 34 words per plane and
  // thread (72 registers at 3 blocks of 288 threads per SM).
  extern __shared__ __align__(16) unsigned char fz_smem_raw[];
  FusedZSmem& sm = *reinterpret_cast<FusedZSmem*>(fz_smem_raw);
  const int lane = threadIdx.x, w = threadIdx.y;
  const int ny = d.n[1], nz = d.n[2], P = d.P;
  const int g = (int)blockIdx.x * 32 + lane, ngroups = nz / 4;
  const bool own_grp = g < ngroups;
  const int k0 = min(g, ngroups - 1) * 4;
  const int jraw = a.lo[1] + (int)blockIdx.y * FUSED_TR + w - 1;
  const int xs = a.lo[0] + (int)blockIdx.z * a.xseg, xe = min(xs + a.xseg, a.hi[0]);
  const int j = min(jraw, a.hi[1] - 1);
  const bool own = w >= 1 && jraw < a.hi[1] && own_grp;
  const bool yp_smem = w < FUSED_TR && jraw + 1 < a.hi[1];
  const bool zs = P > 0 && in_slab(k0, nz, P);          // P % 4 == 0: a group lies in a z slab as a whole or not at all
  const bool wall = k0 == 0, top = k0 + 4 >= nz;
  const bool edge = lane == 0 && blockIdx.x > 0 && own_grp;   // the cell below this group belongs to the neighbouring tile
  const bool zp_load = (lane == 31 || g + 1 >= ngroups) && !top;   // no lane above holds the next group
  const idx_t sx = d.sx, sy = d.sy;
  const float mS = -d.S;
  idx_t q = ((idx_t)(xs - 1) * ny + j) * nz + k0;
  const int szl = zs ? slab_s(k0, nz, P) : 0;           // position of the group inside the compact psi rows of the z axis
  const int sl = szl / 4;                               // rank of the slab lane among the 2P/4 slab groups of a row (< FUSED_ZSL)
  if (zs && w == 0) {
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      sm.C[0][sl * 4 + v] = __ldg(d.tab[2][3] + k0 + v); sm.C[1][sl * 4 + v] = __ldg(d.tab[2][4] + k0 + v); sm.C[2][sl * 4 + v] = __ldg(d.tab[2][5] + k0 + v);
      sm.C[3][sl * 4 + v] = __ldg(d.tab[2][0] + k0 + v); sm.C[4][sl * 4 + v] = __ldg(d.tab[2][1] + k0 + v); sm.C[5][sl * 4 + v] = __ldg(d.tab[2][2] + k0 + v);
    }
  }
  // psi of the z axis for the slab lanes, requested one plane ahead with cp.async: no registers held while the lines travel
  auto stage_psi = [&](int plane, int st) {
    if (zs) {
      const idx_t qp = ((idx_t)plane * ny + j) * (2 * P) + szl;
      fused_cp_async16(&sm.P[st][0][w][sl], a.pHz_in[0] + qp);
      fused_cp_async16(&sm.P[st][1][w][sl], a.pHz_in[1] + qp);
      fused_cp_async16(&sm.P[st][2][w][sl], a.pEz[0] + qp);
      fused_cp_async16(&sm.P[st][3][w][sl], a.pEz[1] + qp);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  auto put = [](float4& dst, const VF<4>& x) { dst = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]); };
  auto get = [](const float4& t) { VF<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; };
  stage_psi(xs - 1, (xs - 1) & 1);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    put(sm.E[0][w][c][lane], ldv<4>(a.Ein[c] + q));
    sm.H[1][w][c][lane] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
  __syncthreads();                                      // sm.C
  int buf = 0;
  for (int i = xs - 1; i < xe; ++i, q += sx, buf ^= 1) {
    const idx_t qz = ((idx_t)i * ny + j) * (2 * P) + szl;
    stage_psi(min(i + 1, xe - 1), (i + 1) & 1);        // (the last step re-requests its own plane into the idle stage: harmless)
    // ---- loads: E of the next plane, H of this plane; E of this plane from the thread's own slots ----
    const VF<4> exn = ldv<4>(a.Ein[0] + q + sx), eyn = ldv<4>(a.Ein[1] + q + sx), ezn = ldv<4>(a.Ein[2] + q + sx);
    VF<4> hx = ldv<4>(a.Hin[0] + q), hy = ldv<4>(a.Hin[1] + q), hz = ldv<4>(a.Hin[2] + q);
    const VF<4> ex = get(sm.E[buf][w][0][lane]), ey = get(sm.E[buf][w][1][lane]), ez = get(sm.E[buf][w][2][lane]);
    VF<4> ex_yp, ez_yp;
    if (yp_smem && i >= xs) {
      ex_yp = get(sm.E[buf][w + 1][0][lane]);
      ez_yp = get(sm.E[buf][w + 1][2][lane]);
    } else {
      ex_yp = ldv<4>(a.Ein[0] + q + sy);
      ez_yp = ldv<4>(a.Ein[2] + q + sy);
    }
    float ex_zp = __shfl_down_sync(0xffffffffu, ex.v[0], 1), ey_zp = __shfl_down_sync(0xffffffffu, ey.v[0], 1);
    if (zp_load) { ex_zp = a.Ein[0][q + 4]; ey_zp = a.Ein[1][q + 4]; }
    if (top) { ex_zp = 0.0f; ey_zp = 0.0f; }          // ghost E[nz] = 0
    // edge lanes: the new H_x, H_y of the cell below the group (a plain cell), in the arithmetic of the plain H update, from a
    // handful of scalar loads out of lines the neighbouring tile streams anyway
    float hx_e = 0.0f, hy_e = 0.0f;
    if (edge) {
      const float exm = a.Ein[0][q - 1], eym = a.Ein[1][q - 1], ezm = a.Ein[2][q - 1];
      hx_e = fmaf(mS, (a.Ein[2][q - 1 + sy] - ezm) - (ey.v[0] - eym), a.Hin[0][q - 1]);
      hy_e = fmaf(mS, (ex.v[0] - exm) - (a.Ein[2][q - 1 + sx] - ezm), a.Hin[1][q - 1]);
    }
    const bool store_plane = own && i >= xs;
    VF<4> ce;
    if (store_plane) ce = ldv<4>(d.ce + q);            // requested here, consumed after the barrier

    // ---- H half-step (gen_h_body, class Z): plain update, then the z term of H_x (a2, sign -) and of H_y (a1, sign +) ----
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float ey_zq = v == 3 ? ey_zp : ey.v[v < 3 ? v + 1 : v];
      const float ex_zq = v == 3 ? ex_zp : ex.v[v < 3 ? v + 1 : v];
      hx.v[v] = fmaf(mS, (ez_yp.v[v] - ez.v[v]) - (ey_zq - ey.v[v]), hx.v[v]);
      hy.v[v] = fmaf(mS, (ex_zq - ex.v[v]) - (ezn.v[v] - ez.v[v]), hy.v[v]);
      hz.v[v] = fmaf(mS, (eyn.v[v] - ey.v[v]) - (ex_yp.v[v] - ex.v[v]), hz.v[v]);
    }
    asm volatile("cp.async.wait_group 1;" ::: "memory");   // the psi groups of THIS plane have landed (requested a step ago)
    if (zs) {
      VF<4> pa = get(sm.P[i & 1][0][w][sl]), pb = get(sm.P[i & 1][1][w][sl]);
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float ey_zq = v == 3 ? ey_zp : ey.v[v < 3 ? v + 1 : v];
        const float ex_zq = v == 3 ? ex_zp : ex.v[v < 3 ? v + 1 : v];
        const float dz_ey = ey_zq - ey.v[v], dz_ex = ex_zq - ex.v[v];
        const float bz = sm.C[0][sl * 4 + v], cz = sm.C[1][sl * 4 + v], kz = sm.C[2][sl * 4 + v];
        const float px = fmaf(bz, pa.v[v], cz * dz_ey);
        pa.v[v] = px;
        hx.v[v] = fmaf(-1.0f * mS, fmaf(kz, dz_ey, px), hx.v[v]);
        const float py = fmaf(bz, pb.v[v], cz * dz_ex);
        pb.v[v] = py;
        hy.v[v] = fmaf(1.0f * mS, fmaf(kz, dz_ex, py), hy.v[v]);
      }
      if (store_plane) { stv<4>(a.pHz_out[0] + qz, pa); stv<4>(a.pHz_out[1] + qz, pb); }
    }
    // the new H of the cell below the group: from the lane below, or recomputed by an edge lane
    float hx_z0 = __shfl_up_sync(0xffffffffu, hx.v[3], 1), hy_z0 = __shfl_up_sync(0xffffffffu, hy.v[3], 1);
    if (edge) { hx_z0 = hx_e; hy_z0 = hy_e; }
    if (wall) { hx_z0 = 0.0f; hy_z0 = 0.0f; }          // H[-1] ghost (only reaches the masked E_x, E_y at z = 0)
    put(sm.H[buf][w][0][lane], hx); put(sm.H[buf][w][1][lane], hy); put(sm.H[buf][w][2][lane], hz);
    put(sm.E[buf ^ 1][w][0][lane], exn); put(sm.E[buf ^ 1][w][1][lane], eyn); put(sm.E[buf ^ 1][w][2][lane], ezn);
    __syncthreads();
    if (store_plane) {
      stv<4>(a.Hout[0] + q, hx); stv<4>(a.Hout[1] + q, hy); stv<4>(a.Hout[2] + q, hz);
      // ---- E half-step (gen_e_body, class Z): plain update, then the z term of E_x (a2, sign -) and of E_y (a1, sign +).  E_x, E_y
      //      are finished and stored before E_z is computed ----
      VF<4> eo, e1;
      {
        const VF<4> hz_ym = get(sm.H[buf][w - 1][2][lane]), hz_xm = get(sm.H[buf ^ 1][w][2][lane]);
        const VF<4> ex2 = get(sm.E[buf][w][0][lane]), ey2 = get(sm.E[buf][w][1][lane]);
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
          const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
          eo.v[v] = fmaf(ce.v[v], (hz.v[v] - hz_ym.v[v]) - (hy.v[v] - hy_zm), ex2.v[v]);
          e1.v[v] = fmaf(ce.v[v], (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]), ey2.v[v]);
        }
      }
      if (zs) {
        VF<4> pa = get(sm.P[i & 1][2][w][sl]), pb = get(sm.P[i & 1][3][w][sl]);
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          if (k0 + v == 0) continue;                    // PEC-masked nodes keep their psi
          const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
          const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
          const float dz_hy = hy.v[v] - hy_zm, dz_hx = hx.v[v] - hx_zm;
          const float bz = sm.C[3][sl * 4 + v], cz = sm.C[4][sl * 4 + v], kz = sm.C[5][sl * 4 + v];
          const float px = fmaf(bz, pa.v[v], cz * dz_hy);
          pa.v[v] = px;
          eo.v[v] = fmaf(-1.0f * ce.v[v], fmaf(kz, dz_hy, px), eo.v[v]);
          const float py = fmaf(bz, pb.v[v], cz * dz_hx);
          pb.v[v] = py;
          e1.v[v] = fmaf(1.0f * ce.v[v], fmaf(kz, dz_hx, py), e1.v[v]);
        }
        stv<4>(a.pEz[0] + qz, pa); stv<4>(a.pEz[1] + qz, pb);
      }
      if (wall) { eo.v[0] = 0.0f; e1.v[0] = 0.0f; }     // PEC-masked nodes: E_x = E_y = 0 at z = 0
      stv<4>(a.Eout[0] + q, eo); stv<4>(a.Eout[1] + q, e1);
      {
        const VF<4> hx_ym = get(sm.H[buf][w - 1][0][lane]), hy_xm = get(sm.H[buf ^ 1][w][1][lane]);
        const VF<4> ez2 = get(sm.E[buf][w][2][lane]);
        VF<4> e2;
#pragma unroll
        for (int v = 0; v < 4; ++v) e2.v[v] = fmaf(ce.v[v], (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym.v[v]), ez2.v[v]);
        stv<4>(a.Eout[2] + q, e2);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// k_fused_iz — reverse twin of k_fused_fz: inverse-H + inverse-E of the inner interior in one marching pass, in the structure of
// the whole-row kernel (every lane owns a group of 4 z cells, shared memory as register overflow, edge lanes for the cell below a
// tile).  Groups cover z in [P, n - P): the two interface cells of a row are element 0 of its first group and element 3 of its
// last one, so every group is stored whole — H shell elements are written back as inject H has put them into the output buffer
// (they are the z neighbours of the first / last inner cell), E shell elements are placeholders that inject E overwrites in the
// next phase.  The row below the first y tile and the plane below the first x segment are interface cells too: their H comes from
// the output buffer.  Sources are ignored here and redone by k_inv_e_sources, as with k_fused_he<true>.
// ---------------------------------------------------------------------------------------------------------
struct FusedIArgs {
  const float* Ein[3];
  const float* Hin[3];
  float* Eout[3];
  float* Hout[3];
  int lo[2], hi[2];      // inner-interior x and y range
  int zlo, zhi;          // z range covered by whole groups: [P, n - P)
  int xseg;
};
struct FusedISmem {
  float4 H[2][FUSED_TR + 1][3][32];
  float4 E[2][FUSED_TR + 1][3][32];
};
__global__ void __launch_bounds__(32 * (FUSED_TR + 1), 3) k_fused_iz(const __grid_constant__ Dev d, const __grid_constant__ FusedIArgs a) {
  extern __shared__ __align__(16) unsigned char iz_smem_raw[];
  FusedISmem& sm = *reinterpret_cast<FusedISmem*>(iz_smem_raw);
  const int lane = threadIdx.x, w = threadIdx.y;
  const int ny = d.n[1], nz = d.n[2];
  const int g = (int)blockIdx.x * 32 + lane;
  const int k0 = min(max(4 * g, a.zlo), a.zhi - 4);     // clamped for the lanes outside [zlo, zhi): they own nothing
  const bool own_grp = 4 * g >= a.zlo && 4 * g < a.zhi;
  const int jraw = a.lo[1] + (int)blockIdx.y * FUSED_TR + w - 1;
  const int xs = a.lo[0] + (int)blockIdx.z * a.xseg, xe = min(xs + a.xseg, a.hi[0]);
  const int j = min(jraw, a.hi[1] - 1);
  const bool own = w >= 1 && jraw < a.hi[1] && own_grp;
  const bool yp_smem = w < FUSED_TR && jraw + 1 < a.hi[1];
  const bool shell_row = jraw < a.lo[1];                // the interface row below the first y tile
  const bool zs_lo = own_grp && k0 == a.zlo, zs_hi = own_grp && k0 + 4 == a.zhi;   // group holds an interface cell (element 0 / 3)
  const bool edge = own_grp && (lane == 0 || 4 * (g - 1) < a.zlo) && !zs_lo;        // no lane below holds the cell below the group
  const bool zp_load = lane == 31 || !own_grp || zs_hi;                             // no lane above holds the next group
  const idx_t sx = d.sx, sy = d.sy;
  const float S = d.S;
  idx_t q = ((idx_t)(xs - 1) * ny + j) * nz + k0;
  auto put = [](float4& dst, const VF<4>& x) { dst = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]); };
  auto get = [](const float4& t) { VF<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; };
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    put(sm.E[0][w][c][lane], ldv<4>(a.Ein[c] + q));
    sm.H[1][w][c][lane] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
  int buf = 0;
  for (int i = xs - 1; i < xe; ++i, q += sx, buf ^= 1) {
    const bool shell_plane = i < a.lo[0];               // the interface plane below the first x segment
    const bool from_out = shell_row || shell_plane;     // this worker's H is an interface value: taken from the output buffer
    const VF<4> exn = ldv<4>(a.Ein[0] + q + sx), eyn = ldv<4>(a.Ein[1] + q + sx), ezn = ldv<4>(a.Ein[2] + q + sx);
    VF<4> hx, hy, hz;
    if (from_out) { hx = ldv<4>(a.Hout[0] + q); hy = ldv<4>(a.Hout[1] + q); hz = ldv<4>(a.Hout[2] + q); }
    else { hx = ldv<4>(a.Hin[0] + q); hy = ldv<4>(a.Hin[1] + q); hz = ldv<4>(a.Hin[2] + q); }
    // interface cells at the row ends: H^{m-1/2} as inject H has written it (requested here, used after the H update)
    float sh[3] = {0.0f, 0.0f, 0.0f}, sh3[3] = {0.0f, 0.0f, 0.0f};
    if (zs_lo && !from_out) { sh[0] = a.Hout[0][q]; sh[1] = a.Hout[1][q]; sh[2] = a.Hout[2][q]; }
    if (zs_hi && !from_out) { sh3[0] = a.Hout[0][q + 3]; sh3[1] = a.Hout[1][q + 3]; sh3[2] = a.Hout[2][q + 3]; }
    const VF<4> ex = get(sm.E[buf][w][0][lane]), ey = get(sm.E[buf][w][1][lane]), ez = get(sm.E[buf][w][2][lane]);
    VF<4> ex_yp, ez_yp;
    if (yp_smem && i >= xs) {
      ex_yp = get(sm.E[buf][w + 1][0][lane]);
      ez_yp = get(sm.E[buf][w + 1][2][lane]);
    } else {
      ex_yp = ldv<4>(a.Ein[0] + q + sy);
      ez_yp = ldv<4>(a.Ein[2] + q + sy);
    }
    float ex_zp = __shfl_down_sync(0xffffffffu, ex.v[0], 1), ey_zp = __shfl_down_sync(0xffffffffu, ey.v[0], 1);
    if (zp_load) { ex_zp = a.Ein[0][q + 4]; ey_zp = a.Ein[1][q + 4]; }   // q + 4 <= n - P: inside the row
    float hx_e = 0.0f, hy_e = 0.0f;
    if (edge) {   // new H_x, H_y of the inner cell below the group, in the arithmetic of the inverse-H update
      const float exm = a.Ein[0][q - 1], eym = a.Ein[1][q - 1], ezm = a.Ein[2][q - 1];
      hx_e = fmaf(S, (a.Ein[2][q - 1 + sy] - ezm) - (ey.v[0] - eym), a.Hin[0][q - 1]);
      hy_e = fmaf(S, (ex.v[0] - exm) - (a.Ein[2][q - 1 + sx] - ezm), a.Hin[1][q - 1]);
    }
    const bool store_plane = own && i >= xs;
    VF<4> ce;
    if (store_plane) ce = ldv<4>(d.ce + q);
    // ---- inverse of the H half-step ----
    if (!from_out) {
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float ey_zq = v == 3 ? ey_zp : ey.v[v < 3 ? v + 1 : v];
        const float ex_zq = v == 3 ? ex_zp : ex.v[v < 3 ? v + 1 : v];
        hx.v[v] = fmaf(S, (ez_yp.v[v] - ez.v[v]) - (ey_zq - ey.v[v]), hx.v[v]);
        hy.v[v] = fmaf(S, (ex_zq - ex.v[v]) - (ezn.v[v] - ez.v[v]), hy.v[v]);
        hz.v[v] = fmaf(S, (eyn.v[v] - ey.v[v]) - (ex_yp.v[v] - ex.v[v]), hz.v[v]);
      }
      if (zs_lo) { hx.v[0] = sh[0]; hy.v[0] = sh[1]; hz.v[0] = sh[2]; }
      if (zs_hi) { hx.v[3] = sh3[0]; hy.v[3] = sh3[1]; hz.v[3] = sh3[2]; }
    }
    float hx_z0 = __shfl_up_sync(0xffffffffu, hx.v[3], 1), hy_z0 = __shfl_up_sync(0xffffffffu, hy.v[3], 1);
    if (edge) { hx_z0 = hx_e; hy_z0 = hy_e; }
    put(sm.H[buf][w][0][lane], hx); put(sm.H[buf][w][1][lane], hy); put(sm.H[buf][w][2][lane], hz);
    put(sm.E[buf ^ 1][w][0][lane], exn); put(sm.E[buf ^ 1][w][1][lane], eyn); put(sm.E[buf ^ 1][w][2][lane], ezn);
    __syncthreads();
    if (store_plane) {
      stv<4>(a.Hout[0] + q, hx); stv<4>(a.Hout[1] + q, hy); stv<4>(a.Hout[2] + q, hz);
      // ---- inverse of the E half-step; the interface elements keep E^m as a placeholder (inject E overwrites them) ----
      const VF<4> hx_ym = get(sm.H[buf][w - 1][0][lane]), hz_ym = get(sm.H[buf][w - 1][2][lane]);
      const VF<4> hy_xm = get(sm.H[buf ^ 1][w][1][lane]), hz_xm = get(sm.H[buf ^ 1][w][2][lane]);
      const VF<4> ex2 = get(sm.E[buf][w][0][lane]), ey2 = get(sm.E[buf][w][1][lane]), ez2 = get(sm.E[buf][w][2][lane]);
      VF<4> eo, e1, e2;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
        const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
        eo.v[v] = fmaf(-ce.v[v], (hz.v[v] - hz_ym.v[v]) - (hy.v[v] - hy_zm), ex2.v[v]);
        e1.v[v] = fmaf(-ce.v[v], (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]), ey2.v[v]);
        e2.v[v] = fmaf(-ce.v[v], (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym.v[v]), ez2.v[v]);
      }
      if (zs_lo) { eo.v[0] = ex2.v[0]; e1.v[0] = ey2.v[0]; e2.v[0] = ez2.v[0]; }
      if (zs_hi) { eo.v[3] = ex2.v[3]; e1.v[3] = ey2.v[3]; e2.v[3] = ez2.v[3]; }
      stv<4>(a.Eout[0] + q, eo); stv<4>(a.Eout[1] + q, e1); stv<4>(a.Eout[2] + q, e2);
    }
  }
}

// Source cells of the reverse variant.  The canonical order (R9) subtracts the source of step m from E^m BEFORE the
// inverse-E update, while the marching kernel's inverse-H update needs the untouched E^m; so the marching kernel ignores
// the sources and this small kernel redoes the inverse-E update of the (few) source cells of the inner interior afterwards,
// from the same inputs in the canonical order:  E^{m-1} = fma(-ce, curl^-(H^{m-1/2}), E^m - src).  blockIdx.y = source; a
// cell covered by several sources is written by the lowest-numbered one, which subtracts all of them in index order.
struct InvFixArgs {
  const float* Eold[3];   // E^m (input buffer of the marching kernel)
  const float* Hnew[3];   // H^{m-1/2} (its output buffer)
  float* Eout[3];
  const SrcDev* src;
  const float* waves;
  int nsrc, m_base;
  const int* step_dev;
};
__global__ void k_inv_e_sources(const __grid_constant__ Dev d, const __grid_constant__ InvFixArgs a) {
  const SrcDev S = a.src[blockIdx.y];
  const int P = d.P, ey_ = S.hi[1] - S.lo[1], ez_ = S.hi[2] - S.lo[2];
  const long long cells = (long long)(S.hi[0] - S.lo[0]) * ey_ * ez_;
  const int m = a.m_base + (a.step_dev ? *a.step_dev : 0);
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < cells; t += (long long)gridDim.x * blockDim.x) {
    const int c[3] = {S.lo[0] + (int)(t / ((long long)ez_ * ey_)), S.lo[1] + (int)((t / ez_) % ey_), S.lo[2] + (int)(t % ez_)};
    bool inner = true;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) inner = inner && c[ax] >= P + 1 && c[ax] < d.n[ax] - P - 1;
    if (!inner) continue;                       // shell cells are overwritten by inject
    const idx_t q = ((idx_t)c[0] * d.n[1] + c[1]) * d.n[2] + c[2];
    float e[3] = {a.Eold[0][q], a.Eold[1][q], a.Eold[2][q]};
    bool touched[3] = {false, false, false};
    bool first = true;
    for (int u = 0; u < a.nsrc; ++u) {
      const SrcDev U = a.src[u];
      if (c[0] < U.lo[0] || c[0] >= U.hi[0] || c[1] < U.lo[1] || c[1] >= U.hi[1] || c[2] < U.lo[2] || c[2] >= U.hi[2]) continue;
      if (u < (int)blockIdx.y) { first = false; break; }
      const long long ti = ((long long)(c[0] - U.lo[0]) * (U.hi[1] - U.lo[1]) + (c[1] - U.lo[1])) * (U.hi[2] - U.lo[2]) + (c[2] - U.lo[2]);
      const float v = (U.amp ? U.amp[ti] : 1.0f) * a.waves[U.wave_off + m - 1];
#pragma unroll
      for (int cc = 0; cc < 3; ++cc)
        if (U.comp == cc) { e[cc] += -1.0f * v; touched[cc] = true; }
    }
    if (!first) continue;
    const idx_t sx = d.sx, sy = d.sy;
    const float hx = a.Hnew[0][q], hy = a.Hnew[1][q], hz = a.Hnew[2][q];
    const float ce = d.ce[q];
    if (touched[0]) a.Eout[0][q] = fmaf(-ce, (hz - a.Hnew[2][q - sy]) - (hy - a.Hnew[1][q - 1]), e[0]);
    if (touched[1]) a.Eout[1][q] = fmaf(-ce, (hx - a.Hnew[0][q - 1]) - (hz - a.Hnew[2][q - sx]), e[1]);
    if (touched[2]) a.Eout[2][q] = fmaf(-ce, (hy - a.Hnew[1][q - sx]) - (hx - a.Hnew[0][q - sy]), e[2]);
  }
}

}  // namespace fdtd
