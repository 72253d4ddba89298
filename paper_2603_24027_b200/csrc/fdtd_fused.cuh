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
// Forward marching kernel over WHOLE rows (k_fused_fp below): the plain cells of the lean x-y range and the z-slab cells at both ends of
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

// ---------------------------------------------------------------------------------------------------------
// k_fused_fp — the whole-row forward marching kernel described above, with every global load of the march staged through shared
// memory by cp.async, one plane ahead (E two planes ahead): the loads of plane i+1 travel while plane i is computed, and they
// hold no registers while they do.  Its predecessor (k_fused_fz, round 2, removed) issued the loads of a plane at the top of its
// march step and consumed them a few instructions later, in front of a block-wide barrier; ncu: 5.4 TB/s of DRAM traffic against
// 7.0 for k_row, long-scoreboard and barrier stalls, 41 % occupancy, and no register left (72 at 3 blocks of 288 threads) to
// prefetch into — shared memory served as the register file's overflow there.  1186 -> 1009 us per launch on C4 (0.96 of the
// measured copy bandwidth in algorithmic bytes).
//  * Stages: E of plane p in stage p % 3 (plane i, i+1 in use, i+2 arriving), old H and psi of plane p in stage p % 2, new H of
//    plane p in stage p % 2.  Everything a thread or its neighbours read of plane i has landed before the barrier of step i-1.
//  * The halo accesses ride on the same pipeline: the row above the top warp is an extra row slot filled by the top warp; the
//    group below a tile (edge lanes) and the group above it (last lane) are extra float4 slots.
//  * 112 KB of shared memory per block, two blocks per SM (93 registers: nothing spills, E of the plane stays in registers across
//    the barrier).  ce is prefetched one plane ahead into registers.
// ---------------------------------------------------------------------------------------------------------
struct FusedPSmem {
  float4 E[3][FUSED_TR + 2][3][32];     // row slot w = the warp's row; slot TR + 1 = the row above the top warp's
  float4 Hin[2][FUSED_TR + 1][3][32];
  float4 Hn[2][FUSED_TR + 1][3][32];
  float4 Elo[3][FUSED_TR + 2][3];       // E of the group below the tile's first group (edge lanes)
  float4 Hlo[2][FUSED_TR + 1][2];       // old H_x, H_y of that group
  float4 Ehi[3][FUSED_TR + 1][2];       // E_x, E_y of the group above the warp's last group
  float4 P[2][4][FUSED_TR + 1][FUSED_ZSL];
  float C[6][FUSED_ZSL * 4];
};
__global__ void __launch_bounds__(32 * (FUSED_TR + 1), 2) k_fused_fp(const __grid_constant__ Dev d, const __grid_constant__ FusedZArgs a) {
  extern __shared__ __align__(16) unsigned char fp_smem_raw[];
  FusedPSmem& sm = *reinterpret_cast<FusedPSmem*>(fp_smem_raw);
  const int lane = threadIdx.x, w = threadIdx.y;
  const int ny = d.n[1], nz = d.n[2], P = d.P;
  const int g = (int)blockIdx.x * 32 + lane, ngroups = nz / 4;
  const bool own_grp = g < ngroups;
  const int k0 = min(g, ngroups - 1) * 4;
  const int jraw = a.lo[1] + (int)blockIdx.y * FUSED_TR + w - 1;
  const int xs = a.lo[0] + (int)blockIdx.z * a.xseg, xe = min(xs + a.xseg, a.hi[0]);
  // rows beyond the region clamp to the first row above it (inside the grid; they are loaded for their neighbour below, never stored)
  const int j = min(jraw, a.hi[1]), j2 = min(jraw + 1, a.hi[1]);
  const bool own = w >= 1 && jraw < a.hi[1] && own_grp;
  const bool zs = P > 0 && in_slab(k0, nz, P);
  const bool wall = k0 == 0, top = k0 + 4 >= nz;
  const bool edge = lane == 0 && blockIdx.x > 0 && own_grp;
  const bool zp_lane = (lane == 31 || g + 1 >= ngroups) && !top;
  const bool topw = w == FUSED_TR;
  const idx_t sx = d.sx;
  const float mS = -d.S;
  const int szl = zs ? slab_s(k0, nz, P) : 0;
  const int sl = szl / 4;
  const idx_t rowoff = (idx_t)j * nz + k0, rowoff2 = (idx_t)j2 * nz + k0;
  if (zs && w == 0) {
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      sm.C[0][sl * 4 + v] = __ldg(d.tab[2][3] + k0 + v); sm.C[1][sl * 4 + v] = __ldg(d.tab[2][4] + k0 + v); sm.C[2][sl * 4 + v] = __ldg(d.tab[2][5] + k0 + v);
      sm.C[3][sl * 4 + v] = __ldg(d.tab[2][0] + k0 + v); sm.C[4][sl * 4 + v] = __ldg(d.tab[2][1] + k0 + v); sm.C[5][sl * 4 + v] = __ldg(d.tab[2][2] + k0 + v);
    }
  }
  auto issueE = [&](int p) {            // E of plane p
    const int st = p % 3;
    const idx_t q = (idx_t)p * sx + rowoff;
#pragma unroll
    for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.E[st][w][c][lane], a.Ein[c] + q);
    if (topw) {
      const idx_t q2 = (idx_t)p * sx + rowoff2;
#pragma unroll
      for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.E[st][FUSED_TR + 1][c][lane], a.Ein[c] + q2);
      if (edge) fused_cp_async16(&sm.Elo[st][FUSED_TR + 1][2], a.Ein[2] + q2 - 4);
    }
    if (edge) {
#pragma unroll
      for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.Elo[st][w][c], a.Ein[c] + q - 4);
    }
    if (zp_lane) {
      fused_cp_async16(&sm.Ehi[st][w][0], a.Ein[0] + q + 4);
      fused_cp_async16(&sm.Ehi[st][w][1], a.Ein[1] + q + 4);
    }
  };
  auto issueH = [&](int p) {            // old H and psi of plane p
    const int st = p & 1;
    const idx_t q = (idx_t)p * sx + rowoff;
#pragma unroll
    for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.Hin[st][w][c][lane], a.Hin[c] + q);
    if (edge) {
      fused_cp_async16(&sm.Hlo[st][w][0], a.Hin[0] + q - 4);
      fused_cp_async16(&sm.Hlo[st][w][1], a.Hin[1] + q - 4);
    }
    if (zs) {
      const idx_t qp = ((idx_t)p * ny + j) * (2 * P) + szl;
      fused_cp_async16(&sm.P[st][0][w][sl], a.pHz_in[0] + qp);
      fused_cp_async16(&sm.P[st][1][w][sl], a.pHz_in[1] + qp);
      fused_cp_async16(&sm.P[st][2][w][sl], a.pEz[0] + qp);
      fused_cp_async16(&sm.P[st][3][w][sl], a.pEz[1] + qp);
    }
  };
  auto put = [](float4& dst, const VF<4>& x) { dst = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]); };
  auto get = [](const float4& t) { VF<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; };
  issueE(xs - 1);
  issueE(xs);
  issueH(xs - 1);
  asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll
  for (int c = 0; c < 3; ++c) sm.Hn[xs & 1][w][c][lane] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);   // "new H of plane xs - 2": never used in a stored value
  VF<4> ce_n = zerov<4>();
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();                                      // the priming planes and sm.C are visible to every warp
  for (int i = xs - 1; i < xe; ++i) {
    const idx_t q = (idx_t)i * sx + rowoff;
    const idx_t qz = ((idx_t)i * ny + j) * (2 * P) + szl;
    if (i + 2 <= xe) issueE(i + 2);
    if (i + 1 < xe) issueH(i + 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const VF<4> ce = ce_n;
    if (own && i + 1 < xe) ce_n = ldv<4>(d.ce + q + sx);    // ce of the next plane: a whole march step to arrive
    asm volatile("cp.async.wait_group 1;" ::: "memory");    // all but the newest group: E(i+1), old H(i), psi(i) have landed
    const int se = i % 3, sn = (i + 1) % 3, sh = i & 1;
    const VF<4> ex = get(sm.E[se][w][0][lane]), ey = get(sm.E[se][w][1][lane]), ez = get(sm.E[se][w][2][lane]);
    const VF<4> eyn = get(sm.E[sn][w][1][lane]), ezn = get(sm.E[sn][w][2][lane]);
    VF<4> hx = get(sm.Hin[sh][w][0][lane]), hy = get(sm.Hin[sh][w][1][lane]), hz = get(sm.Hin[sh][w][2][lane]);
    const VF<4> ex_yp = get(sm.E[se][w + 1][0][lane]), ez_yp = get(sm.E[se][w + 1][2][lane]);
    float ex_zp = __shfl_down_sync(0xffffffffu, ex.v[0], 1), ey_zp = __shfl_down_sync(0xffffffffu, ey.v[0], 1);
    if (zp_lane) { ex_zp = sm.Ehi[se][w][0].x; ey_zp = sm.Ehi[se][w][1].x; }
    if (top) { ex_zp = 0.0f; ey_zp = 0.0f; }          // ghost E[nz] = 0
    float hx_e = 0.0f, hy_e = 0.0f;
    if (edge) {   // new H_x, H_y of the (plain) cell below the group, in the arithmetic of the plain H update
      const float exm = sm.Elo[se][w][0].w, eym = sm.Elo[se][w][1].w, ezm = sm.Elo[se][w][2].w;
      hx_e = fmaf(mS, (sm.Elo[se][w + 1][2].w - ezm) - (ey.v[0] - eym), sm.Hlo[sh][w][0].w);
      hy_e = fmaf(mS, (ex.v[0] - exm) - (sm.Elo[sn][w][2].w - ezm), sm.Hlo[sh][w][1].w);
    }
    const bool store_plane = own && i >= xs;
    // ---- H half-step (gen_h_body, class Z): plain update, then the z term of H_x (a2, sign -) and of H_y (a1, sign +) ----
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float ey_zq = v == 3 ? ey_zp : ey.v[v < 3 ? v + 1 : v];
      const float ex_zq = v == 3 ? ex_zp : ex.v[v < 3 ? v + 1 : v];
      hx.v[v] = fmaf(mS, (ez_yp.v[v] - ez.v[v]) - (ey_zq - ey.v[v]), hx.v[v]);
      hy.v[v] = fmaf(mS, (ex_zq - ex.v[v]) - (ezn.v[v] - ez.v[v]), hy.v[v]);
      hz.v[v] = fmaf(mS, (eyn.v[v] - ey.v[v]) - (ex_yp.v[v] - ex.v[v]), hz.v[v]);
    }
    if (zs) {
      VF<4> pa = get(sm.P[sh][0][w][sl]), pb = get(sm.P[sh][1][w][sl]);
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
    float hx_z0 = __shfl_up_sync(0xffffffffu, hx.v[3], 1), hy_z0 = __shfl_up_sync(0xffffffffu, hy.v[3], 1);
    if (edge) { hx_z0 = hx_e; hy_z0 = hy_e; }
    if (wall) { hx_z0 = 0.0f; hy_z0 = 0.0f; }
    put(sm.Hn[sh][w][0][lane], hx); put(sm.Hn[sh][w][1][lane], hy); put(sm.Hn[sh][w][2][lane], hz);
    __syncthreads();
    if (store_plane) {
      stv<4>(a.Hout[0] + q, hx); stv<4>(a.Hout[1] + q, hy); stv<4>(a.Hout[2] + q, hz);
      // ---- E half-step (gen_e_body, class Z): plain update, then the z term of E_x (a2, sign -) and of E_y (a1, sign +) ----
      const VF<4> hx_ym = get(sm.Hn[sh][w - 1][0][lane]), hz_ym = get(sm.Hn[sh][w - 1][2][lane]);
      const VF<4> hy_xm = get(sm.Hn[sh ^ 1][w][1][lane]), hz_xm = get(sm.Hn[sh ^ 1][w][2][lane]);
      VF<4> eo, e1, e2;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
        const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
        eo.v[v] = fmaf(ce.v[v], (hz.v[v] - hz_ym.v[v]) - (hy.v[v] - hy_zm), ex.v[v]);
        e1.v[v] = fmaf(ce.v[v], (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]), ey.v[v]);
        e2.v[v] = fmaf(ce.v[v], (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym.v[v]), ez.v[v]);
      }
      if (zs) {
        VF<4> pa = get(sm.P[sh][2][w][sl]), pb = get(sm.P[sh][3][w][sl]);
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
      stv<4>(a.Eout[0] + q, eo); stv<4>(a.Eout[1] + q, e1); stv<4>(a.Eout[2] + q, e2);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// Reverse twin of the whole-row kernel (k_fused_ip below): inverse-H + inverse-E of the inner interior in one marching pass, in the structure of
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
// ---------------------------------------------------------------------------------------------------------
// k_fused_ip — the reverse twin described above, in the pipelined form of k_fused_fp: the loads of the march are staged through
// shared memory by cp.async, a plane ahead.  The interface H of the row below the first y tile and of the plane below the first x
// segment (put into the output buffer by inject H, earlier on the same stream) is staged from that buffer into the same slots; the
// interface elements at the two ends of a row are prefetched a plane ahead into registers.  Its predecessor with direct loads
// (k_fused_iz, removed) took 1202 us per launch on C4, this one 980 us (5.8 TB/s): the first fused reverse primal that beats the
// two inverse kernels on 512^3 (reverse run 3090 -> 2924 us per step).
// ---------------------------------------------------------------------------------------------------------
struct FusedQSmem {
  float4 E[3][FUSED_TR + 2][3][32];
  float4 Hin[2][FUSED_TR + 1][3][32];
  float4 Hn[2][FUSED_TR + 1][3][32];
  float4 Elo[3][FUSED_TR + 2][3];
  float4 Hlo[2][FUSED_TR + 1][2];
  float4 Ehi[3][FUSED_TR + 1][2];
};
__global__ void __launch_bounds__(32 * (FUSED_TR + 1), 2) k_fused_ip(const __grid_constant__ Dev d, const __grid_constant__ FusedIArgs a) {
  extern __shared__ __align__(16) unsigned char ip_smem_raw[];
  FusedQSmem& sm = *reinterpret_cast<FusedQSmem*>(ip_smem_raw);
  const int lane = threadIdx.x, w = threadIdx.y;
  const int nz = d.n[2];
  const int g = (int)blockIdx.x * 32 + lane;
  const int k0 = min(max(4 * g, a.zlo), a.zhi - 4);
  const bool own_grp = 4 * g >= a.zlo && 4 * g < a.zhi;
  const int jraw = a.lo[1] + (int)blockIdx.y * FUSED_TR + w - 1;
  const int xs = a.lo[0] + (int)blockIdx.z * a.xseg, xe = min(xs + a.xseg, a.hi[0]);
  const int j = min(jraw, a.hi[1]), j2 = min(jraw + 1, a.hi[1]);   // hi[1] = n - P - 1: the interface row above the region, in the grid
  const bool own = w >= 1 && jraw < a.hi[1] && own_grp;
  const bool shell_row = jraw < a.lo[1];
  const bool zs_lo = own_grp && k0 == a.zlo, zs_hi = own_grp && k0 + 4 == a.zhi;
  const bool edge = own_grp && lane == 0 && !zs_lo;
  // the one lane per warp whose z+1 neighbour lies in the next tile.  (The row's last group, zs_hi, needs it for its interface
  // element only, which is replaced; lanes outside [zlo, zhi) own nothing.  They must NOT share the staging slot: the slot has one
  // writer per warp.)
  const bool zp_lane = lane == 31 && own_grp && !zs_hi;
  const bool topw = w == FUSED_TR;
  const idx_t sx = d.sx;
  const float S = d.S;
  const idx_t rowoff = (idx_t)j * nz + k0, rowoff2 = (idx_t)j2 * nz + k0;
  auto issueE = [&](int p) {
    const int st = p % 3;
    const idx_t q = (idx_t)p * sx + rowoff;
#pragma unroll
    for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.E[st][w][c][lane], a.Ein[c] + q);
    if (topw) {
      const idx_t q2 = (idx_t)p * sx + rowoff2;
#pragma unroll
      for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.E[st][FUSED_TR + 1][c][lane], a.Ein[c] + q2);
      if (edge) fused_cp_async16(&sm.Elo[st][FUSED_TR + 1][2], a.Ein[2] + q2 - 4);
    }
    if (edge) {
#pragma unroll
      for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.Elo[st][w][c], a.Ein[c] + q - 4);
    }
    if (zp_lane) {
      fused_cp_async16(&sm.Ehi[st][w][0], a.Ein[0] + q + 4);
      fused_cp_async16(&sm.Ehi[st][w][1], a.Ein[1] + q + 4);
    }
  };
  auto issueH = [&](int p) {            // H^{m+1/2} of plane p; for interface rows / planes H^{m-1/2} as inject H has written it
    const int st = p & 1;
    const idx_t q = (idx_t)p * sx + rowoff;
    const bool from_out = shell_row || p < a.lo[0];
#pragma unroll
    for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.Hin[st][w][c][lane], (from_out ? a.Hout[c] : a.Hin[c]) + q);
    if (edge) {   // the cell below an edge lane's group is an inner cell of this row: its H^{m+1/2} (recomputed below)
      fused_cp_async16(&sm.Hlo[st][w][0], a.Hin[0] + q - 4);
      fused_cp_async16(&sm.Hlo[st][w][1], a.Hin[1] + q - 4);
    }
  };
  auto put = [](float4& dst, const VF<4>& x) { dst = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]); };
  auto get = [](const float4& t) { VF<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; };
  issueE(xs - 1);
  issueE(xs);
  issueH(xs - 1);
  asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll
  for (int c = 0; c < 3; ++c) sm.Hn[xs & 1][w][c][lane] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  VF<4> ce_n = zerov<4>();
  float shn[3] = {0.0f, 0.0f, 0.0f};                    // interface H of the NEXT plane at this row's end (zs_lo: element 0, zs_hi: element 3)
  const int vi = zs_lo ? 0 : 3;
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  for (int i = xs - 1; i < xe; ++i) {
    const idx_t q = (idx_t)i * sx + rowoff;
    const bool from_out = shell_row || i < a.lo[0];
    if (i + 2 <= xe) issueE(i + 2);
    if (i + 1 < xe) issueH(i + 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const VF<4> ce = ce_n;
    const float sh[3] = {shn[0], shn[1], shn[2]};
    if (own && i + 1 < xe) {
      ce_n = ldv<4>(d.ce + q + sx);
      if ((zs_lo || zs_hi) && !shell_row) {
#pragma unroll
        for (int c = 0; c < 3; ++c) shn[c] = a.Hout[c][q + sx + vi];
      }
    }
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    const int se = i % 3, sn = (i + 1) % 3, sh_ = i & 1;
    const VF<4> ex = get(sm.E[se][w][0][lane]), ey = get(sm.E[se][w][1][lane]), ez = get(sm.E[se][w][2][lane]);
    const VF<4> eyn = get(sm.E[sn][w][1][lane]), ezn = get(sm.E[sn][w][2][lane]);
    VF<4> hx = get(sm.Hin[sh_][w][0][lane]), hy = get(sm.Hin[sh_][w][1][lane]), hz = get(sm.Hin[sh_][w][2][lane]);
    const VF<4> ex_yp = get(sm.E[se][w + 1][0][lane]), ez_yp = get(sm.E[se][w + 1][2][lane]);
    float ex_zp = __shfl_down_sync(0xffffffffu, ex.v[0], 1), ey_zp = __shfl_down_sync(0xffffffffu, ey.v[0], 1);
    if (zp_lane) { ex_zp = sm.Ehi[se][w][0].x; ey_zp = sm.Ehi[se][w][1].x; }
    float hx_e = 0.0f, hy_e = 0.0f;
    if (edge) {
      const float exm = sm.Elo[se][w][0].w, eym = sm.Elo[se][w][1].w, ezm = sm.Elo[se][w][2].w;
      hx_e = fmaf(S, (sm.Elo[se][w + 1][2].w - ezm) - (ey.v[0] - eym), sm.Hlo[sh_][w][0].w);
      hy_e = fmaf(S, (ex.v[0] - exm) - (sm.Elo[sn][w][2].w - ezm), sm.Hlo[sh_][w][1].w);
    }
    const bool store_plane = own && i >= xs;
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
      if (store_plane && (zs_lo || zs_hi)) {
#pragma unroll
        for (int v = 0; v < 4; ++v)
          if (v == vi) { hx.v[v] = sh[0]; hy.v[v] = sh[1]; hz.v[v] = sh[2]; }
      }
    }
    float hx_z0 = __shfl_up_sync(0xffffffffu, hx.v[3], 1), hy_z0 = __shfl_up_sync(0xffffffffu, hy.v[3], 1);
    if (edge) { hx_z0 = hx_e; hy_z0 = hy_e; }
    put(sm.Hn[sh_][w][0][lane], hx); put(sm.Hn[sh_][w][1][lane], hy); put(sm.Hn[sh_][w][2][lane], hz);
    __syncthreads();
    if (store_plane) {
      stv<4>(a.Hout[0] + q, hx); stv<4>(a.Hout[1] + q, hy); stv<4>(a.Hout[2] + q, hz);
      const VF<4> hx_ym = get(sm.Hn[sh_][w - 1][0][lane]), hz_ym = get(sm.Hn[sh_][w - 1][2][lane]);
      const VF<4> hy_xm = get(sm.Hn[sh_ ^ 1][w][1][lane]), hz_xm = get(sm.Hn[sh_ ^ 1][w][2][lane]);
      VF<4> eo, e1, e2;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float hy_zm = v == 0 ? hy_z0 : hy.v[v > 0 ? v - 1 : 0];
        const float hx_zm = v == 0 ? hx_z0 : hx.v[v > 0 ? v - 1 : 0];
        eo.v[v] = fmaf(-ce.v[v], (hz.v[v] - hz_ym.v[v]) - (hy.v[v] - hy_zm), ex.v[v]);
        e1.v[v] = fmaf(-ce.v[v], (hx.v[v] - hx_zm) - (hz.v[v] - hz_xm.v[v]), ey.v[v]);
        e2.v[v] = fmaf(-ce.v[v], (hy.v[v] - hy_xm.v[v]) - (hx.v[v] - hx_ym.v[v]), ez.v[v]);
      }
      if (zs_lo) { eo.v[0] = ex.v[0]; e1.v[0] = ey.v[0]; e2.v[0] = ez.v[0]; }   // interface elements: placeholders, inject E overwrites them
      if (zs_hi) { eo.v[3] = ex.v[3]; e1.v[3] = ey.v[3]; e2.v[3] = ez.v[3]; }
      stv<4>(a.Eout[0] + q, eo); stv<4>(a.Eout[1] + q, e1); stv<4>(a.Eout[2] + q, e2);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// k_fused_ap — adjoint marching kernel: the adjoint of the H half-step (A: lambda_E += -S curl^-(lambda_H), transposed psi_H terms)
// and the adjoint of the E half-step (B: lambda_H += curl^+(ce lambda_E), transposed psi_E terms) of one reverse step in ONE pass
// over the rows of [P+1, n-P-1)^2, whole rows in z: 52 B per cell instead of 36 + 40.  The mirror image of k_fused_fp: A reads the
// LOW-side neighbours of the old lambda_H, B the HIGH-side neighbours of the new lambda_E, so the march runs DOWN in x, the halo
// workers sit on the high side (the warp above the tile, the plane above the segment: they compute A from the old values and store
// nothing — hence ping-ponged lambda_E / lambda_H), and the cell above a tile's last group is recomputed by the last lane.
// Loads are staged through shared memory by cp.async a plane ahead, as in k_fused_fp.  The transposed z CPML runs in the lanes of
// the z slabs in the arithmetic of gen_adj_h_body / gen_adj_e_body for a class-Z box; the W terms of the neighbouring cell travel by
// warp shuffle (same expression, same inputs: same bits).  lambda_psi is ping-ponged by the step parity already (pb -> pb ^ 1).
// ---------------------------------------------------------------------------------------------------------
struct FusedAArgs {
  const float* lEin[3];
  const float* lHin[3];
  float* lEout[3];
  float* lHout[3];
  const float* pH_in[2];    // old lambda_psi_H of the z axis: [0] the H_x term (lpsiH[pb][0][1]), [1] the H_y term (lpsiH[pb][1][0])
  float* pH_out[2];
  const float* pE_in[2];    // old lambda_psi_E of the z axis: [0] the E_x term (lpsiE[pb][0][1]), [1] the E_y term (lpsiE[pb][1][0])
  float* pE_out[2];
  int lo[2], hi[2];
  int xseg;
};
struct FusedASmem {
  float4 H[3][FUSED_TR + 2][3][32];     // old lambda_H of plane p in stage p % 3; row slot r = row (first row of the tile) - 1 + r
  float4 E[2][FUSED_TR + 1][3][32];     // old lambda_E of plane p in stage p % 2; row slot w
  float4 G[2][FUSED_TR + 1][3][32];     // new ce * lambda_E of plane p in stage p % 2
  float4 P[2][4][FUSED_TR + 1][FUSED_ZSL];   // lambda_psi of the z axis: psiH x-term, psiH y-term, psiE x-term, psiE y-term
  float4 Hlo[3][FUSED_TR + 1][2];       // lambda_H_x, lambda_H_y of the group below the tile's first group (lane 0)
  float4 Hhi[3][FUSED_TR + 2][3];       // lambda_H of the group above the warp's last group (last lane), rows as H
  float4 Ehi[2][FUSED_TR + 1][2];       // old lambda_E_x, lambda_E_y of that group
  float4 Chi[2][FUSED_TR + 1];          // ce of that group
  float C[6][FUSED_ZSL * 4];
};
__global__ void __launch_bounds__(32 * (FUSED_TR + 1), 2) k_fused_ap(const __grid_constant__ Dev d, const __grid_constant__ FusedAArgs a) {
  extern __shared__ __align__(16) unsigned char ap_smem_raw[];
  FusedASmem& sm = *reinterpret_cast<FusedASmem*>(ap_smem_raw);
  const int lane = threadIdx.x, w = threadIdx.y;
  const int ny = d.n[1], nz = d.n[2], P = d.P;
  const int g = (int)blockIdx.x * 32 + lane, ngroups = nz / 4;
  const bool own_grp = g < ngroups;
  const int k0 = min(g, ngroups - 1) * 4;
  const int j0 = a.lo[1] + (int)blockIdx.y * FUSED_TR;          // first row of the tile
  const int jraw = j0 + w;
  const int xs = a.lo[0] + (int)blockIdx.z * a.xseg, xe = min(xs + a.xseg, a.hi[0]);
  const int j = min(jraw, a.hi[1]);                              // rows above the region clamp to the first row above it
  const bool own = w < FUSED_TR && jraw < a.hi[1] && own_grp;
  const bool zs = P > 0 && in_slab(k0, nz, P);
  const bool za = zs || (k0 > 0 && P > 0 && in_slab(k0 - 1, nz, P));          // A needs W of the cell below
  const bool zb = zs || (k0 + 4 < nz && P > 0 && in_slab(k0 + 4, nz, P));      // B needs W of the cell above
  const bool wall = k0 == 0, top = k0 + 4 >= nz;
  const bool lo_lane = lane == 0 && blockIdx.x > 0 && own_grp;                 // the cell below the group belongs to the tile below
  const bool hi_lane = (lane == 31 || g + 1 >= ngroups) && !top && own_grp;    // no lane above holds the next group
  const idx_t sx = d.sx;
  const float S = d.S;
  const int szl = zs ? slab_s(k0, nz, P) : 0;
  const int sl = szl / 4;
  const idx_t rowoff = (idx_t)j * nz + k0, rowoff_m = (idx_t)(j0 - 1) * nz + k0;
  if (zs && w == 0) {
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      sm.C[0][sl * 4 + v] = __ldg(d.tab[2][3] + k0 + v); sm.C[1][sl * 4 + v] = __ldg(d.tab[2][4] + k0 + v); sm.C[2][sl * 4 + v] = __ldg(d.tab[2][5] + k0 + v);
      sm.C[3][sl * 4 + v] = __ldg(d.tab[2][0] + k0 + v); sm.C[4][sl * 4 + v] = __ldg(d.tab[2][1] + k0 + v); sm.C[5][sl * 4 + v] = __ldg(d.tab[2][2] + k0 + v);
    }
  }
  auto issueH = [&](int p) {            // old lambda_H of plane p (rows: own slot w + 1; warp 0 also slot 0 = the row below the tile)
    const int st = p % 3;
    const idx_t q = (idx_t)p * sx + rowoff;
#pragma unroll
    for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.H[st][w + 1][c][lane], a.lHin[c] + q);
    if (lo_lane) {
      fused_cp_async16(&sm.Hlo[st][w][0], a.lHin[0] + q - 4);
      fused_cp_async16(&sm.Hlo[st][w][1], a.lHin[1] + q - 4);
    }
    if (hi_lane) {
#pragma unroll
      for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.Hhi[st][w + 1][c], a.lHin[c] + q + 4);
    }
    if (w == 0) {
      const idx_t qm = (idx_t)p * sx + rowoff_m;
#pragma unroll
      for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.H[st][0][c][lane], a.lHin[c] + qm);
      if (hi_lane) fused_cp_async16(&sm.Hhi[st][0][2], a.lHin[2] + qm + 4);
    }
  };
  auto issueE = [&](int p) {            // old lambda_E, lambda_psi of plane p
    const int st = p & 1;
    const idx_t q = (idx_t)p * sx + rowoff;
#pragma unroll
    for (int c = 0; c < 3; ++c) fused_cp_async16(&sm.E[st][w][c][lane], a.lEin[c] + q);
    if (hi_lane) {
      fused_cp_async16(&sm.Ehi[st][w][0], a.lEin[0] + q + 4);
      fused_cp_async16(&sm.Ehi[st][w][1], a.lEin[1] + q + 4);
      fused_cp_async16(&sm.Chi[st][w], d.ce + q + 4);
    }
    if (zs) {
      const idx_t qp = ((idx_t)p * ny + j) * (2 * P) + szl;
      fused_cp_async16(&sm.P[st][0][w][sl], a.pH_in[0] + qp);
      fused_cp_async16(&sm.P[st][1][w][sl], a.pH_in[1] + qp);
      fused_cp_async16(&sm.P[st][2][w][sl], a.pE_in[0] + qp);
      fused_cp_async16(&sm.P[st][3][w][sl], a.pE_in[1] + qp);
    }
  };
  auto put = [](float4& dst, const VF<4>& x) { dst = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]); };
  auto get = [](const float4& t) { VF<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; };
  issueH(xe);
  issueH(xe - 1);
  issueE(xe);
  asm volatile("cp.async.commit_group;" ::: "memory");
  VF<4> ce_n = ldv<4>(d.ce + (idx_t)xe * sx + rowoff);   // ce of the priming plane
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  for (int i = xe; i >= xs; --i) {
    const idx_t q = (idx_t)i * sx + rowoff;
    const idx_t qz = ((idx_t)i * ny + j) * (2 * P) + szl;
    if (i - 2 >= xs - 1) issueH(i - 2);
    if (i - 1 >= xs) issueE(i - 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const VF<4> ce = ce_n;
    if (i - 1 >= xs) ce_n = ldv<4>(d.ce + q - sx);
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    const int s0 = i % 3, s1 = (i - 1) % 3, se = i & 1;
    const bool store_plane = own && i < xe;
    // ---- A: adjoint of the H half-step at plane i ----
    const VF<4> lhx = get(sm.H[s0][w + 1][0][lane]), lhy = get(sm.H[s0][w + 1][1][lane]), lhz = get(sm.H[s0][w + 1][2][lane]);
    const VF<4> lhy_xm = get(sm.H[s1][w + 1][1][lane]), lhz_xm = get(sm.H[s1][w + 1][2][lane]);
    const VF<4> lhx_ym = get(sm.H[s0][w][0][lane]), lhz_ym = get(sm.H[s0][w][2][lane]);
    VF<4> lex = get(sm.E[se][w][0][lane]), ley = get(sm.E[se][w][1][lane]), lez = get(sm.E[se][w][2][lane]);
    float lhx_z0 = __shfl_up_sync(0xffffffffu, lhx.v[3], 1), lhy_z0 = __shfl_up_sync(0xffffffffu, lhy.v[3], 1);
    if (lo_lane) { lhx_z0 = sm.Hlo[s0][w][0].w; lhy_z0 = sm.Hlo[s0][w][1].w; }
    if (wall) { lhx_z0 = 0.0f; lhy_z0 = 0.0f; }
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float lhy_zm = v == 0 ? lhy_z0 : lhy.v[v > 0 ? v - 1 : 0];
      const float lhx_zm = v == 0 ? lhx_z0 : lhx.v[v > 0 ? v - 1 : 0];
      lex.v[v] = fmaf(-S, (lhz.v[v] - lhz_ym.v[v]) - (lhy.v[v] - lhy_zm), lex.v[v]);
      ley.v[v] = fmaf(-S, (lhx.v[v] - lhx_zm) - (lhz.v[v] - lhz_xm.v[v]), ley.v[v]);
      lez.v[v] = fmaf(-S, (lhy.v[v] - lhy_xm.v[v]) - (lhx.v[v] - lhx_ym.v[v]), lez.v[v]);
    }
    {   // transposed psi_H terms of the z axis: (c=0,t=1: g = +S*lH_x -> lE_y) and (c=1,t=0: g = -S*lH_y -> lE_x)
      float w01[4] = {0.0f, 0.0f, 0.0f, 0.0f}, w10[4] = {0.0f, 0.0f, 0.0f, 0.0f};
      if (zs) {
        const VF<4> o01 = get(sm.P[se][0][w][sl]), o10 = get(sm.P[se][1][w][sl]);
        VF<4> n01, n10;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float bz = sm.C[0][sl * 4 + v], cz = sm.C[1][sl * 4 + v], kz = sm.C[2][sl * 4 + v];
          w01[v] = cpml_adjoint_term(S * lhx.v[v], o01.v[v], bz, cz, kz, n01.v[v]);
          w10[v] = cpml_adjoint_term(-S * lhy.v[v], o10.v[v], bz, cz, kz, n10.v[v]);
        }
        if (store_plane) { stv<4>(a.pH_out[0] + qz, n01); stv<4>(a.pH_out[1] + qz, n10); }
      }
      float w01_m = __shfl_up_sync(0xffffffffu, w01[3], 1), w10_m = __shfl_up_sync(0xffffffffu, w10[3], 1);
      if (lane == 0) { w01_m = 0.0f; w10_m = 0.0f; }   // the cell below a tile is a plain cell without a slab neighbour (host check)
      if (za) {
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float w01m = v == 0 ? w01_m : w01[v > 0 ? v - 1 : 0];
          const float w10m = v == 0 ? w10_m : w10[v > 0 ? v - 1 : 0];
          lex.v[v] -= (w10[v] - w10m);
          ley.v[v] -= (w01[v] - w01m);
        }
      }
    }
    if (wall) { lex.v[0] = 0.0f; ley.v[0] = 0.0f; }   // PEC-masked nodes (z = 0)
    if (store_plane) { stv<4>(a.lEout[0] + q, lex); stv<4>(a.lEout[1] + q, ley); stv<4>(a.lEout[2] + q, lez); }
    // ---- G = ce * lambda_E (new) at the cell; at the cell above the warp's last group by the last lane ----
    VF<4> gx, gy, gz;
#pragma unroll
    for (int v = 0; v < 4; ++v) { gx.v[v] = ce.v[v] * lex.v[v]; gy.v[v] = ce.v[v] * ley.v[v]; gz.v[v] = ce.v[v] * lez.v[v]; }
    float gx_zp = __shfl_down_sync(0xffffffffu, gx.v[0], 1), gy_zp = __shfl_down_sync(0xffffffffu, gy.v[0], 1);
    if (hi_lane) {   // A at (i, j, k0 + 4), a plain cell: new lambda_E_x, lambda_E_y there
      const float hxq = sm.Hhi[s0][w + 1][0].x, hyq = sm.Hhi[s0][w + 1][1].x, hzq = sm.Hhi[s0][w + 1][2].x;
      const float ex_q = fmaf(-S, (hzq - sm.Hhi[s0][w][2].x) - (hyq - lhy.v[3]), sm.Ehi[se][w][0].x);
      const float ey_q = fmaf(-S, (hxq - lhx.v[3]) - (hzq - sm.Hhi[s1][w + 1][2].x), sm.Ehi[se][w][1].x);
      const float ceq = sm.Chi[se][w].x;
      gx_zp = ceq * ex_q;
      gy_zp = ceq * ey_q;
    }
    if (top) { gx_zp = 0.0f; gy_zp = 0.0f; }
    // transposed psi_E terms of the z axis: (c=0,t=1: g = -G_x -> lH_y) and (c=1,t=0: g = +G_y -> lH_x); W of the cell above by shuffle
    float u01[4] = {0.0f, 0.0f, 0.0f, 0.0f}, u10[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    VF<4> m01 = zerov<4>(), m10 = zerov<4>();
    if (zs) {
      const VF<4> o01 = get(sm.P[se][2][w][sl]), o10 = get(sm.P[se][3][w][sl]);
      m01 = o01; m10 = o10;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        if (k0 + v == 0) continue;                      // PEC-masked nodes: W = 0, lambda_psi kept
        const float bz = sm.C[3][sl * 4 + v], cz = sm.C[4][sl * 4 + v], kz = sm.C[5][sl * 4 + v];
        u01[v] = cpml_adjoint_term(-gx.v[v], o01.v[v], bz, cz, kz, m01.v[v]);
        u10[v] = cpml_adjoint_term(gy.v[v], o10.v[v], bz, cz, kz, m10.v[v]);
      }
    }
    float u01_p = __shfl_down_sync(0xffffffffu, u01[0], 1), u10_p = __shfl_down_sync(0xffffffffu, u10[0], 1);
    if (lane == 31 || g + 1 >= ngroups) { u01_p = 0.0f; u10_p = 0.0f; }   // the cell above a tile is a plain cell (host check) or the ghost
    put(sm.G[se][w][0][lane], gx); put(sm.G[se][w][1][lane], gy); put(sm.G[se][w][2][lane], gz);
    __syncthreads();
    if (store_plane) {
      // ---- B: adjoint of the E half-step at plane i ----
      const VF<4> gx_yp = get(sm.G[se][w + 1][0][lane]), gz_yp = get(sm.G[se][w + 1][2][lane]);
      const VF<4> gy_xp = get(sm.G[se ^ 1][w][1][lane]), gz_xp = get(sm.G[se ^ 1][w][2][lane]);
      VF<4> nhx, nhy, nhz;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float gx_zq = v == 3 ? gx_zp : gx.v[v < 3 ? v + 1 : v];
        const float gy_zq = v == 3 ? gy_zp : gy.v[v < 3 ? v + 1 : v];
        nhx.v[v] = lhx.v[v] + ((gz_yp.v[v] - gz.v[v]) - (gy_zq - gy.v[v]));
        nhy.v[v] = lhy.v[v] + ((gx_zq - gx.v[v]) - (gz_xp.v[v] - gz.v[v]));
        nhz.v[v] = lhz.v[v] + ((gy_xp.v[v] - gy.v[v]) - (gx_yp.v[v] - gx.v[v]));
      }
      if (zb) {
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float u01p = v == 3 ? u01_p : u01[v < 3 ? v + 1 : v];
          const float u10p = v == 3 ? u10_p : u10[v < 3 ? v + 1 : v];
          nhx.v[v] -= (u10p - u10[v]);
          nhy.v[v] -= (u01p - u01[v]);
        }
      }
      if (zs) { stv<4>(a.pE_out[0] + qz, m01); stv<4>(a.pE_out[1] + qz, m10); }
      stv<4>(a.lHout[0] + q, nhx); stv<4>(a.lHout[1] + q, nhy); stv<4>(a.lHout[2] + q, nhz);
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
