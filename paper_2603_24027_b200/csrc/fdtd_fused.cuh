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
// shell cells, whose H^{m-1/2} the inject kernel has already put into the OUTPUT buffer; they are read from there.
// Arithmetic is that of the lean kernels (R3), so results are bit-identical to the two-kernel path.
#pragma once
#include "fdtd_dev.cuh"

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
__global__ void __launch_bounds__(32 * (FUSED_TR + 1)) k_fused_he(const __grid_constant__ Dev d, const __grid_constant__ FusedArgs a) {
  __shared__ float4 shH[2][FUSED_TR + 1][32][2];   // new Hx, Hz of the current plane, double-buffered over the march
  __shared__ float4 shE[2][FUSED_TR + 1][32][2];   // Ex, Ez of the NEXT plane (read one march step later by the row below)
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
  const bool low_yz = j < a.lo[1] || !zfull;      // INV: some element takes its new H from the output buffer
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
      const float4 t0 = shE[buf][w + 1][lane][0], t1 = shE[buf][w + 1][lane][1];
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
    if (INV && (low_yz || i < a.lo[0])) {         // shell cells: their new H is already in the output buffer (inject)
      const VF<4> ox = ldv<4>(a.Hout[0] + q), oy = ldv<4>(a.Hout[1] + q), oz = ldv<4>(a.Hout[2] + q);
      const bool all = j < a.lo[1] || i < a.lo[0];
#pragma unroll
      for (int v = 0; v < 4; ++v)
        if (all || !zv[v]) { hx.v[v] = ox.v[v]; hy.v[v] = oy.v[v]; hz.v[v] = oz.v[v]; }
    }
    // ---- hand the new H to the row above (shared memory) and to the lane above (shuffle); E of the next plane to the
    //      row below for the next march step ----
    shH[buf][w][lane][0] = make_float4(hx.v[0], hx.v[1], hx.v[2], hx.v[3]);
    shH[buf][w][lane][1] = make_float4(hz.v[0], hz.v[1], hz.v[2], hz.v[3]);
    shE[buf ^ 1][w][lane][0] = make_float4(exn.v[0], exn.v[1], exn.v[2], exn.v[3]);
    shE[buf ^ 1][w][lane][1] = make_float4(ezn.v[0], ezn.v[1], ezn.v[2], ezn.v[3]);
    const float hx_z0 = __shfl_up_sync(0xffffffffu, hx.v[3], 1), hy_z0 = __shfl_up_sync(0xffffffffu, hy.v[3], 1);
    __syncthreads();
    if (store_plane) {
      const float4 t0 = shH[buf][w - 1][lane][0], t1 = shH[buf][w - 1][lane][1];
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

}  // namespace fdtd
