/* roundtrip.c — a plain C99 translation unit against include/fdtd.h (tests/test_abi_c.py).
 *
 * Proves that the boundary is a C ABI: this file is compiled with gcc -std=c99 -Wall -Werror, linked against
 * libfdtd_b200.so (and libcudart for the device buffers a caller owns), and runs
 *   create -> set_design -> workspace_bytes -> set_workspace -> forward -> reverse -> store_bytes -> destroy
 * on a problem read from a binary file; the gradient it writes is compared with the oracle's by the test.
 *
 * Input file (little endian): int32 nx ny nz P nsteps k dtype interp; int32 src_comp, src_lo[3], src_hi[3];
 * int32 design_lo[3], design_hi[3]; int32 cot_lo[3], cot_hi[3], uint32 cot_mask;
 * float32 eps[nx*ny*nz]; float32 wave[nsteps]; float32 g[ncomp * cot box].
 * Output file: uint64 store_bytes; float32 grad[design box].
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include <cuda_runtime_api.h>

#include "fdtd.h"

#define CHECK(call)                                                                                  \
  do {                                                                                               \
    fdtd_status st_ = (call);                                                                        \
    if (st_ != FDTD_OK) {                                                                            \
      fprintf(stderr, "%s -> %d: %s\n", #call, (int)st_, sim ? fdtd_last_error(sim) : "(no handle)"); \
      return 2;                                                                                      \
    }                                                                                                \
  } while (0)
#define CU(call)                                                             \
  do {                                                                       \
    cudaError_t e_ = (call);                                                 \
    if (e_ != cudaSuccess) {                                                 \
      fprintf(stderr, "%s -> %s\n", #call, cudaGetErrorString(e_));          \
      return 3;                                                              \
    }                                                                        \
  } while (0)

static int rd(void* p, size_t n, FILE* f) { return fread(p, 1, n, f) == n; }

int main(int argc, char** argv) {
  fdtd_sim* sim = NULL;
  int32_t h[8], sc, slo[3], shi[3], dlo[3], dhi[3], clo[3], chi[3];
  uint32_t cmask;
  size_t N, dcells, ccells, ncomp = 0, ws_bytes;
  float *eps, *wave, *g, *grad, *eps_dev, *g_dev, *grad_dev;
  void* ws_dev;
  FILE* f;
  int c;
  if (argc != 3) { fprintf(stderr, "usage: roundtrip in.bin out.bin\n"); return 1; }
  f = fopen(argv[1], "rb");
  if (!f) { perror(argv[1]); return 1; }
  if (!rd(h, sizeof h, f) || !rd(&sc, 4, f) || !rd(slo, 12, f) || !rd(shi, 12, f) || !rd(dlo, 12, f) || !rd(dhi, 12, f) ||
      !rd(clo, 12, f) || !rd(chi, 12, f) || !rd(&cmask, 4, f)) { fprintf(stderr, "short header\n"); return 1; }
  N = (size_t)h[0] * h[1] * h[2];
  dcells = (size_t)(dhi[0] - dlo[0]) * (dhi[1] - dlo[1]) * (dhi[2] - dlo[2]);
  ccells = (size_t)(chi[0] - clo[0]) * (chi[1] - clo[1]) * (chi[2] - clo[2]);
  for (c = 0; c < 6; ++c) ncomp += (cmask >> c) & 1u;
  eps = (float*)malloc(N * 4); wave = (float*)malloc((size_t)h[4] * 4); g = (float*)malloc(ncomp * ccells * 4);
  grad = (float*)malloc(dcells * 4);
  if (!eps || !wave || !g || !grad) return 1;
  if (!rd(eps, N * 4, f) || !rd(wave, (size_t)h[4] * 4, f) || !rd(g, ncomp * ccells * 4, f)) { fprintf(stderr, "short body\n"); return 1; }
  fclose(f);

  CU(cudaMalloc((void**)&eps_dev, N * 4));
  CU(cudaMemcpy(eps_dev, eps, N * 4, cudaMemcpyHostToDevice));
  CU(cudaMalloc((void**)&g_dev, ncomp * ccells * 4));
  CU(cudaMemcpy(g_dev, g, ncomp * ccells * 4, cudaMemcpyHostToDevice));
  CU(cudaMalloc((void**)&grad_dev, dcells * 4));
  {
    const double dx = 20e-9, dt = 0.99 * dx / (299792458.0 * 1.7320508075688772);   /* PAPER.md:39-41, eq. (1) */
    CHECK(fdtd_create(&sim, h[0], h[1], h[2], dx, dt, h[3], eps_dev, NULL));
  }
  CHECK(fdtd_set_design(sim, dlo, dhi));
  ws_bytes = fdtd_workspace_bytes(sim, h[4], (fdtd_dtype)h[6], h[5], FDTD_WS_REVERSE);
  if (!ws_bytes) { fprintf(stderr, "workspace_bytes = 0\n"); return 2; }
  CU(cudaMalloc(&ws_dev, ws_bytes));
  CHECK(fdtd_set_workspace(sim, ws_dev, ws_bytes, h[4], (fdtd_dtype)h[6], h[5], FDTD_WS_REVERSE));
  {
    fdtd_source src;
    fdtd_cotangent cot;
    uint64_t sb;
    src.comp = sc;
    for (c = 0; c < 3; ++c) { src.lo[c] = slo[c]; src.hi[c] = shi[c]; cot.lo[c] = clo[c]; cot.hi[c] = chi[c]; }
    src.amp = NULL;
    src.wave = wave;
    cot.comp_mask = cmask;
    cot.g_dev = g_dev;
    CHECK(fdtd_forward(sim, h[4], &src, 1, (fdtd_dtype)h[6], h[5]));
    sb = (uint64_t)fdtd_store_bytes(sim);
    CHECK(fdtd_reverse(sim, &cot, NULL, (fdtd_interp)h[7], grad_dev));
    CHECK(fdtd_sync(sim));
    CU(cudaMemcpy(grad, grad_dev, dcells * 4, cudaMemcpyDeviceToHost));
    f = fopen(argv[2], "wb");
    if (!f) { perror(argv[2]); return 1; }
    fwrite(&sb, 8, 1, f);
    fwrite(grad, 4, dcells, f);
    fclose(f);
    printf("roundtrip: %d slots, store %llu bytes\n", fdtd_num_slots(sim), (unsigned long long)sb);
  }
  fdtd_destroy(sim);
  cudaFree(ws_dev); cudaFree(grad_dev); cudaFree(g_dev); cudaFree(eps_dev);
  free(eps); free(wave); free(g); free(grad);
  return 0;
}
