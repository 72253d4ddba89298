/* fdtd.h — C ABI of the B200-native time-reversible FDTD gradient loop with compressed boundary storage.
 *
 * Method: arxiv/paper_2603_24027.  Time-reversible gradient computation "begins at the final time
 * step of the forward simulation and propagates backward through time"; because PML is "non-invertible in
 * time, field values for these boundaries need to be saved during the forward simulation".  The
 * paper's two contributions are applied to that boundary store: "converting the recorded field values to
 * smaller bit-widths" and casting them back in the reverse run, and "subsampling at every k-th
 * time step and applying linear interpolation".  Everything the paper leaves open (staggering,
 * normalisation, CPML constants, injection order, rounding order) follows the readings R1..R19 in DESIGN.md.
 *
 * Conventions
 *  - Pointers named *_dev are CUDA device pointers owned by the caller (e.g. torch tensors); the library never
 *    frees them.  Pointers named *_host are host pointers.  All field-shaped arrays are float32, C-contiguous
 *    [nx][ny][nz] (z fastest).  Component order is Ex,Ey,Ez,Hx,Hy,Hz = 0..5; boxes are half-open [lo,hi).
 *  - Every call returns fdtd_status (FDTD_OK = 0) and never throws; fdtd_last_error() gives the message.
 *  - Calls enqueue work on the stream given at create and do NOT synchronise unless stated; asynchronous CUDA
 *    errors surface on a later call or on fdtd_sync().  *_host calls synchronise before returning.
 *  - The library allocates no device memory: all state lives in the caller's workspace (fdtd_set_workspace).
 *  - There is no CPU fallback: every step of the path runs in the sm_100a kernels of this library.
 */
#ifndef FDTD_B200_H
#define FDTD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdtd_sim fdtd_sim; /* opaque handle, owned by the library, freed by fdtd_destroy */

typedef enum {
  FDTD_OK = 0,
  FDTD_ERR_INVALID_ARG = 1, /* bad sizes, boxes outside the interior, k < 1, dt above the CFL limit, eps < 1 ... */
  FDTD_ERR_OOM = 2,         /* workspace missing or too small for the requested run */
  FDTD_ERR_CUDA = 3,        /* a CUDA runtime call or kernel failed */
  FDTD_ERR_STATE = 4,       /* call order violated, e.g. reverse before forward */
  FDTD_ERR_UNSUPPORTED = 5
} fdtd_status;

/* Storage type of the interface store.  F8E4M3_SCALED = OCP E4M3 ("e4m3fn", max 448) with one
 * float32 absmax scale per (slot, face, component) slice — DESIGN.md R13/R14. */
typedef enum {
  FDTD_F32 = 0, FDTD_F16 = 1, FDTD_BF16 = 2, FDTD_F8E4M3_SCALED = 3,
  /* Micro-scaled E4M3 (SURVEY 8(f)-1 "finer scale granularity"; R20): every slice is cut into blocks of 32
   * consecutive values that share one power-of-two scale 2^X, X = the smallest integer with amax * 2^-X <= 448 (clamped
   * to [-127, 127]), stored as the byte X + 127 behind the slot's codes: slot = [slot_values codes][sum over slices of ceil(face/32) scale bytes]. */
  FDTD_F8E4M3_MX32 = 5,
  /* The paper's own float8 flavours, cast WITHOUT a scale, exactly like an array astype: round to
   * nearest even, subnormals kept; a value above the largest finite one becomes NaN ("fn"/"fnuz": no infinities) or
   * inf (e4m3, e3m4).  e4m3b11fnuz with k = 16 is the paper's 64x configuration.  Software casts (no hardware cvt). */
  FDTD_F8E4M3B11FNUZ = 10, /* bias 11, max 30,    min subnormal 2^-13 */
  FDTD_F8E5M2FNUZ = 11,    /* bias 16, max 57344, min subnormal 2^-17 */
  FDTD_F8E4M3FNUZ = 12,    /* bias 8,  max 240,   min subnormal 2^-10 */
  FDTD_F8E4M3 = 13,        /* IEEE-like, bias 7, max 240,  min subnormal 2^-9 */
  FDTD_F8E3M4 = 14         /* IEEE-like, bias 3, max 15.5, min subnormal 2^-6 */
} fdtd_dtype;
/* Temporal interpolation between stored steps: linear is the paper's; cubic = 4-point Lagrange. */
typedef enum { FDTD_LINEAR = 0, FDTD_CUBIC = 1 } fdtd_interp;

/* Additive soft source: in step m (1-based) E_comp += amp * wave[m-1] on the box (R8).  Sources of one component whose
 * boxes overlap are added in index order (one launch per source instead of one for all), so the sum is the same on every run. */
typedef struct {
  int comp;          /* 0..2 = Ex,Ey,Ez */
  int lo[3], hi[3];  /* cell box inside the interior */
  const float* amp;  /* [hi-lo] spatial amplitude or NULL (= 1).  DEVICE pointer for fdtd_forward, HOST pointer
                        for fdtd_forward_host */
  const float* wave; /* HOST array of length nsteps (copied during the call) */
} fdtd_source;

/* Cotangent of the final state on a box: lambda_comp += g on the box before the reverse sweep. */
typedef struct {
  int lo[3], hi[3];
  unsigned comp_mask; /* bit c set: component c (0..5) present, in increasing c */
  const float* g_dev; /* [ncomp][hi-lo] */
} fdtd_cotangent;

/* ---------------------------------------------------------------------------------------------------------
 * The four calls BASELINE.json's north_star names
 * ------------------------------------------------------------------------------------------------------- */

/* Create a simulation (eq. 1): grid nx*ny*nz cells of size dx [m], time step dt [s] (must satisfy
 * dt <= dx/(c*sqrt(3)); the Courant number used by the kernels is S = c*dt/dx), CPML of pml_width cells on all six
 * faces backed by a PEC wall (R4,R5), relative permittivity eps_dev[nx][ny][nz] (all >= 1; read during
 * fdtd_set_workspace / fdtd_set_eps, and again by fdtd_reverse, so it must stay valid and unchanged).
 * cuda_stream is a cudaStream_t (NULL = default stream).  Requires n_a - 2*pml_width >= 2 on every axis.
 * Synchronises once (eps validation). */
fdtd_status fdtd_create(fdtd_sim** out, int nx, int ny, int nz, double dx, double dt, int pml_width,
                        const float* eps_dev, void* cuda_stream);

/* Forward run of nsteps leapfrog steps from the current state (zeros after set_workspace/reset): E half-step with
 * CPML psi_E, sources, H half-step with psi_H (R1-R5), monitor write, and the record step:
 * state m is cast to store_dtype and written to the interface store when m % k == 0 or m == nsteps, state 0
 * included (R6,R7,R10).  FDTD_ERR_OOM if the workspace is too small,
 * FDTD_ERR_INVALID_ARG for nsteps < 1, k < 1 or a source outside the interior.
 * Repeated calls without fdtd_reset in between (R21; SURVEY 8(b) sketched "extend the run"): the FIELDS continue
 * from the current state, but every call opens a new SEGMENT — the store is recorded anew from this call's first state, the
 * monitor rows and the source samples are counted from this call's step 1 — and fdtd_reverse unwinds the last segment only
 * (the gradient of a loss on that segment with the segment's initial state held fixed). */
fdtd_status fdtd_forward(fdtd_sim*, int nsteps, const fdtd_source* src, int nsrc, fdtd_dtype store_dtype, int k);

/* Reverse run (step order DESIGN.md R9): starting from the live final state, for m = nsteps..1
 * invert the H and E half-steps on the inner interior, overwrite the interface shell with the dequantised,
 * interpolated stored values, carry the adjoint fields (transposed Yee + transposed CPML) on all cells, add the
 * cotangents (dL_dfinal once, dL_dmon_dev[m-1] every step; either may be NULL) and accumulate dL/d(1/eps) on the
 * design box.  grad_eps_dev [design box] is overwritten with dL/d(eps_r) (float32); NULL or no design box = skip.
 * Leaves the reconstructed state 0 in the interior of the fields.  FDTD_ERR_STATE without a prior forward with
 * reverse-capable workspace. */
fdtd_status fdtd_reverse(fdtd_sim*, const fdtd_cotangent* dL_dfinal, const float* dL_dmon_dev, fdtd_interp interp,
                         float* grad_eps_dev);

/* Bytes of the interface store of the last forward run, scales included:
 * nslots * (slot_values * sizeof(store_dtype) + (FDTD_F8E4M3_SCALED ? slices*4 : 0) + (FDTD_F8E4M3_MX32 ? blocks : 0));
 * 0 before any forward. */
size_t fdtd_store_bytes(const fdtd_sim*);

/* ---------------------------------------------------------------------------------------------------------
 * Auxiliaries
 * ------------------------------------------------------------------------------------------------------- */

/* CPML constants (ref. 17; the paper prints none — DESIGN.md R5).  Defaults 0.8, 1, 0.01, 3.
 * Must be called before fdtd_set_workspace. */
fdtd_status fdtd_set_cpml(fdtd_sim*, double sigma_factor, double kappa_max, double alpha_max, double grade_m);
/* Design box (inside the interior) over which dL/d(eps) is accumulated.  Before fdtd_set_workspace. */
fdtd_status fdtd_set_design(fdtd_sim*, const int lo[3], const int hi[3]);
/* Monitor: after every step m the components in comp_mask on the box are written to
 * record_dev[(m-1)][ncomp][box] (caller-owned, >= nsteps*ncomp*box floats).  record_dev may be NULL to clear. */
fdtd_status fdtd_set_monitor(fdtd_sim*, const int lo[3], const int hi[3], unsigned comp_mask, float* record_dev);

/* What each interface face stores (before fdtd_set_workspace).  FDTD_STORE_ALL (default, R6): all six field
 * components, 36 slices per slot.  FDTD_STORE_TANGENTIAL: only what the inner interior ever reads from the
 * shell — the two H components tangential to each LOW face and the two E components tangential to each HIGH face, 12 slices
 * per slot: a third of the bytes on top of dtype and k.  The shell itself is then not reconstructed in the reverse run:
 * the design box must lie in the inner interior [P+1, n-P-1) (fdtd_reverse answers FDTD_ERR_INVALID_ARG otherwise), and
 * the fields left after fdtd_reverse are state 0 on the inner interior only.  Slot layout: [face][2 comps ascending][u][v]. */
#define FDTD_STORE_ALL 0
#define FDTD_STORE_TANGENTIAL 1
fdtd_status fdtd_set_store_mode(fdtd_sim*, int mode);

/* Workspace: the caller allocates device memory, the library sub-allocates fields, psi, adjoint fields, the
 * store and staging buffers from it.  flags: bit 0 = reverse pass buffers, bit 1 = staging for the *_host calls.
 * nsrc_cells = total number of source amplitude cells (host staging only; 0 otherwise). */
#define FDTD_WS_REVERSE 1u
#define FDTD_WS_HOST_IO 2u
size_t fdtd_workspace_bytes(const fdtd_sim*, int nsteps, fdtd_dtype store_dtype, int k, unsigned flags);
/* Installs the workspace (256-byte aligned), builds S/eps and the CPML tables, zeroes the state.  The sizes
 * (nsteps, dtype, k, flags) are the maxima later runs may use. */
fdtd_status fdtd_set_workspace(fdtd_sim*, void* ws_dev, size_t bytes, int nsteps, fdtd_dtype store_dtype, int k,
                               unsigned flags);
/* New permittivity (next design iteration): rebuilds S/eps, zeroes the state. */
fdtd_status fdtd_set_eps(fdtd_sim*, const float* eps_dev);
/* Zero E, H, psi (state 0) and drop the store. */
fdtd_status fdtd_reset(fdtd_sim*);
/* Replay runs of k steps through CUDA graphs (default 1 = on). */
fdtd_status fdtd_set_graphs(fdtd_sim*, int enabled);
/* Fused marching kernels (two dependent half-steps per pass over the rows of the lean x-y range): mode -1
 * (default) = forward run, reverse primal and adjoint fused where the marching kernels have at least one block per multiprocessor
 * (256x256x128 and larger; 128^3 lives in L2 and keeps the split kernels); 0 = never; 1 = forward, reverse primal and adjoint
 * whenever the grid allows (nz % 4 == 0, pml_width % 4 == 0, pml_width >= 4, nz - 2 * pml_width >= 8).  xseg = planes marched per block (0 = chosen by the
 * library: 16 or 32 in the forward run; in the reverse run the count in [16, 64] with the fewest waves x (planes + 1)).  Results are bit-identical
 * in every mode (sources that overlap on one cell excepted in the fused reverse run: they are summed before being subtracted).
 * With the fused reverse run the fields left after fdtd_reverse are state 0 on the interior only. */
fdtd_status fdtd_set_fused(fdtd_sim*, int mode, int xseg);
/* Row kernels: the plain cells and the z-slab cells of the same rows in one launch, so that whole rows
 * are streamed.  mode -1 (default) = on grids that stream from HBM (forward working set > 1.5 x L2), 0 = never, 1 = whenever
 * the vector path applies (nz % 4 == 0, pml_width % 4 == 0).  Bit-identical results in every mode.  Before fdtd_set_workspace. */
fdtd_status fdtd_set_rows(fdtd_sim*, int mode);
/* 1 if fdtd_forward(nsteps) would take the fused path with the current settings (after fdtd_set_workspace), else 0. */
int fdtd_uses_fused(const fdtd_sim*, int nsteps);
/* 1 if fdtd_reverse would rebuild the primal with the fused marching kernel (inverse-H + inverse-E in one pass), else 0. */
int fdtd_uses_fused_reverse(const fdtd_sim*);
/* 1 if fdtd_reverse would also carry the adjoint fields with the adjoint marching kernel (adjoint of H + adjoint of E in one pass). */
int fdtd_uses_fused_adjoint(const fdtd_sim*);

/* Current fields: out_dev[6][nx][ny][nz].  fdtd_get_box: out_dev[ncomp][hi-lo] for the components in comp_mask. */
fdtd_status fdtd_get_fields(fdtd_sim*, float* out_dev);
fdtd_status fdtd_get_box(fdtd_sim*, const int lo[3], const int hi[3], unsigned comp_mask, float* out_dev);
/* Adjoint fields after fdtd_reverse: out_dev[6][nx][ny][nz] (lambda_E, lambda_H). */
fdtd_status fdtd_get_adjoint(fdtd_sim*, float* out_dev);

/* Interface store introspection (layout: DESIGN.md "Store layout"): slot j holds state min(j*k, nsteps) as
 * [face 0..5][comp 0..5][u][v] in store_dtype, face = 2*axis + side. */
int fdtd_num_slots(const fdtd_sim*);
size_t fdtd_slot_values(const fdtd_sim*);
fdtd_status fdtd_slot_ptr(const fdtd_sim*, int j, const void** data_dev, const float** scales_dev /* [36] */);
/* Bytes one slot occupies at data_dev for the given store dtype (codes, plus the block-scale bytes of FDTD_F8E4M3_MX32;
 * the float32 slice scales of FDTD_F8E4M3_SCALED live in scales_dev and are not counted).  0 for an unknown dtype. */
size_t fdtd_slot_bytes(const fdtd_sim*, fdtd_dtype store_dtype);

/* ---------------------------------------------------------------------------------------------------------
 * Host-buffer variants (end-to-end path): same computation, host<->device copies inside the call, synchronous.
 * Need a workspace created with FDTD_WS_HOST_IO (and FDTD_WS_REVERSE for fdtd_reverse_host).
 * ------------------------------------------------------------------------------------------------------- */
fdtd_status fdtd_set_eps_host(fdtd_sim*, const float* eps_host /* [nx][ny][nz] */);
/* src[].amp are HOST pointers; mon_host (may be NULL) receives the monitor record [nsteps][ncomp][box]. */
fdtd_status fdtd_forward_host(fdtd_sim*, int nsteps, const fdtd_source* src, int nsrc, fdtd_dtype store_dtype, int k,
                              float* mon_host);
/* dmon_host: per-step monitor cotangents [nsteps][ncomp][box] or NULL; grad_eps_host [design box]. */
fdtd_status fdtd_reverse_host(fdtd_sim*, const float* dmon_host, fdtd_interp interp, float* grad_eps_host);

/* ---------------------------------------------------------------------------------------------------------
 * Stand-alone codec entry points: the same device functions the record / inject kernels use, exposed so that
 * quantise, dequantise and interpolate can be checked bit for bit on identical slices.
 * ------------------------------------------------------------------------------------------------------- */
/* Encode one slice x_dev[n] (float32) to codes_dev[n * sizeof(dtype)]; scale_dev[1] receives the slice scale
 * (1 unless FDTD_F8E4M3_SCALED).  scratch_dev: one uint32 used for the absmax reduction.  FDTD_F8E4M3_MX32: codes_dev
 * must hold n + ceil(n/32) bytes — the codes, then one scale byte per block of 32 values (the slot convention). */
fdtd_status fdtd_codec_encode(fdtd_dtype dtype, const float* x_dev, size_t n, void* codes_dev, float* scale_dev,
                              unsigned* scratch_dev, void* cuda_stream);
/* Dequantise and interpolate: out_dev[i] = value at (num/den) between slices 1 and 2 (linear: slices 1,2; cubic:
 * slices 0..3 = steps -1,0,1,2).  num == 0 returns slice 1 exactly.  scales[4] are HOST floats (ignored by
 * FDTD_F8E4M3_MX32, whose block-scale bytes follow the n codes in each codes_dev[j]). */
fdtd_status fdtd_codec_fetch(fdtd_dtype dtype, fdtd_interp interp, const void* const codes_dev[4],
                             const float scales[4], int num, int den, size_t n, float* out_dev, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * Allocation-free variant of the slice encoder, for callers that cannot allocate device memory around the call (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Encodes a batch of nslices equally long slices,
 * x_dev[nslices][slice_len] (float32), exactly as fdtd_codec_encode does slice by slice (R12-R14):
 * codes_dev[nslices][slice_len * sizeof(dtype)], scales_dev[nslices] (1 unless FDTD_F8E4M3_SCALED).  The absmax reduction words
 * that fdtd_codec_encode takes from the caller (scratch_dev) live in a file-scope `static __device__` array of the library
 * instead: FDTD_NOALLOC_MAX_SLICES words = 16 KiB, held by every GPU that loads the library until the process exits.  The call
 * performs no cudaMalloc / cudaFree and calls no allocating library routine; the caller still owns inputs and outputs.
 *  - nslices > FDTD_NOALLOC_MAX_SLICES, nslices < 1, slice_len < 1 or FDTD_F8E4M3_MX32 (its slot layout carries scale bytes
 *    behind the codes: use fdtd_codec_encode) -> FDTD_ERR_INVALID_ARG / FDTD_ERR_UNSUPPORTED, message in
 *    fdtd_noalloc_last_error().
 *  - The array is shared by ALL calls on a device and keeps the last call's contents: each call clears the words it uses, on
 *    its stream, before reducing into them.  Calls that overlap on the GPU (different streams, or two host threads) race on it:
 *    serialise them (one stream, or an event between them).
 *  - Enqueues on cuda_stream and does not synchronise. */
#define FDTD_NOALLOC_MAX_SLICES 4096
fdtd_status fdtd_codec_encode_slices_noalloc(fdtd_dtype dtype, const float* x_dev, int nslices, size_t slice_len, void* codes_dev,
                                             float* scales_dev, void* cuda_stream);
/* Message of the last failed fdtd_codec_encode_slices_noalloc call of this host thread ("" if none). */
const char* fdtd_noalloc_last_error(void);

fdtd_status fdtd_sync(fdtd_sim*);
const char* fdtd_last_error(const fdtd_sim*);
void fdtd_destroy(fdtd_sim*);
#ifdef __cplusplus
}
#endif
#endif /* FDTD_B200_H */
