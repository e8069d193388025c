/*
 * strata_na3d.h -- C ABI of libstrata_na3d.so: StereoRoPE + 3D neighbourhood attention for sm_100a.
 *
 * The one data-parallel hot path of STRATA's transformer (arxiv/paper_2606_31248):
 *   PAPER.md:79     "3D Neighborhood Attention (NATTEN), with stereographic rotary position
 *                    embeddings inside local (x,y,lev) windows"
 *   PAPER.md:93-99  StereoRoPE: tile-centred stereographic coordinates (eq. (1)) "replace
 *                    row/column indices as inputs to axial 2D RoPE"
 * For every query token i = (l, y, x) of a (L x Y x X) token grid and every head:
 *   phi[t][j]   = sum_a coords[t][a] * freqs[a][j]                      rotary angle, j < d/2
 *   qrot, krot  = each channel pair of q, k rotated by phi (V is not rotated)
 *   window(i)   = box of k_L x k_Y x k_X keys starting at clamp(i_a - floor(k_a/2), 0, n_a - k_a)
 *                 on every axis (inward-clamped NATTEN window, reading R1)
 *   s_ij        = scale * qrot_i . krot_j,  j in window(i)
 *   lse_i       = ln sum_j exp(s_ij)                                      (natural log)
 *   o_i         = sum_j exp(s_ij - lse_i) v_j
 * and, for the backward, dq, dk, dv of  sum_i dO_i . o_i  including the transpose rotation R(-phi)
 * (no gradient flows to coords, freqs or through lse).
 *
 * Conventions common to every entry point
 *   - Tensors are contiguous in the fixed layouts below; base pointers must be 16-byte aligned.
 *       q, k, v, o, d_o, dq, dk, dv : [B, L, Y, X, H, d]   element type desc->dtype
 *       lse                         : [B, H, L, Y, X]      float32
 *       coords                      : [B, L, Y, X, A]      float32  (A = desc->rope_axes)
 *       freqs                       : [A, d/2]             float32
 *   - Device entry points take DEVICE pointers owned by the caller; the library allocates no
 *     device memory (scratch comes from `workspace`), never frees caller memory, never
 *     synchronises, and enqueues all work on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  They are safe to capture in a CUDA graph.
 *   - `_host` entry points take HOST pointers (pinned memory recommended) plus a DEVICE workspace;
 *     they enqueue H2D copies, the same kernels, and D2H copies on `stream` and return without
 *     synchronising: the caller synchronises the stream before reading the outputs.
 *   - Outputs are fully overwritten (gradients are not accumulated into).
 *   - Errors are return codes only: no exceptions, no abort, no printing.
 *       INVALID_ARG  null required pointer, misaligned pointer, odd or non-positive head_dim,
 *                    window[a] < 1 or > grid[a], non-positive sizes, bad enum value
 *       UNSUPPORTED  legal but not implemented (head_dim not in {32, 64, 128}; rope_axes > 3;
 *                    impl = TCGEN05 for a shape the tensor-core path does not cover)
 *       WORKSPACE    workspace null or smaller than the *_workspace_bytes query says
 *       CUDA         a CUDA runtime / driver call failed (cudaGetLastError is consumed)
 */
#ifndef STRATA_NA3D_H_
#define STRATA_NA3D_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  STRATA_OK = 0,
  STRATA_ERR_INVALID_ARG = 1,
  STRATA_ERR_UNSUPPORTED = 2,
  STRATA_ERR_WORKSPACE = 3,
  STRATA_ERR_CUDA = 4,
  STRATA_ERR_STATIC_SCRATCH = 5 /* strata_na3d_fwd_static only: needs more than STRATA_STATIC_SCRATCH_BYTES */
} strata_status_t;

typedef enum { STRATA_DTYPE_F32 = 0, STRATA_DTYPE_BF16 = 1 } strata_dtype_t;

/* Which channels form a rotary pair: (2j, 2j+1) [complex form of RoFormer] or (j, j + d/2). */
typedef enum { STRATA_ROPE_INTERLEAVED = 0, STRATA_ROPE_HALF = 1 } strata_rope_pairing_t;

/* Kernel family.  AUTO picks the tcgen05 tensor-core kernels when they cover the problem
 * (bf16, see strata_na3d_impl_selected) and the fp32 CUDA-core kernels otherwise. */
typedef enum {
  STRATA_IMPL_AUTO = 0,
  STRATA_IMPL_SIMT = 1,
  STRATA_IMPL_TCGEN05 = 2,      /* tensor-core kernels; the fused forward (na3d_fwd_plane.cu) where it applies */
  STRATA_IMPL_TCGEN05_TILE = 3  /* tensor-core kernel with one query tile per CTA (any covered shape) */
} strata_impl_t;

typedef struct {
  int32_t batch, heads, head_dim; /* B, H, d; d in {32, 64, 128}                               */
  int32_t grid[3];                /* L, Y, X (levels, y, x), each >= 1                          */
  int32_t window[3];              /* k_L, k_Y, k_X with 1 <= k_a <= grid[a]; even sizes allowed */
  int32_t rope_axes;              /* A: 0 = no RoPE, 2 = (x, y) [paper], 3 = (x, y, level)      */
  int32_t rope_pairing;           /* strata_rope_pairing_t                                      */
  int32_t dtype;                  /* strata_dtype_t of q, k, v, o, d_o, dq, dk, dv              */
  int32_t impl;                   /* strata_impl_t                                              */
  float scale;                    /* softmax scale; <= 0 means 1/sqrt(head_dim)                 */
} strata_na3d_desc_t;

/* Bytes of DEVICE scratch the device entry points need for this problem (backward != 0: for
 * strata_na3d_bwd).  0 on an invalid descriptor.  PAPER.md has no counterpart; the scratch holds
 * the rotary tables / rotated operands (A1, A2) and the backward's row statistics (B1). */
size_t strata_na3d_workspace_bytes(const strata_na3d_desc_t* desc, int backward);

/* Bytes of DEVICE scratch the _host entry points need (staging for every tensor + the above). */
size_t strata_na3d_host_workspace_bytes(const strata_na3d_desc_t* desc, int backward);

/* Kernel family AUTO resolves to for this descriptor (a strata_impl_t), or -1 if invalid. */
int strata_na3d_impl_selected(const strata_na3d_desc_t* desc, int backward);

/* Forward: A1-A6 of DESIGN.md.  Reads q, k, v, coords, freqs; writes o and
 * lse.  coords / freqs may be NULL iff rope_axes == 0. */
strata_status_t strata_na3d_fwd(const strata_na3d_desc_t* desc,
                                const void* q, const void* k, const void* v,
                                const float* coords, const float* freqs,
                                void* o, float* lse,
                                void* workspace, size_t workspace_bytes, void* stream);

/* Exponent range of the tensor-core forwards, and what leaving it costs.  The bf16 tensor-core kernels
 * (strata_na3d_impl_selected == STRATA_IMPL_TCGEN05) exponentiate scale * q~ . k~ without subtracting a row maximum.
 * A row whose sum of exponentials leaves [2^-80, 2^100] (|logit| beyond ~55..69: "logits reach +-100..1000 without
 * QK-norm", App. B.5) is listed in the workspace and recomputed exactly, one warp per row, by a second kernel
 * that every such call enqueues: a few listed rows cost microseconds.  But when more than 65 535 rows are listed, or
 * when (fused head_dim-64 forward, column kernel) the rotary coordinates of a (y, x) column differ between levels,
 * EVERY row is recomputed that way: still exact, about two orders of magnitude slower, and not predictable from the
 * descriptor.  To see it, read the first 16 bytes of `workspace` after the stream has completed the call: two
 * uint64, [0] = rows listed (counts past 65 535 too), [1] != 0 = every row was recomputed.  With QK-RMSNorm
 * (|logit| <= sqrt(head_dim)) and the paper's level-independent coordinates neither happens.  Only the row SUM is
 * checked: inputs with |v| near the bf16 maximum can still overflow the fp32 output accumulator. */

/* Backward: B1-B4 of DESIGN.md.  o and lse are the forward's outputs for the same inputs.
 * Writes dq, dk, dv (same layout and dtype as q). */
strata_status_t strata_na3d_bwd(const strata_na3d_desc_t* desc,
                                const void* q, const void* k, const void* v,
                                const void* o, const void* d_o, const float* lse,
                                const float* coords, const float* freqs,
                                void* dq, void* dk, void* dv,
                                void* workspace, size_t workspace_bytes, void* stream);

/* ---- QK-RMSNorm and the sigmoid head gate around the attention (App. B.5) -------------------------
 * "QK RMSNorm, which applies RMSNorm (without learnable scale) to the query and key vectors before their dot
 * product" and "gated attention, which applies a head-specific sigmoid gate to the attention output":
 *   q^ = q / sqrt(mean_c q_c^2 + eps)  (per (token, head) vector; same for k),   a, lse = NA3D(RoPE(q^), RoPE(k^), v),
 *   o = sigmoid(gate[b, l, y, x, h]) * a.
 * gate: float32 logits [B, L, Y, X, H] (DEVICE), NULL = no gate.  eps >= 0.  lse is that of the normalised logits.
 * The backward takes the GATED output o of the forward and the gradient d_o wrt it; writes dq, dk, dv and, with a
 * gate, dgate [B, L, Y, X, H] float32.  Workspace: strata_na3d_normgate_workspace_bytes (device memory).
 * In this version the normalisation and the gate run as streaming kernels around strata_na3d_fwd / _bwd (one extra
 * read + write of Q and K, one of O); everything else (layouts, asynchrony, errors) as for those calls. */
size_t strata_na3d_normgate_workspace_bytes(const strata_na3d_desc_t* desc, int backward);
strata_status_t strata_na3d_normgate_fwd(const strata_na3d_desc_t* desc,
                                         const void* q, const void* k, const void* v,
                                         const float* coords, const float* freqs, const float* gate, float eps,
                                         void* o, float* lse,
                                         void* workspace, size_t workspace_bytes, void* stream);
strata_status_t strata_na3d_normgate_bwd(const strata_na3d_desc_t* desc,
                                         const void* q, const void* k, const void* v,
                                         const void* o, const void* d_o, const float* lse,
                                         const float* coords, const float* freqs, const float* gate, float eps,
                                         void* dq, void* dk, void* dv, float* dgate,
                                         void* workspace, size_t workspace_bytes, void* stream);

/* Same operations on HOST buffers; `workspace` is DEVICE memory of at least
 * strata_na3d_host_workspace_bytes() (two staging slots of ONE sample each + the device scratch of a one-sample
 * call).  The samples of the batch are independent: they go through one at a time, the copies in of
 * sample b + 1 and the copies out of sample b - 1 overlapping the kernels of sample b on two internal streams that
 * are joined back into `stream` before the call returns.  Asynchronous and ordered on `stream`; the host buffers
 * should be page-locked (pageable memory makes the copies synchronous) and must stay valid until the work on `stream`
 * has completed. */
strata_status_t strata_na3d_fwd_host(const strata_na3d_desc_t* desc,
                                     const void* q, const void* k, const void* v,
                                     const float* coords, const float* freqs,
                                     void* o, float* lse,
                                     void* workspace, size_t workspace_bytes, void* stream);

strata_status_t strata_na3d_bwd_host(const strata_na3d_desc_t* desc,
                                     const void* q, const void* k, const void* v,
                                     const void* o, const void* d_o, const float* lse,
                                     const float* coords, const float* freqs,
                                     void* dq, void* dk, void* dv,
                                     void* workspace, size_t workspace_bytes, void* stream);

/* ---- forward for callers that have no device memory to hand over ---------------------------------------------------
 * strata_na3d_fwd wants a `workspace` that the caller allocated.  Some callers cannot get one: a plug-in running
 * inside a host application whose memory pool has already claimed the whole GPU (a cudaMalloc there fails, or takes
 * memory the host has promised elsewhere), code that is called inside a latency-critical loop where the implicit
 * device synchronisation of cudaMalloc / cudaFree is not acceptable, and code that runs where the allocator may not be
 * called at all (between the host's "no more allocations" point and shutdown).  For them this one call runs the same
 * forward (same kernels, same results, same argument meaning as strata_na3d_fwd) with the scratch taken from a
 * fixed array of STRATA_STATIC_SCRATCH_BYTES that is part of the library image: every GPU on which the library is
 * loaded holds that 1 MiB from load until the process exits, used or not.
 *   - The call allocates nothing: no cudaMalloc, no cudaFree, no allocating library routine, on any call.  (Keep
 *     strata_na3d_set_profiling off around it: the profiler creates CUDA events.)
 *   - Limit: the problem's scratch need, strata_na3d_workspace_bytes(desc, 0), must be <= STRATA_STATIC_SCRATCH_BYTES,
 *     else STRATA_ERR_STATIC_SCRATCH is returned and nothing is enqueued.  The fused bf16 forward (head_dim 64,
 *     k_L = 3: configs 1 and 3) and the column-wise forward need 524 544 bytes at ANY batch and grid size; the fp32
 *     kernels and the bf16 tile kernel keep rotated copies of Q and K in scratch and fit up to B * L * Y * X * H * d
 *     = 131 072 elements (config 0 has 65 536).  There is no such variant of the backward.
 *   - The first call on each device (with that device current) looks up the array's address on that device; every
 *     later call on it reuses the address.  Make that first call before starting any stream capture.
 *   - All calls on a device share the one array, and it keeps what the previous call left in it.  The only part that
 *     has to start at zero -- the 16-byte header (row count, take-all flag) of the list of rows for the fix-up kernel
 *     -- is cleared on `stream` by every call before its kernels; the rest is written before it is read.  Two calls
 *     that can overlap on the GPU (different streams without an event between them, or different host threads on the
 *     same device) race on the array and give wrong results: order them on one stream or with events.  A call that
 *     uses strata_na3d_fwd with its own workspace never touches the array.
 *   - The sentence on CUDA graphs in the conventions at the top of this header was written for the calls that take a
 *     workspace; nothing is stated here, either way, about capturing this call. */
#define STRATA_STATIC_SCRATCH_BYTES 1048576
strata_status_t strata_na3d_fwd_static(const strata_na3d_desc_t* desc,
                                       const void* q, const void* k, const void* v,
                                       const float* coords, const float* freqs,
                                       void* o, float* lse, void* stream);

/* Number of kernel launches the last successful call on this thread enqueued (for bench.py's
 * `gpu_launches`; memcpy nodes are not counted). */
int strata_na3d_last_launch_count(void);

/* Per-kernel device timing for bench.py's roofline line.  While profiling is enabled (per host
 * thread), every kernel a device entry point launches is bracketed by CUDA events recorded on
 * `stream` (up to 4096 kernels; later ones are not recorded).  After the caller has synchronised
 * the stream, strata_na3d_profile_read copies the durations (milliseconds, launch order) of all
 * kernels recorded since profiling was enabled into ms[0..capacity) and returns their number (-1 if
 * an event query failed); names[i], if names != NULL, receives a static string naming kernel i.
 * strata_na3d_set_profiling(1) also clears the record.  Do not enable it while capturing a graph. */
void strata_na3d_set_profiling(int enable);
int strata_na3d_profile_read(float* ms, const char** names, int capacity);

/* Host-side index helpers the kernels use, exported so that CPU tests can hold them against brute
 * force.  strata_na3d_window_start: A3, first key of query i's window on an axis of n tokens with
 * window k.  strata_na3d_inverse_window: B3, the queries whose window holds key j form the interval
 * [*lo, *hi] (inclusive).  Both return -1 on invalid arguments (k < 1, k > n, index outside [0, n)). */
int strata_na3d_window_start(int i, int k, int n);
int strata_na3d_inverse_window(int j, int k, int n, int* lo, int* hi);

/* ---- geometry of the StereoRoPE inputs on the device --------------------------------------
 * Both calls are elementwise over n points, asynchronous on `stream`, and take DEVICE pointers.  lat / lon are
 * float64 radians (the coordinates reach ~1.5e3 at l_scale of the 2048^2-cell faces: float32 inputs would not
 * resolve the float32 result).
 *
 * strata_stereo_coords: eq. (1).  Tile-centred stereographic coordinates of the points
 * (lat[i], lon[i]) about the tile centre (lat0, lon0), divided by l_scale = sqrt(4 pi / n_total):
 *   cos c = sin p0 sin p + cos p0 cos p cos(l - l0),  k = 2 / (1 + cos c),
 *   x = (k / l_scale) cos p sin(l - l0),  y = (k / l_scale) (cos p0 sin p - sin p0 cos p cos(l - l0)).
 * Writes coords[i * stride + 0] = x, coords[i * stride + 1] = y (float32; stride >= 2: the [.., A] layout of
 * strata_na3d_fwd's coords with A = stride).  INVALID_ARG if n < 0, stride < 2, n_total <= 0 or a pointer is NULL.
 *
 * strata_wind_to_tile_frame: eq. (2).  The wind (u[i], v[i]) (East, North at its own point)
 * as a 3D vector, projected onto the tangent plane at the tile centre, in the centre's East-North frame:
 *   v3 = u e + v n,  v_perp = v3 - (v3 . r0) r0,  u_loc = v_perp . e0,  v_loc = v_perp . n0.
 * u_loc / v_loc may alias u / v. */
strata_status_t strata_stereo_coords(const double* lat, const double* lon, long long n, double lat0, double lon0,
                                     double n_total, float* coords, int stride, void* stream);
strata_status_t strata_wind_to_tile_frame(const float* u, const float* v, const double* lat, const double* lon,
                                          long long n, double lat0, double lon0, float* u_loc, float* v_loc,
                                          void* stream);

/* strata_tile_stitch: eq. (5), S = D^-1 P^T W: "each tile's output is weighted by a 2D ... window ...;
 * the final value at each grid cell is the weighted average of all overlapping tile outputs".  tiles [T, C, th, tw]
 * float32; origins [T, 2] int32 = (y0, x0) of each tile in the [C, gh, gw] field (tiles inside the field: P copies
 * cells; cross-face interpolation is not modelled); wy [th], wx [tw]: the separable window (an input: the paper names a
 * Kaiser-Bessel-derived window without parameters; a top-hat makes this a crop).  Cells no tile covers with a
 * positive weight are set to 0.  All pointers DEVICE memory; asynchronous on `stream`. */
strata_status_t strata_tile_stitch(const float* tiles, const int32_t* origins, int n_tiles, int channels, int th, int tw,
                                   const float* wy, const float* wx, float* out, int gh, int gw, void* stream);

const char* strata_status_string(strata_status_t status);
int strata_version(void);

#ifdef __cplusplus
}
#endif
#endif /* STRATA_NA3D_H_ */
