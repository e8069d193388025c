// common.cuh -- shared declarations of the CUDA path (never included by oracle/).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace strata {

// Problem description in the paper's notation: B samples, H heads, head_dim D,
// token grid (L, Y, X), window (kL, kY, kX), A rotary axes.
struct Problem {
  int B, H, D;
  int L, Y, X;
  int kL, kY, kX;
  int A;        // rotary axes (0 = no RoPE)
  int pairing;  // 0: (2j, 2j+1)   1: (j, j + D/2)
  int dtype;    // 0 f32, 1 bf16
  int force_tile;  // tcgen05: use the one-tile-per-CTA kernel on pre-rotated operands even where the fused forward applies
  float scale;  // resolved softmax scale (> 0)
  long long N;  // L * Y * X
  __host__ __device__ long long rows() const { return (long long)B * N * H; }    // (b, token, h) rows
  __host__ __device__ long long elems() const { return rows() * D; }
};

// A3 (inward clamp): first key of query i's window on an axis.
__host__ __device__ inline int window_start(int i, int k, int n) {
  int s = i - k / 2;
  s = s < 0 ? 0 : s;
  return s > n - k ? n - k : s;
}

// B3: queries whose window holds key j on one axis form the interval [lo, hi] (any k >= 1).
__host__ __device__ inline void inverse_window(int j, int k, int n, int& lo, int& hi) {
  lo = (j - k + 1 <= 0) ? 0 : j - k + 1 + k / 2;
  hi = (j >= n - k) ? n - 1 : j + k / 2;
}

__device__ __forceinline__ float to_f32(float x) { return x; }
__device__ __forceinline__ float to_f32(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f32(float x);
template <> __device__ __forceinline__ float from_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

// Optional per-kernel timing (strata_na3d_set_profiling): launchers call prof_begin/prof_end around
// each kernel; both are no-ops unless profiling is on for this host thread.
void prof_begin(const char* name, cudaStream_t stream);
void prof_end(cudaStream_t stream);

// ---- launchers (each enqueues on `stream`, returns the launch error, adds to *launches) ----
// rope.cu: y = R(sign*phi) x for up to two tensors at once; in/out dtype tags 0 f32, 1 bf16.
cudaError_t launch_rope_rotate(const Problem& p, const void* x0, const void* x1, int in_dtype,
                               void* y0, void* y1, int out_dtype, const float* coords,
                               const float* freqs, float sign, cudaStream_t stream, int* launches);

// rope.cu: A1 as an fp32 table [B, L, Y, X, D/2] float2 (cos, sin), for the backward epilogues (B4).
cudaError_t launch_rope_rotate_table(const Problem& p, const void* x0, const void* x1, void* y0, void* y1,
                                     const void* table, float sign, cudaStream_t stream, int* launches);
cudaError_t launch_rope_table_f32(const Problem& p, void* table, const float* coords, const float* freqs,
                                  cudaStream_t stream, int* launches);

// na3d_fwd_plane.cu: tcgen05 forward (head_dim 64, k_L = 3), everything (A1-A6) in one kernel; whole key planes per
// softmax hand-off, Q~ in TMEM.  `fix` is plane_fwd_workspace_bytes() of device scratch (rows for the fix-up kernel).
// The fix-up list: [0] number of listed rows, [1] != 0: every row, [2 ...] up to kFixCap row ids ((b * H + h) * N + token).
// A forward kernel that exponentiates without a reference lists the rows whose sum left [kRowSumMin, kRowSumMax].
constexpr unsigned int kFixCap = 65535;
constexpr float kRowSumMax = 1.2676506e30f, kRowSumMin = 8.2718061e-25f;   // 2^100, 2^-80
bool plane_fwd_supported(const Problem& p);
size_t plane_fwd_workspace_bytes();
cudaError_t launch_fwd_plane(const Problem& p, const void* q, const void* k, const void* v, const float* coords,
                             const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches);

cudaError_t launch_fix_rows(const Problem& p, const void* q, const void* k, const void* v, const float* coords,
                            const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches);

// na3d_column.cu: column-wise attention (window (L, 1, 1)), bf16, head_dim 64, L <= 32; same `fix`.
bool column_fwd_supported(const Problem& p);
cudaError_t launch_fwd_column(const Problem& p, const void* q, const void* k, const void* v, const float* coords,
                              const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches);

// na3d_simt.cu: fp32 CUDA-core kernels on pre-rotated fp32 operands (qr, kr in workspace).
cudaError_t launch_fwd_simt(const Problem& p, const float* qr, const float* kr, const void* v,
                            void* o, float* lse, cudaStream_t stream, int* launches);
// (d_o_main: the upstream gradient the main kernels use; d_o only enters B1 with o -- they differ for the gated
// attention of PAPER.md:390, where D_i = sum_c dO_c o_c with the gated output and the raw gradient)
cudaError_t launch_bwd_simt(const Problem& p, const float* qr, const float* kr, const void* v,
                            const void* o, const void* d_o, const void* d_o_main, const float* lse, float* delta,
                            float* dqr, float* dkr, void* dv, cudaStream_t stream, int* launches);

// na3d_bwd_tc.cu: tcgen05 backward on pre-rotated bf16 operands (head_dim 64).  stat is [B, H, N] float2
// scratch; rtab the fp32 rotary table (nullptr: no rotation): the epilogues apply B4 and write bf16 dq, dk.
bool tc_bwd_supported(const Problem& p);
cudaError_t launch_bwd_tc(const Problem& p, const void* qr, const void* kr, const void* v, const void* o,
                          const void* d_o, const void* d_o_main, const float* lse, void* stat, const void* rtab, void* dq,
                          void* dk, void* dv, cudaStream_t stream, int* launches);

// normgate.cu: the elementwise steps of QK-RMSNorm and the sigmoid head gate, rows in memory order.
cudaError_t launch_rmsnorm_rows(const Problem& p, const void* x, void* y, float eps, cudaStream_t st, int* launches);
cudaError_t launch_gate_rows(const Problem& p, const void* x, void* y, const float* gate, cudaStream_t st, int* launches);
cudaError_t launch_rmsnorm_bwd_rows(const Problem& p, const void* x, void* dx, float eps, cudaStream_t st, int* launches);
cudaError_t launch_dgate_rows(const Problem& p, const void* d_o, const void* o, const float* gate, float* dgate,
                              cudaStream_t st, int* launches);

// na3d_tc_fwd.cu: tcgen05 forward on pre-rotated bf16 operands; lists rows for launch_fix_rows in `fix` (cleared here).
bool tc_fwd_supported(const Problem& p);
cudaError_t launch_fwd_tc(const Problem& p, const void* qr, const void* kr, const void* v, void* o,
                          float* lse, void* fix, cudaStream_t stream, int* launches);

}  // namespace strata
