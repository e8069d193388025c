// rope.cu -- StereoRoPE rotation kernels (steps A1, A2 and B4 of DESIGN.md).
//
// the tile-centred stereographic coordinates of a token replace the row/column
// indices of axial 2D RoPE.  phi[t][j] = sum_a coords[t][a] * F[a][j]; every channel pair of a head
// vector is rotated by phi (sign = +1) or by -phi (sign = -1: the transpose, used on gradients).
//
// The angle is accumulated in fp64 and reduced to [-pi, pi] before the fp32 sincos: coordinates
// are in native-cell units (|x| up to ~1.5e3 for cfg 0), so an fp32 product would already carry
// ~1e-4 rad of rounding -- the whole fp32 error budget of BASELINE.json.
#include "common.cuh"

namespace strata {
namespace {

template <typename T> struct Pair;
template <> struct Pair<float> {
  using V = float2;
  static __device__ __forceinline__ float2 unpack(float2 v) { return v; }
  static __device__ __forceinline__ float2 pack(float a, float b) { return make_float2(a, b); }
};
template <> struct Pair<__nv_bfloat16> {
  using V = __nv_bfloat162;
  static __device__ __forceinline__ float2 unpack(__nv_bfloat162 v) { return __bfloat1622float2(v); }
  static __device__ __forceinline__ __nv_bfloat162 pack(float a, float b) { return __floats2bfloat162_rn(a, b); }
};

// One thread per (token, pair j); loops over the heads (and over both tensors) re-using the sincos.
template <typename TIn, typename TOut>
__global__ void __launch_bounds__(256)
rope_rotate_kernel(const TIn* __restrict__ x0, const TIn* __restrict__ x1, TOut* __restrict__ y0,
                   TOut* __restrict__ y1, const float* __restrict__ coords,
                   const float* __restrict__ freqs, long long tokens, int H, int D, int A,
                   int pairing, float sign) {
  const int half = D >> 1;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= tokens * half) return;
  const long long t = gid / half;
  const int j = (int)(gid - t * half);
  float cs = 1.f, sn = 0.f;
  if (A > 0) {
    double phi = 0.0;
    for (int a = 0; a < A; ++a) phi += (double)coords[t * A + a] * (double)freqs[a * half + j];
    const double r = phi - 6.283185307179586477 * rint(phi * 0.15915494309189533577);
    sincosf((float)r, &sn, &cs);
    sn *= sign;
  }
  for (int h = 0; h < H; ++h) {
    const long long base = (t * H + h) * (long long)D;
#pragma unroll
    for (int which = 0; which < 2; ++which) {
      const TIn* x = which ? x1 : x0;
      TOut* y = which ? y1 : y0;
      if (x == nullptr) continue;
      float a, b;
      if (pairing == 0) {
        float2 ab = Pair<TIn>::unpack(reinterpret_cast<const typename Pair<TIn>::V*>(x + base)[j]);
        a = ab.x; b = ab.y;
      } else {
        a = to_f32(x[base + j]); b = to_f32(x[base + j + half]);
      }
      const float ra = a * cs - b * sn, rb = a * sn + b * cs;
      if (pairing == 0) {
        reinterpret_cast<typename Pair<TOut>::V*>(y + base)[j] = Pair<TOut>::pack(ra, rb);
      } else {
        y[base + j] = from_f32<TOut>(ra); y[base + j + half] = from_f32<TOut>(rb);
      }
    }
  }
}

// A1 for the fused tensor-core kernels: one 2*D-byte table row per token (all heads of a token share
// it) of bf16x2 words, two per pair of rotary pairs (m, m+1), m even:
//   word m     = (cos phi[t][m], cos phi[t][m+1])      word m + 1 = (sin phi[t][m], sin phi[t][m+1])
// -- the operand layout of the packed bf16x2 rotation in na3d_fwd_fused.cu.  One thread per (token, m).
__global__ void __launch_bounds__(256)
rope_table_kernel(uint2* __restrict__ table, const float* __restrict__ coords, const float* __restrict__ freqs,
                  long long tokens, int half, int A) {
  const int quarter = half >> 1;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= tokens * quarter) return;
  const long long t = gid / quarter;
  const int m = 2 * (int)(gid - t * quarter);
  float cs[2], sn[2];
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    double phi = 0.0;
    for (int a = 0; a < A; ++a) phi += (double)coords[t * A + a] * (double)freqs[a * half + m + u];
    const double r = phi - 6.283185307179586477 * rint(phi * 0.15915494309189533577);
    sincosf((float)r, &sn[u], &cs[u]);
  }
  const __nv_bfloat162 c2 = __floats2bfloat162_rn(cs[0], cs[1]), s2 = __floats2bfloat162_rn(sn[0], sn[1]);
  uint2 w;
  w.x = *reinterpret_cast<const uint32_t*>(&c2);
  w.y = *reinterpret_cast<const uint32_t*>(&s2);
  table[gid] = w;
}

// A1 as an fp32 table for the backward epilogues (B4): table[t][j] = (cos phi[t][j], sin phi[t][j]).
__global__ void __launch_bounds__(256)
rope_table_f32_kernel(float2* __restrict__ table, const float* __restrict__ coords, const float* __restrict__ freqs,
                      long long tokens, int half, int A) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= tokens * half) return;
  const long long t = gid / half;
  const int j = (int)(gid - t * half);
  double phi = 0.0;
  for (int a = 0; a < A; ++a) phi += (double)coords[t * A + a] * (double)freqs[a * half + j];
  const double r = phi - 6.283185307179586477 * rint(phi * 0.15915494309189533577);
  float sn, cs;
  sincosf((float)r, &sn, &cs);
  table[gid] = make_float2(cs, sn);
}

}  // namespace

cudaError_t launch_rope_table_f32(const Problem& p, void* table, const float* coords, const float* freqs,
                                  cudaStream_t stream, int* launches) {
  const long long tokens = (long long)p.B * p.N;
  const long long threads = tokens * (p.D / 2);
  const long long grid = (threads + 255) / 256;
  if (grid <= 0 || grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin("rope_table_f32", stream);
  rope_table_f32_kernel<<<(unsigned)grid, 256, 0, stream>>>((float2*)table, coords, freqs, tokens, p.D / 2, p.A);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

cudaError_t launch_rope_table(const Problem& p, void* table, const float* coords, const float* freqs,
                              cudaStream_t stream, int* launches) {
  const long long tokens = (long long)p.B * p.N;
  const long long threads = tokens * (p.D / 4);
  const int block = 256;
  const long long grid = (threads + block - 1) / block;
  if (grid <= 0 || grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin("rope_table", stream);
  rope_table_kernel<<<(unsigned)grid, block, 0, stream>>>((uint2*)table, coords, freqs, tokens, p.D / 2, p.A);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

cudaError_t launch_rope_rotate(const Problem& p, const void* x0, const void* x1, int in_dtype,
                               void* y0, void* y1, int out_dtype, const float* coords,
                               const float* freqs, float sign, cudaStream_t stream, int* launches) {
  const long long tokens = (long long)p.B * p.N;
  const long long threads = tokens * (p.D / 2);
  const int block = 256;
  const long long grid = (threads + block - 1) / block;
  if (grid <= 0 || grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin(sign > 0 ? "rope_rotate" : "rope_unrotate", stream);
#define STRATA_ROPE(TI, TO)                                                                        \
  rope_rotate_kernel<TI, TO><<<(unsigned)grid, block, 0, stream>>>(                                \
      (const TI*)x0, (const TI*)x1, (TO*)y0, (TO*)y1, coords, freqs, tokens, p.H, p.D, p.A,        \
      p.pairing, sign)
  if (in_dtype == 0 && out_dtype == 0) STRATA_ROPE(float, float);
  else if (in_dtype == 1 && out_dtype == 0) STRATA_ROPE(__nv_bfloat16, float);
  else if (in_dtype == 0 && out_dtype == 1) STRATA_ROPE(float, __nv_bfloat16);
  else STRATA_ROPE(__nv_bfloat16, __nv_bfloat16);
#undef STRATA_ROPE
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace strata
