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

// A1 + A2 for bf16 -> bf16 (the operands of the tensor-core kernels that take pre-rotated Q, K): 16-byte
// accesses, one thread per (token, group of 8 channels) looping over the heads and both tensors with the
// group's cos / sin in registers.  The result is rounded to bf16 (2^-9), so the angle is reduced and
// evaluated in fp32 (two-term Cody-Waite, MUFU sin / cos: ~1e-4 abs at |phi| ~ 2e3 rad).
// PAIR 0: group = channels [8g, 8g+8) = pairs 4g .. 4g+3.  PAIR 1: group = pairs 8g .. 8g+7, i.e. channels
// [8g, 8g+8) and [D/2 + 8g, D/2 + 8g + 8).
template <int PAIR>
__global__ void __launch_bounds__(256)
rope_rotate_bf16_kernel(const __nv_bfloat16* __restrict__ x0, const __nv_bfloat16* __restrict__ x1,
                        __nv_bfloat16* __restrict__ y0, __nv_bfloat16* __restrict__ y1, const float* __restrict__ coords,
                        const float* __restrict__ freqs, long long tokens, int H, int D, int A, float sign) {
  constexpr int NP = PAIR ? 8 : 4;
  const int half = D >> 1, groups = half / NP;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= tokens * groups) return;
  const long long t = gid / groups;
  const int g = (int)(gid - t * groups);
  float cs[NP], sn[NP];
#pragma unroll
  for (int u = 0; u < NP; ++u) {
    float phi = 0.f;
    for (int a = 0; a < A; ++a) phi = fmaf(coords[t * A + a], freqs[a * half + NP * g + u], phi);
    const float n = rintf(phi * 0.15915494309189535f);
    const float r = fmaf(n, 1.7484555e-7f, fmaf(n, -6.2831854820251465f, phi));
    __sincosf(r, &sn[u], &cs[u]);
    sn[u] *= sign;
  }
  for (int h = 0; h < H; ++h) {
    const long long base = (t * H + h) * (long long)D;
#pragma unroll
    for (int which = 0; which < 2; ++which) {
      const __nv_bfloat16* x = which ? x1 : x0;
      __nv_bfloat16* y = which ? y1 : y0;
      if (x == nullptr) continue;
      if (PAIR == 0) {
        uint4 v = *reinterpret_cast<const uint4*>(x + base + 8 * g);
        uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const float2 ab = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&w[u]));
          const __nv_bfloat162 r2 = __floats2bfloat162_rn(ab.x * cs[u] - ab.y * sn[u], ab.x * sn[u] + ab.y * cs[u]);
          w[u] = *reinterpret_cast<const uint32_t*>(&r2);
        }
        *reinterpret_cast<uint4*>(y + base + 8 * g) = make_uint4(w[0], w[1], w[2], w[3]);
      } else {
        uint4 va = *reinterpret_cast<const uint4*>(x + base + 8 * g), vb = *reinterpret_cast<const uint4*>(x + base + half + 8 * g);
        uint32_t wa[4] = {va.x, va.y, va.z, va.w}, wb[4] = {vb.x, vb.y, vb.z, vb.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const float2 a2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wa[u]));
          const float2 b2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wb[u]));
          const __nv_bfloat162 ra = __floats2bfloat162_rn(a2.x * cs[2 * u] - b2.x * sn[2 * u], a2.y * cs[2 * u + 1] - b2.y * sn[2 * u + 1]);
          const __nv_bfloat162 rb = __floats2bfloat162_rn(a2.x * sn[2 * u] + b2.x * cs[2 * u], a2.y * sn[2 * u + 1] + b2.y * cs[2 * u + 1]);
          wa[u] = *reinterpret_cast<const uint32_t*>(&ra);
          wb[u] = *reinterpret_cast<const uint32_t*>(&rb);
        }
        *reinterpret_cast<uint4*>(y + base + 8 * g) = make_uint4(wa[0], wa[1], wa[2], wa[3]);
        *reinterpret_cast<uint4*>(y + base + half + 8 * g) = make_uint4(wb[0], wb[1], wb[2], wb[3]);
      }
    }
  }
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

// A2 from that table, bf16 -> bf16: one thread per ((token, head) row, group of 8 channels) and tensor pair, every access
// 16 bytes and all of a thread's loads independent (the per-token loop over heads of rope_rotate_bf16_kernel keeps two
// loads in flight per thread and ran at a fifth of the HBM rate).  The table rows of a token are re-read by its H
// heads out of L1.  PAIR 0: group = pairs 4g .. 4g + 3.  PAIR 1: group = pairs 8g .. 8g + 7 (two 16-byte halves).
template <int PAIR>
__global__ void __launch_bounds__(256)
rope_rotate_table_bf16_kernel(const __nv_bfloat16* __restrict__ x0, const __nv_bfloat16* __restrict__ x1,
                              __nv_bfloat16* __restrict__ y0, __nv_bfloat16* __restrict__ y1,
                              const float4* __restrict__ table, long long rows, int H, int D, float sign) {
  constexpr int NP = PAIR ? 8 : 4;
  const int half = D >> 1, groups = half / NP;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= rows * groups) return;
  const long long r = gid / groups, t = r / H;
  const int g = (int)(gid - r * groups);
  const long long base = r * (long long)D;
  const float4* trow = table + (t * half + NP * g) / 2;              // (cos, sin) x 2 per float4
  float cs[NP], sn[NP];
#pragma unroll
  for (int u = 0; u < NP; u += 2) {
    const float4 c = __ldg(trow + (u >> 1));
    cs[u] = c.x; sn[u] = c.y * sign; cs[u + 1] = c.z; sn[u + 1] = c.w * sign;
  }
  uint4 va[2], vb[2];
#pragma unroll
  for (int which = 0; which < 2; ++which) {
    const __nv_bfloat16* x = which ? x1 : x0;
    if (x == nullptr) continue;
    va[which] = *reinterpret_cast<const uint4*>(x + base + 8 * g);
    if (PAIR) vb[which] = *reinterpret_cast<const uint4*>(x + base + half + 8 * g);
  }
#pragma unroll
  for (int which = 0; which < 2; ++which) {
    __nv_bfloat16* y = which ? y1 : y0;
    if ((which ? x1 : x0) == nullptr) continue;
    uint32_t wa[4] = {va[which].x, va[which].y, va[which].z, va[which].w};
    if (PAIR == 0) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float2 ab = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wa[u]));
        const __nv_bfloat162 r2 = __floats2bfloat162_rn(ab.x * cs[u] - ab.y * sn[u], ab.x * sn[u] + ab.y * cs[u]);
        wa[u] = *reinterpret_cast<const uint32_t*>(&r2);
      }
      *reinterpret_cast<uint4*>(y + base + 8 * g) = make_uint4(wa[0], wa[1], wa[2], wa[3]);
    } else {
      uint32_t wb[4] = {vb[which].x, vb[which].y, vb[which].z, vb[which].w};
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float2 a2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wa[u]));
        const float2 b2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wb[u]));
        const __nv_bfloat162 ra = __floats2bfloat162_rn(a2.x * cs[2 * u] - b2.x * sn[2 * u], a2.y * cs[2 * u + 1] - b2.y * sn[2 * u + 1]);
        const __nv_bfloat162 rb = __floats2bfloat162_rn(a2.x * sn[2 * u] + b2.x * cs[2 * u], a2.y * sn[2 * u + 1] + b2.y * cs[2 * u + 1]);
        wa[u] = *reinterpret_cast<const uint32_t*>(&ra);
        wb[u] = *reinterpret_cast<const uint32_t*>(&rb);
      }
      *reinterpret_cast<uint4*>(y + base + 8 * g) = make_uint4(wa[0], wa[1], wa[2], wa[3]);
      *reinterpret_cast<uint4*>(y + base + half + 8 * g) = make_uint4(wb[0], wb[1], wb[2], wb[3]);
    }
  }
}

}  // namespace

// bf16 -> bf16 rotation of one or two tensors from the fp32 table of launch_rope_table_f32 (head_dim % 16 == 0).
cudaError_t launch_rope_rotate_table(const Problem& p, const void* x0, const void* x1, void* y0, void* y1,
                                     const void* table, float sign, cudaStream_t stream, int* launches) {
  if (p.D % 16 != 0) return cudaErrorInvalidValue;
  const long long rows = p.rows(), threads = rows * (p.D / 2 / (p.pairing ? 8 : 4)), grid = (threads + 255) / 256;
  if (grid <= 0 || grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin(sign > 0 ? "rope_rotate" : "rope_unrotate", stream);
  if (p.pairing)
    rope_rotate_table_bf16_kernel<1><<<(unsigned)grid, 256, 0, stream>>>((const __nv_bfloat16*)x0, (const __nv_bfloat16*)x1,
        (__nv_bfloat16*)y0, (__nv_bfloat16*)y1, (const float4*)table, rows, p.H, p.D, sign);
  else
    rope_rotate_table_bf16_kernel<0><<<(unsigned)grid, 256, 0, stream>>>((const __nv_bfloat16*)x0, (const __nv_bfloat16*)x1,
        (__nv_bfloat16*)y0, (__nv_bfloat16*)y1, (const float4*)table, rows, p.H, p.D, sign);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

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

cudaError_t launch_rope_rotate(const Problem& p, const void* x0, const void* x1, int in_dtype,
                               void* y0, void* y1, int out_dtype, const float* coords,
                               const float* freqs, float sign, cudaStream_t stream, int* launches) {
  const long long tokens = (long long)p.B * p.N;
  const long long threads = tokens * (p.D / 2);
  const int block = 256;
  const long long grid = (threads + block - 1) / block;
  if (grid <= 0 || grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin(sign > 0 ? "rope_rotate" : "rope_unrotate", stream);
  if (in_dtype == 1 && out_dtype == 1 && (p.D % 16) == 0) {       // vectorised bf16 -> bf16 path
    const int np = p.pairing ? 8 : 4;
    const long long vthreads = tokens * (p.D / 2 / np), vgrid = (vthreads + block - 1) / block;
    if (p.pairing)
      rope_rotate_bf16_kernel<1><<<(unsigned)vgrid, block, 0, stream>>>((const __nv_bfloat16*)x0, (const __nv_bfloat16*)x1,
          (__nv_bfloat16*)y0, (__nv_bfloat16*)y1, coords, freqs, tokens, p.H, p.D, p.A, sign);
    else
      rope_rotate_bf16_kernel<0><<<(unsigned)vgrid, block, 0, stream>>>((const __nv_bfloat16*)x0, (const __nv_bfloat16*)x1,
          (__nv_bfloat16*)y0, (__nv_bfloat16*)y1, coords, freqs, tokens, p.H, p.D, p.A, sign);
    prof_end(stream);
    if (launches) ++*launches;
    return cudaGetLastError();
  }
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
