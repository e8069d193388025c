// na3d_simt.cu -- fp32 CUDA-core kernels for 3D neighbourhood attention (forward and backward).
//
// This is the path for fp32 tensors (BASELINE.json config 0: 1e-4 tolerance rules out single-pass
// tensor-core arithmetic) and for every shape the tcgen05 kernels do not cover.  It is plain SIMT:
// one (b, token, head) row per group of D/32 lanes, each lane owning a 32-channel slice, the key /
// value rows of the window read straight from global memory (they hit L1/L2: neighbouring rows
// share most of their window).  Operands are pre-rotated fp32 copies of Q and K (rope.cu).
//
// Steps: A3 window, A4 logits, A5 online softmax + LSE, A6 output;
// B1 delta, B2 gradients w.r.t. rotated operands, B3 inverse neighbourhood (dK/dV are
// key-stationary: no atomics, deterministic).  B4 (rotation by -phi) is done by rope.cu afterwards.
#include "common.cuh"

namespace strata {
namespace {

constexpr int kBlock = 128;

template <int LPR> __device__ __forceinline__ float group_sum(float v) {
  if (LPR >= 2) v += __shfl_xor_sync(0xffffffffu, v, 1);
  if (LPR >= 4) v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}

__device__ __forceinline__ void load32(const float* __restrict__ p, float (&r)[32]) {
  const float4* p4 = reinterpret_cast<const float4*>(p);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    float4 t = p4[i];
    r[4 * i] = t.x; r[4 * i + 1] = t.y; r[4 * i + 2] = t.z; r[4 * i + 3] = t.w;
  }
}
__device__ __forceinline__ void load32(const __nv_bfloat16* __restrict__ p, float (&r)[32]) {
  const uint4* p4 = reinterpret_cast<const uint4*>(p);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint4 t = p4[i];
    const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      r[8 * i + 2 * u] = __uint_as_float(w[u] << 16);
      r[8 * i + 2 * u + 1] = __uint_as_float(w[u] & 0xffff0000u);
    }
  }
}
__device__ __forceinline__ void store32(float* p, const float (&r)[32]) {
  float4* p4 = reinterpret_cast<float4*>(p);
#pragma unroll
  for (int i = 0; i < 8; ++i) p4[i] = make_float4(r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]);
}
__device__ __forceinline__ void store32(__nv_bfloat16* p, const float (&r)[32]) {
  uint4* p4 = reinterpret_cast<uint4*>(p);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint32_t w[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      __nv_bfloat162 h = __floats2bfloat162_rn(r[8 * i + 2 * u], r[8 * i + 2 * u + 1]);
      w[u] = *reinterpret_cast<uint32_t*>(&h);
    }
    p4[i] = make_uint4(w[0], w[1], w[2], w[3]);
  }
}

struct RowId {
  long long row;  // flat (b, token, h)
  int b, h, l, y, x;
  long long tok;
  bool active;
};

template <int LPR>
__device__ __forceinline__ RowId decode_row(const Problem& p) {
  RowId r;
  const long long rows = p.rows();
  long long row = (long long)blockIdx.x * (kBlock / LPR) + threadIdx.x / LPR;
  r.active = row < rows;
  if (!r.active) row = rows - 1;  // keep the whole warp in the shuffles; results are discarded
  r.row = row;
  r.h = (int)(row % p.H);
  const long long bt = row / p.H;
  r.b = (int)(bt / p.N);
  r.tok = bt - (long long)r.b * p.N;
  r.x = (int)(r.tok % p.X);
  r.y = (int)((r.tok / p.X) % p.Y);
  r.l = (int)(r.tok / ((long long)p.X * p.Y));
  return r;
}

// ------------------------------------------------------------------------------------------------
// Forward: A3-A6
// ------------------------------------------------------------------------------------------------
template <int D, typename TV>
__global__ void __launch_bounds__(kBlock)
na3d_fwd_simt_kernel(const float* __restrict__ qr, const float* __restrict__ kr,
                     const TV* __restrict__ v, TV* __restrict__ o, float* __restrict__ lse, Problem p) {
  constexpr int LPR = D / 32;
  const RowId r = decode_row<LPR>(p);
  const int sub = threadIdx.x % LPR;
  float q[32], acc[32];
  load32(qr + r.row * D + sub * 32, q);
#pragma unroll
  for (int c = 0; c < 32; ++c) acc[c] = 0.f;
  const int sl = window_start(r.l, p.kL, p.L), sy = window_start(r.y, p.kY, p.Y), sx = window_start(r.x, p.kX, p.X);
  float m = -INFINITY, lsum = 0.f;
  for (int a = 0; a < p.kL; ++a)
    for (int bb = 0; bb < p.kY; ++bb)
      for (int c = 0; c < p.kX; ++c) {
        const long long j = ((long long)(sl + a) * p.Y + (sy + bb)) * p.X + (sx + c);
        const long long jrow = ((long long)r.b * p.N + j) * p.H + r.h;
        float kk[32];
        load32(kr + jrow * D + sub * 32, kk);
        float part = 0.f;
#pragma unroll
        for (int u = 0; u < 32; ++u) part = fmaf(q[u], kk[u], part);
        const float s = group_sum<LPR>(part) * p.scale;
        if (s > m) {  // online softmax: rescale the running sum and output
          const float corr = expf(m - s);
          lsum *= corr;
#pragma unroll
          for (int u = 0; u < 32; ++u) acc[u] *= corr;
          m = s;
        }
        const float pj = expf(s - m);
        lsum += pj;
        load32(v + jrow * D + sub * 32, kk);
#pragma unroll
        for (int u = 0; u < 32; ++u) acc[u] = fmaf(pj, kk[u], acc[u]);
      }
  if (!r.active) return;
  const float inv = 1.f / lsum;
#pragma unroll
  for (int u = 0; u < 32; ++u) acc[u] *= inv;
  store32(o + r.row * D + sub * 32, acc);
  if (sub == 0) lse[((long long)r.b * p.H + r.h) * p.N + r.tok] = m + logf(lsum);
}

// ------------------------------------------------------------------------------------------------
// Backward
// ------------------------------------------------------------------------------------------------
// B1: delta_i = sum_c dO_ic * O_ic, stored like lse ([B, H, N]).
template <int D, typename TV>
__global__ void __launch_bounds__(kBlock)
na3d_delta_kernel(const TV* __restrict__ o, const TV* __restrict__ d_o, float* __restrict__ delta, Problem p) {
  constexpr int LPR = D / 32;
  const RowId r = decode_row<LPR>(p);
  const int sub = threadIdx.x % LPR;
  float a[32], b[32];
  load32(o + r.row * D + sub * 32, a);
  load32(d_o + r.row * D + sub * 32, b);
  float part = 0.f;
#pragma unroll
  for (int u = 0; u < 32; ++u) part = fmaf(a[u], b[u], part);
  part = group_sum<LPR>(part);
  if (r.active && sub == 0) delta[((long long)r.b * p.H + r.h) * p.N + r.tok] = part;
}

// B2 (query-stationary half): dqrot_i = scale * sum_j dS_ij krot_j.
template <int D, typename TV>
__global__ void __launch_bounds__(kBlock)
na3d_dq_simt_kernel(const float* __restrict__ qr, const float* __restrict__ kr, const TV* __restrict__ v,
                    const TV* __restrict__ d_o, const float* __restrict__ lse,
                    const float* __restrict__ delta, float* __restrict__ dqr, Problem p) {
  constexpr int LPR = D / 32;
  const RowId r = decode_row<LPR>(p);
  const int sub = threadIdx.x % LPR;
  float q[32], g[32], acc[32];
  load32(qr + r.row * D + sub * 32, q);
  load32(d_o + r.row * D + sub * 32, g);
#pragma unroll
  for (int c = 0; c < 32; ++c) acc[c] = 0.f;
  const long long stat = ((long long)r.b * p.H + r.h) * p.N + r.tok;
  const float lse_i = lse[stat], delta_i = delta[stat];
  const int sl = window_start(r.l, p.kL, p.L), sy = window_start(r.y, p.kY, p.Y), sx = window_start(r.x, p.kX, p.X);
  for (int a = 0; a < p.kL; ++a)
    for (int bb = 0; bb < p.kY; ++bb)
      for (int c = 0; c < p.kX; ++c) {
        const long long j = ((long long)(sl + a) * p.Y + (sy + bb)) * p.X + (sx + c);
        const long long jrow = ((long long)r.b * p.N + j) * p.H + r.h;
        float kk[32], vv[32];
        load32(kr + jrow * D + sub * 32, kk);
        load32(v + jrow * D + sub * 32, vv);
        float ps = 0.f, pd = 0.f;
#pragma unroll
        for (int u = 0; u < 32; ++u) { ps = fmaf(q[u], kk[u], ps); pd = fmaf(g[u], vv[u], pd); }
        const float s = group_sum<LPR>(ps) * p.scale;
        const float dP = group_sum<LPR>(pd);
        const float dS = expf(s - lse_i) * (dP - delta_i) * p.scale;
#pragma unroll
        for (int u = 0; u < 32; ++u) acc[u] = fmaf(dS, kk[u], acc[u]);
      }
  if (r.active) store32(dqr + r.row * D + sub * 32, acc);
}

// B2 + B3 (key-stationary half): dV_j = sum_i p_ij dO_i, dkrot_j = scale * sum_i dS_ij qrot_i over
// the queries i whose window holds j.
template <int D, typename TV>
__global__ void __launch_bounds__(kBlock)
na3d_dkdv_simt_kernel(const float* __restrict__ qr, const float* __restrict__ kr, const TV* __restrict__ v,
                      const TV* __restrict__ d_o, const float* __restrict__ lse,
                      const float* __restrict__ delta, float* __restrict__ dkr, TV* __restrict__ dv, Problem p) {
  constexpr int LPR = D / 32;
  const RowId r = decode_row<LPR>(p);
  const int sub = threadIdx.x % LPR;
  float kk[32], vv[32], acck[32], accv[32];
  load32(kr + r.row * D + sub * 32, kk);
  load32(v + r.row * D + sub * 32, vv);
#pragma unroll
  for (int c = 0; c < 32; ++c) { acck[c] = 0.f; accv[c] = 0.f; }
  int l0, l1, y0, y1, x0, x1;
  inverse_window(r.l, p.kL, p.L, l0, l1);
  inverse_window(r.y, p.kY, p.Y, y0, y1);
  inverse_window(r.x, p.kX, p.X, x0, x1);
  // the loop bounds differ between the rows of a warp: iterate over the warp-wide maximum extent
  // so that the group shuffles stay converged; rows outside their own range contribute zero.
  int nl = l1 - l0 + 1, ny = y1 - y0 + 1, nx = x1 - x0 + 1;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    nl = max(nl, __shfl_xor_sync(0xffffffffu, nl, off));
    ny = max(ny, __shfl_xor_sync(0xffffffffu, ny, off));
    nx = max(nx, __shfl_xor_sync(0xffffffffu, nx, off));
  }
  for (int a = 0; a < nl; ++a)
    for (int bb = 0; bb < ny; ++bb)
      for (int c = 0; c < nx; ++c) {
        const int il = l0 + a, iy = y0 + bb, ix = x0 + c;
        bool ok = il <= l1 && iy <= y1 && ix <= x1;
        // membership re-checked from the definition (A3); also covers rows past their own range
        if (ok) {
          const int sl = window_start(il, p.kL, p.L), sy = window_start(iy, p.kY, p.Y), sx = window_start(ix, p.kX, p.X);
          ok = r.l >= sl && r.l < sl + p.kL && r.y >= sy && r.y < sy + p.kY && r.x >= sx && r.x < sx + p.kX;
        }
        const long long i = ok ? ((long long)il * p.Y + iy) * p.X + ix : r.tok;
        const long long irow = ((long long)r.b * p.N + i) * p.H + r.h;
        const long long stat = ((long long)r.b * p.H + r.h) * p.N + i;
        float qq[32], gg[32];
        load32(qr + irow * D + sub * 32, qq);
        load32(d_o + irow * D + sub * 32, gg);
        float ps = 0.f, pd = 0.f;
#pragma unroll
        for (int u = 0; u < 32; ++u) { ps = fmaf(qq[u], kk[u], ps); pd = fmaf(gg[u], vv[u], pd); }
        const float s = group_sum<LPR>(ps) * p.scale;
        const float dP = group_sum<LPR>(pd);
        const float pij = ok ? expf(s - lse[stat]) : 0.f;
        const float dS = pij * (dP - delta[stat]) * p.scale;
#pragma unroll
        for (int u = 0; u < 32; ++u) { accv[u] = fmaf(pij, gg[u], accv[u]); acck[u] = fmaf(dS, qq[u], acck[u]); }
      }
  if (!r.active) return;
  store32(dkr + r.row * D + sub * 32, acck);
  store32(dv + r.row * D + sub * 32, accv);
}

template <int D, typename TV>
cudaError_t fwd_t(const Problem& p, const float* qr, const float* kr, const void* v, void* o,
                  float* lse, cudaStream_t st, int* launches) {
  const long long rows_per_block = kBlock / (D / 32);
  const long long grid = (p.rows() + rows_per_block - 1) / rows_per_block;
  if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin("na3d_fwd_simt", st);
  na3d_fwd_simt_kernel<D, TV><<<(unsigned)grid, kBlock, 0, st>>>(qr, kr, (const TV*)v, (TV*)o, lse, p);
  prof_end(st);
  if (launches) ++*launches;
  return cudaGetLastError();
}

template <int D, typename TV>
cudaError_t bwd_t(const Problem& p, const float* qr, const float* kr, const void* v, const void* o,
                  const void* d_o, const void* d_o_main, const float* lse, float* delta, float* dqr, float* dkr, void* dv,
                  cudaStream_t st, int* launches) {
  const long long rows_per_block = kBlock / (D / 32);
  const long long grid = (p.rows() + rows_per_block - 1) / rows_per_block;
  if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin("na3d_delta", st);
  na3d_delta_kernel<D, TV><<<(unsigned)grid, kBlock, 0, st>>>((const TV*)o, (const TV*)d_o, delta, p);
  prof_end(st);
  prof_begin("na3d_dq_simt", st);
  na3d_dq_simt_kernel<D, TV><<<(unsigned)grid, kBlock, 0, st>>>(qr, kr, (const TV*)v, (const TV*)d_o_main, lse, delta, dqr, p);
  prof_end(st);
  prof_begin("na3d_dkdv_simt", st);
  na3d_dkdv_simt_kernel<D, TV><<<(unsigned)grid, kBlock, 0, st>>>(qr, kr, (const TV*)v, (const TV*)d_o_main, lse, delta, dkr, (TV*)dv, p);
  prof_end(st);
  if (launches) *launches += 3;
  return cudaGetLastError();
}

}  // namespace

#define STRATA_DISPATCH(FN, ...)                                                      \
  do {                                                                                \
    if (p.dtype == 0) {                                                               \
      if (p.D == 32) return FN<32, float>(__VA_ARGS__);                               \
      if (p.D == 64) return FN<64, float>(__VA_ARGS__);                               \
      if (p.D == 128) return FN<128, float>(__VA_ARGS__);                             \
    } else {                                                                          \
      if (p.D == 32) return FN<32, __nv_bfloat16>(__VA_ARGS__);                       \
      if (p.D == 64) return FN<64, __nv_bfloat16>(__VA_ARGS__);                       \
      if (p.D == 128) return FN<128, __nv_bfloat16>(__VA_ARGS__);                     \
    }                                                                                 \
    return cudaErrorInvalidValue;                                                     \
  } while (0)

cudaError_t launch_fwd_simt(const Problem& p, const float* qr, const float* kr, const void* v,
                            void* o, float* lse, cudaStream_t stream, int* launches) {
  STRATA_DISPATCH(fwd_t, p, qr, kr, v, o, lse, stream, launches);
}

cudaError_t launch_bwd_simt(const Problem& p, const float* qr, const float* kr, const void* v,
                            const void* o, const void* d_o, const void* d_o_main, const float* lse, float* delta,
                            float* dqr, float* dkr, void* dv, cudaStream_t stream, int* launches) {
  STRATA_DISPATCH(bwd_t, p, qr, kr, v, o, d_o, d_o_main, lse, delta, dqr, dkr, dv, stream, launches);
}

}  // namespace strata
