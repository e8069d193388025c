// normgate.cu -- the elementwise steps around the attention of PAPER.md:390 (App. B.5): QK-RMSNorm ("RMSNorm (without
// learnable scale) to the query and key vectors before their dot product") and gated attention ("a head-specific
// sigmoid gate to the attention output"), forward and backward.  One (b, token, head) row of D channels per D / 8
// consecutive lanes, 8 channels (16 bytes of bf16) per lane, rows in memory order: every access is a coalesced
// 16-byte (bf16) or 2 x 16-byte (fp32) vector; fp32 arithmetic.  HBM-bound streaming kernels.
//   x^ = x r,  r = (mean_c x_c^2 + eps)^(-1/2)                      rmsnorm_rows
//   y  = sigmoid(g) x                                               gate_rows          (o = s a;  da = s dO)
//   dx = r (dx^ - x^ mean_c(x^_c dx^_c))                            rmsnorm_bwd_rows   (in place on dx^)
//   dg = s (1 - s) sum_c dO_c a_c = (1 - s) sum_c dO_c o_c          dgate_rows         (o the gated output)
#include "common.cuh"

namespace strata {
namespace {

template <typename T> struct Vec8;
template <> struct Vec8<float> {
  static __device__ __forceinline__ void load(const float* p, float (&x)[8]) {
    const float4 a = reinterpret_cast<const float4*>(p)[0], b = reinterpret_cast<const float4*>(p)[1];
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
  }
  static __device__ __forceinline__ void store(float* p, const float (&x)[8]) {
    reinterpret_cast<float4*>(p)[0] = make_float4(x[0], x[1], x[2], x[3]);
    reinterpret_cast<float4*>(p)[1] = make_float4(x[4], x[5], x[6], x[7]);
  }
};
template <> struct Vec8<__nv_bfloat16> {
  static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&x)[8]) {
    const uint4 w = *reinterpret_cast<const uint4*>(p);
    const uint32_t u[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) { x[2 * i] = __uint_as_float(u[i] << 16); x[2 * i + 1] = __uint_as_float(u[i] & 0xffff0000u); }
  }
  static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&x)[8]) {
    uint32_t u[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const __nv_bfloat162 h = __floats2bfloat162_rn(x[2 * i], x[2 * i + 1]);
      u[i] = *reinterpret_cast<const uint32_t*>(&h);
    }
    *reinterpret_cast<uint4*>(p) = make_uint4(u[0], u[1], u[2], u[3]);
  }
};

// sum over the D / 8 lanes of a row (lane groups are aligned: D / 8 in {4, 8, 16})
template <int D> __device__ __forceinline__ float row_sum(float x) {
#pragma unroll
  for (int m = D / 16; m > 0; m >>= 1) x += __shfl_xor_sync(0xffffffffu, x, m);
  return x;
}
__device__ __forceinline__ float sigmoidf_(float g) { return 1.f / (1.f + __expf(-g)); }

// MODE 0: y = rmsnorm(x)   MODE 1: y = sigmoid(g[row]) x   MODE 2: dx = rmsnorm backward (y holds dx^ on entry)
// MODE 3: dg[row] = (1 - sigmoid(g)) sum_c x_c y_c   (x = dO, y = gated o; nothing stored to y)
template <typename T, int D, int MODE>
__global__ void __launch_bounds__(256)
normgate_rows_kernel(const T* __restrict__ x, T* y, const float* __restrict__ g, float* __restrict__ dg, long long rows,
                     float eps) {
  constexpr int LPR = D / 8;                                   // lanes per row
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long row = gid / LPR;
  const int sub = (int)(gid % LPR);
  const bool ok = row < rows;                                  // (whole lane groups are in or out together)
  float a[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, b[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (ok) Vec8<T>::load(x + row * D + sub * 8, a);
  if (MODE == 0) {
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) ss = fmaf(a[i], a[i], ss);
    const float r = rsqrtf(row_sum<D>(ss) * (1.f / D) + eps);
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] *= r;
    if (ok) Vec8<T>::store(y + row * D + sub * 8, a);
  } else if (MODE == 1) {
    const float s = ok ? sigmoidf_(g[row]) : 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] *= s;
    if (ok) Vec8<T>::store(y + row * D + sub * 8, a);
  } else if (MODE == 2) {
    if (ok) Vec8<T>::load(y + row * D + sub * 8, b);
    float ss = 0.f, sd = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { ss = fmaf(a[i], a[i], ss); sd = fmaf(a[i], b[i], sd); }
    const float r = rsqrtf(row_sum<D>(ss) * (1.f / D) + eps);
    const float m = row_sum<D>(sd) * r * r * (1.f / D);         // mean(x^ dx^) / r = r mean(x dx^) ... times x^ = x r below
#pragma unroll
    for (int i = 0; i < 8; ++i) b[i] = r * (b[i] - a[i] * m);   // r (dx^ - x r * r mean(x dx^)) = r (dx^ - x^ mean(x^ dx^))
    if (ok) Vec8<T>::store(y + row * D + sub * 8, b);
  } else {
    if (ok) Vec8<T>::load(y + row * D + sub * 8, b);
    float sd = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) sd = fmaf(a[i], b[i], sd);
    sd = row_sum<D>(sd);
    if (ok && sub == 0) dg[row] = (1.f - sigmoidf_(g[row])) * sd;
  }
}

template <typename T, int D, int MODE>
cudaError_t launch_t(const char* name, const void* x, void* y, const float* g, float* dg, long long rows, float eps,
                     cudaStream_t st, int* launches) {
  const long long threads = rows * (D / 8), grid = (threads + 255) / 256;
  if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  prof_begin(name, st);
  normgate_rows_kernel<T, D, MODE><<<(unsigned)grid, 256, 0, st>>>((const T*)x, (T*)y, g, dg, rows, eps);
  prof_end(st);
  if (launches) ++*launches;
  return cudaGetLastError();
}
template <int MODE>
cudaError_t dispatch(const char* name, const Problem& p, const void* x, void* y, const float* g, float* dg, float eps,
                     cudaStream_t st, int* launches) {
  const long long rows = p.rows();
  if (p.dtype == 0) {
    if (p.D == 32) return launch_t<float, 32, MODE>(name, x, y, g, dg, rows, eps, st, launches);
    if (p.D == 64) return launch_t<float, 64, MODE>(name, x, y, g, dg, rows, eps, st, launches);
    if (p.D == 128) return launch_t<float, 128, MODE>(name, x, y, g, dg, rows, eps, st, launches);
  } else {
    if (p.D == 32) return launch_t<__nv_bfloat16, 32, MODE>(name, x, y, g, dg, rows, eps, st, launches);
    if (p.D == 64) return launch_t<__nv_bfloat16, 64, MODE>(name, x, y, g, dg, rows, eps, st, launches);
    if (p.D == 128) return launch_t<__nv_bfloat16, 128, MODE>(name, x, y, g, dg, rows, eps, st, launches);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_rmsnorm_rows(const Problem& p, const void* x, void* y, float eps, cudaStream_t st, int* launches) {
  return dispatch<0>("rmsnorm_rows", p, x, y, nullptr, nullptr, eps, st, launches);
}
cudaError_t launch_gate_rows(const Problem& p, const void* x, void* y, const float* gate, cudaStream_t st, int* launches) {
  return dispatch<1>("gate_rows", p, x, y, gate, nullptr, 0.f, st, launches);
}
cudaError_t launch_rmsnorm_bwd_rows(const Problem& p, const void* x, void* dx, float eps, cudaStream_t st, int* launches) {
  return dispatch<2>("rmsnorm_bwd_rows", p, x, dx, nullptr, nullptr, eps, st, launches);
}
cudaError_t launch_dgate_rows(const Problem& p, const void* d_o, const void* o, const float* gate, float* dgate,
                              cudaStream_t st, int* launches) {
  return dispatch<3>("dgate_rows", p, d_o, const_cast<void*>(o), gate, dgate, 0.f, st, launches);
}

}  // namespace strata
