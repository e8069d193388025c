// na3d_bwd_tc.cu -- entry of the tcgen05 backward (bf16, head_dim 64): step B1 of DESIGN.md as a small streaming
// kernel, then the two persistent kernels of na3d_bwd_tc2.cu (B2-B4).  PAPER.md gives no backward; BASELINE.json
// config 4 and SURVEY.md section 8(a) rows B1-B4 define it:
//   B1  D_i    = sum_c dO_ic O_ic                       (bwd_stat_kernel, stored with lse * log2 e, and a second
//                                                         time as the bias rows of the dK/dV kernel)
#include "tc_common.cuh"
#include "bwd_common.cuh"

namespace strata {
namespace {

using namespace tc;

// B1 (+ the row statistics in the form the kernels of na3d_bwd_tc2.cu consume): stat[b][h][t] = (lse * log2 e, D),
// D = sum_c dO_c O_c.  8 lanes per (b, token, h) row of 64 channels, rows in memory order.
// bias[b][token][h] = 8 bf16 {a1, a2, a3, d1, d2, d3, 0, 0}: a1 + a2 + a3 = -lse / scale and d1 + d2 + d3 = -D to 24
// bits each.  The dK/dV kernel adds them to S' = q.k and dP' = dO.v on the tensor cores (na3d_bwd_tc2.cu, MODE 1).
// A block takes kStatTokens consecutive tokens of one sample with all their heads: the row sums come in (token, head)
// order like O and dO, lse and stat are [B, H, N], so the block transposes its 32 x H values through shared memory and
// every global access is a full line (one thread per row writing stat directly touched a 32-byte sector per 8 bytes).
constexpr int kStatTokens = 32;
__global__ void __launch_bounds__(256)
bwd_stat_kernel(const __nv_bfloat16* __restrict__ o, const __nv_bfloat16* __restrict__ d_o,
                const float* __restrict__ lse, float2* __restrict__ stat, uint4* __restrict__ bias, float inv_scale,
                long long N, int H) {
  extern __shared__ float sm[];                      // part | lse, both [token][H + 1]
  const int HP = H + 1;
  float* sm_part = sm;
  float* sm_lse = sm + kStatTokens * HP;
  const long long nblk = (N + kStatTokens - 1) / kStatTokens;
  const long long b = blockIdx.x / nblk, t0 = (blockIdx.x % nblk) * kStatTokens;
  const int nt = (int)(N - t0 < kStatTokens ? N - t0 : kStatTokens), nrows = nt * H;
  const long long r0 = (b * N + t0) * H;
  const int sub = threadIdx.x & 7;
#pragma unroll 4
  for (int i0 = 0; i0 < nrows; i0 += 32) {
    const int i = i0 + (threadIdx.x >> 3);
    float part = 0.f;
    if (i < nrows) {
      const uint4 a = reinterpret_cast<const uint4*>(o + (r0 + i) * 64)[sub], g = reinterpret_cast<const uint4*>(d_o + (r0 + i) * 64)[sub];
      const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, gw[4] = {g.x, g.y, g.z, g.w};
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float2 fa = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&aw[u]));
        const float2 fg = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&gw[u]));
        part = fmaf(fa.x, fg.x, fmaf(fa.y, fg.y, part));
      }
    }
    part += __shfl_xor_sync(0xffffffffu, part, 1);
    part += __shfl_xor_sync(0xffffffffu, part, 2);
    part += __shfl_xor_sync(0xffffffffu, part, 4);
    if (i < nrows && sub == 0) sm_part[(i / H) * HP + i % H] = part;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nrows; i += 256) {   // (head, token) order: lse and stat rows
    const int h = i / nt, tt = i - h * nt;
    const long long idx = (b * H + h) * N + t0 + tt;
    const float l = lse[idx];
    stat[idx] = make_float2(l * 1.4426950408889634f, sm_part[tt * HP + h]);
    sm_lse[tt * HP + h] = l;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nrows; i += 256) {   // (token, head) order: bias rows
    const int tt = i / H, h = i - tt * H;
    auto split3 = [](float v, uint32_t& h1, uint32_t& h2, uint32_t& h3) {
      const __nv_bfloat16 b1 = __float2bfloat16_rn(v);
      const float r1 = v - __bfloat162float(b1);
      const __nv_bfloat16 b2 = __float2bfloat16_rn(r1);
      const __nv_bfloat16 b3 = __float2bfloat16_rn(r1 - __bfloat162float(b2));
      h1 = __bfloat16_as_ushort(b1); h2 = __bfloat16_as_ushort(b2); h3 = __bfloat16_as_ushort(b3);
    };
    uint32_t a1, a2, a3, d1, d2, d3;
    split3(-sm_lse[tt * HP + h] * inv_scale, a1, a2, a3);
    split3(-sm_part[tt * HP + h], d1, d2, d3);
    bias[r0 + i] = make_uint4(a1 | (a2 << 16), a3 | (d1 << 16), d2 | (d3 << 16), 0u);
  }
}

}  // namespace
cudaError_t launch_bwd_tc2_main(const Problem& p, const void* qr, const void* kr, const void* v, const void* d_o,
                                const void* stat, const void* bias, const void* rtab, void* dq, void* dk, void* dv,
                                cudaStream_t stream, int* launches);
// Shapes the tensor-core backward covers: bf16, head_dim 64, the windows below.
#define STRATA_BWD_CONFIGS(X) \
  X(3, 7, 7)                  \
  X(3, 5, 5)                  \
  X(3, 3, 3)                  \
  X(9, 9, 9)

bool tc_bwd_supported(const Problem& p) {
  if (p.dtype != 1 || p.D != 64) return false;
  // bwd_stat_kernel transposes 2 x kStatTokens x (H + 1) floats through (non-opt-in) shared memory: beyond 191 heads
  // AUTO takes the CUDA-core backward instead of failing at the launch
  if ((size_t)2 * kStatTokens * (p.H + 1) * sizeof(float) > 48 * 1024) return false;
#define X(KL_, KY_, KX_) \
  if (p.kL == KL_ && p.kY == KY_ && p.kX == KX_) return true;
  STRATA_BWD_CONFIGS(X)
#undef X
  return false;
}

// B1 (+ lse in the exp2 domain) -> stat, then the two persistent kernels of na3d_bwd_tc2.cu.
cudaError_t launch_bwd_tc(const Problem& p, const void* qr, const void* kr, const void* v, const void* o,
                          const void* d_o, const void* d_o_main, const float* lse, void* stat, const void* rtab, void* dq,
                          void* dk, void* dv, cudaStream_t stream, int* launches) {
  if (!tc_bwd_supported(p)) return cudaErrorNotSupported;
  const long long rows = p.rows(), sgrid = (long long)p.B * ((p.N + kStatTokens - 1) / kStatTokens);
  const size_t ssmem = (size_t)2 * kStatTokens * (p.H + 1) * sizeof(float);
  if (sgrid > 0x7fffffffLL || ssmem > 48 * 1024) return cudaErrorInvalidValue;
  prof_begin("na3d_bwd_stat", stream);
  // `stat` holds both arrays: float2 per row, then (256-byte aligned) the 16-byte bias rows
  uint4* bias = reinterpret_cast<uint4*>(reinterpret_cast<char*>(stat) + (((size_t)rows * 8 + 255) & ~(size_t)255));
  bwd_stat_kernel<<<(unsigned)sgrid, 256, ssmem, stream>>>((const __nv_bfloat16*)o, (const __nv_bfloat16*)d_o, lse, (float2*)stat, bias,
                                                           1.f / p.scale, p.N, p.H);
  prof_end(stream);
  if (launches) *launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_bwd_tc2_main(p, qr, kr, v, d_o_main, (float2*)stat, bias, rtab, dq, dk, dv, stream, launches);
}

}  // namespace strata
