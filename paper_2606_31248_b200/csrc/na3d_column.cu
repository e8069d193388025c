// na3d_column.cu -- column-wise attention along the vertical ("We alternate these blocks with
// column-wise attention along the vertical dimension"; Fig. S1a): the window (k_L, k_Y, k_X) = (L, 1, 1) of the same
// operation -- every token attends the L tokens of its own (y, x) column.  bf16, head_dim 64, L <= 32.
//
// The tokens of a column share their stereographic coordinates (the coordinates are a function of
// the token's (lat, lon)), hence their rotary angles: R(phi) q . R(phi) k = q . k, StereoRoPE cancels and the path is
// plain batched L x L attention -- 4 L^2 d FLOP against 4 L d e bytes per column (12 FLOP / byte at L = 24): bound
// by HBM bandwidth, by two orders of magnitude.  So: one WARP per column, Q / K / V rows global -> shared memory with
// cp.async (coalesced 128-byte rows, no register staging), S = Q K^T and O = P V with mma.sync m16n8k16 (a 32 x 32
// problem is far below one tcgen05 tile; the tensor work is ~15 % of the HBM time either way), softmax on the
// accumulator fragments, O staged through shared memory for 16-byte stores.  Several warps per SM hide each other's
// load latency.  If the coordinates of a column DO depend on the level (not the paper's case), the kernel says so in
// the fix-up header and na3d_fix_rows (na3d_fwd_plane.cu) recomputes every row with each token's own angles.
#include "tc_common.cuh"

namespace strata {
namespace {

using namespace tc;

constexpr int kColWarps = 4;                  // warps (= columns in flight) per CTA
constexpr int kColSmemPerWarp = 3 * 32 * 128; // Q | K | V, 32 rows x 128 bytes each

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  const int n = valid ? 16 : 0;               // src-size 0: the 16 bytes are zero-filled
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// 16-byte chunk c of row r of a 32 x 64 bf16 tile (128-byte rows, chunks XOR-swizzled by the row)
__device__ __forceinline__ uint32_t tile_off(int r, int c) { return (uint32_t)(r * 128 + ((c ^ (r & 7)) << 4)); }

__global__ void __launch_bounds__(kColWarps * 32)
na3d_column_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k,
                   const __nv_bfloat16* __restrict__ v, const float* __restrict__ coords,
                   __nv_bfloat16* __restrict__ o, float* __restrict__ lse, unsigned long long* fix, Problem p,
                   long long ncols) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long col = (long long)blockIdx.x * kColWarps + warp;
  if (col >= ncols) return;
  // column = (b, y, x, h), head fastest (the heads of a token are contiguous in memory)
  const int h = (int)(col % p.H);
  const long long tok_yx = (col / p.H) % ((long long)p.Y * p.X);
  const long long b = col / p.H / ((long long)p.Y * p.X);
  const long long lstride = (long long)p.Y * p.X * p.H * 64;                 // elements between levels
  const long long base = ((b * p.N + tok_yx) * p.H + h) * 64;               // element offset of level 0
  const uint32_t sq = smem_addr(smem) + warp * kColSmemPerWarp, sk = sq + 32 * 128, sv = sk + 32 * 128;

  // ---- Q, K, V rows -> shared memory: chunk id = lane + 32 i: row id >> 3 (8 lanes per 128-byte row)
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int id = lane + 32 * i, r = id >> 3, c = id & 7;
    const bool ok = r < p.L;
    const long long off = base + (ok ? r : 0) * lstride + c * 8;
    cp_async16(sq + tile_off(r, c), q + off, ok);
    cp_async16(sk + tile_off(r, c), k + off, ok);
    cp_async16(sv + tile_off(r, c), v + off, ok);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  // ---- the rotation cancels only if the column's coordinates are the same on every level
  if (p.A > 0 && lane < p.L) {
    const float* c0 = coords + (b * p.N + tok_yx) * p.A;
    const float* cl = c0 + (long long)lane * p.Y * p.X * p.A;
    bool diff = false;
    for (int a = 0; a < p.A; ++a) diff |= __float_as_uint(cl[a]) != __float_as_uint(c0[a]);
    if (diff) fix[1] = 1ull;
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncwarp();

  const int g = lane >> 2, t = lane & 3;
  // ---- S = Q K^T: 2 m-tiles x 4 n-tiles, K = 64 in 4 steps
  float s[2][4][4];
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int nt = 0; nt < 4; ++nt)
#pragma unroll
      for (int u = 0; u < 4; ++u) s[mt][nt][u] = 0.f;
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
    uint32_t a[2][4], bb[2][4];
    // A fragments: matrix m of ldmatrix.x4 = rows (m & 1) * 8 .., k chunk 2 ks + (m >> 1)
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
      ldsm_x4(sq + tile_off(16 * mt + (lane >> 3 & 1) * 8 + (lane & 7), 2 * ks + (lane >> 4)), a[mt]);
    // B fragments (K rows are the n index): matrix m = keys (m >> 1) * 8 .., k chunk 2 ks + (m & 1): two n-tiles per load
#pragma unroll
    for (int np = 0; np < 2; ++np)
      ldsm_x4(sk + tile_off(16 * np + (lane >> 4) * 8 + (lane & 7), 2 * ks + (lane >> 3 & 1)), bb[np]);
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) mma_bf16(s[mt][nt], a[mt], bb[nt >> 1][2 * (nt & 1)], bb[nt >> 1][2 * (nt & 1) + 1]);
  }
  // ---- softmax over the L keys of the column (A5); rows g and g + 8 of each m-tile, 8 of their columns in this lane
  const float cs = p.scale * 1.4426950408889634f;
  float inv[2][2], lse_row[2][2];
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      float mx = -INFINITY;
#pragma unroll
      for (int nt = 0; nt < 4; ++nt)
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int key = 8 * nt + 2 * t + u;
          float x = s[mt][nt][2 * hf + u] * cs;
          x = key < p.L ? x : -INFINITY;
          s[mt][nt][2 * hf + u] = x;
          mx = fmaxf(mx, x);
        }
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
      float sum = 0.f;
#pragma unroll
      for (int nt = 0; nt < 4; ++nt)
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const float e = exp2f(s[mt][nt][2 * hf + u] - mx);
          s[mt][nt][2 * hf + u] = e;
          sum += e;
        }
      sum += __shfl_xor_sync(0xffffffffu, sum, 1);
      sum += __shfl_xor_sync(0xffffffffu, sum, 2);
      inv[mt][hf] = 1.f / sum;
      lse_row[mt][hf] = (mx + log2f(sum)) * 0.69314718055994531f;
    }
  // ---- O = P V: P (bf16) straight from the accumulator fragments; V fragments with ldmatrix.trans
  float acc[2][8][4];
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int nt = 0; nt < 8; ++nt)
#pragma unroll
      for (int u = 0; u < 4; ++u) acc[mt][nt][u] = 0.f;
#pragma unroll
  for (int ks = 0; ks < 2; ++ks) {
    uint32_t a[2][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
      a[mt][0] = pack_bf16(s[mt][2 * ks][0], s[mt][2 * ks][1]);
      a[mt][1] = pack_bf16(s[mt][2 * ks][2], s[mt][2 * ks][3]);
      a[mt][2] = pack_bf16(s[mt][2 * ks + 1][0], s[mt][2 * ks + 1][1]);
      a[mt][3] = pack_bf16(s[mt][2 * ks + 1][2], s[mt][2 * ks + 1][3]);
    }
#pragma unroll
    for (int np = 0; np < 4; ++np) {
      // matrix m of the transposed load = keys 16 ks + (m & 1) * 8 .., channel chunk 2 np + (m >> 1)
      uint32_t bb[4];
      ldsm_x4_t(sv + tile_off(16 * ks + (lane >> 3 & 1) * 8 + (lane & 7), 2 * np + (lane >> 4)), bb);
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        mma_bf16(acc[mt][2 * np], a[mt], bb[0], bb[1]);
        mma_bf16(acc[mt][2 * np + 1], a[mt], bb[2], bb[3]);
      }
    }
  }
  // ---- O / l -> bf16 -> shared memory (over Q) -> 16-byte stores; LSE
  __syncwarp();
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      const int r = 16 * mt + 8 * hf + g;
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        const uint32_t w = pack_bf16(acc[mt][nt][2 * hf] * inv[mt][hf], acc[mt][nt][2 * hf + 1] * inv[mt][hf]);
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(sq + tile_off(r, nt) + 4 * t), "r"(w) : "memory");
      }
      if (t == 0 && r < p.L) lse[((b * p.H + h) * p.L + r) * ((long long)p.Y * p.X) + tok_yx] = lse_row[mt][hf];
    }
  __syncwarp();
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int id = lane + 32 * i, r = id >> 3, c = id & 7;
    if (r < p.L) {
      uint4 w;
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "r"(sq + tile_off(r, c)) : "memory");
      *reinterpret_cast<uint4*>(o + base + r * lstride + c * 8) = w;
    }
  }
}

DeviceState g_states[64];
std::mutex g_mu;

}  // namespace

bool column_fwd_supported(const Problem& p) {
  return p.dtype == 1 && p.D == 64 && p.kL == p.L && p.kY == 1 && p.kX == 1 && p.L <= 32 && p.A <= 2;
}

cudaError_t launch_fwd_column(const Problem& p, const void* q, const void* k, const void* v, const float* coords,
                              const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches) {
  if (!column_fwd_supported(p)) return cudaErrorNotSupported;
  const long long ncols = (long long)p.B * p.Y * p.X * p.H;
  const long long grid = (ncols + kColWarps - 1) / kColWarps;
  if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  DeviceState* ds = device_state(g_states, g_mu);
  if (!ds) return cudaErrorInvalidDevice;
  constexpr int smem = kColWarps * kColSmemPerWarp;
  cudaError_t e = ensure_smem_attr(ds, g_mu, 0, na3d_column_kernel, smem);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(fix, 0, 16, stream);
  if (e != cudaSuccess) return e;
  prof_begin("na3d_column", stream);
  na3d_column_kernel<<<(unsigned)grid, kColWarps * 32, smem, stream>>>((const __nv_bfloat16*)q, (const __nv_bfloat16*)k,
                                                                     (const __nv_bfloat16*)v, coords, (__nv_bfloat16*)o, lse,
                                                                     reinterpret_cast<unsigned long long*>(fix), p, ncols);
  prof_end(stream);
  if (launches) ++*launches;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_fix_rows(p, q, k, v, coords, freqs, o, lse, fix, stream, launches);
}

}  // namespace strata
