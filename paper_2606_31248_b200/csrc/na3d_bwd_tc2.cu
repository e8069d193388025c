// na3d_bwd_tc2.cu -- tcgen05 / TMEM / TMA backward kernels for 3D neighbourhood attention (sm_100a), bf16, head_dim 64.
//
// Steps B2-B4 of DESIGN.md on pre-rotated bf16 operands (rope.cu rotates Q, K before; the transpose rotation B4 of
// dQrot, dKrot is fused into the epilogues, from an fp32 cos / sin table; B1 is bwd_stat_kernel in na3d_bwd_tc.cu).
// PAPER.md gives no backward; BASELINE.json config 4 and SURVEY.md section 8(a) rows B1-B4 define it:
//   B2  p_ij   = exp(scale qrot_i . krot_j - lse_i),  dP_ij = dO_i . v_j,  dS_ij = p_ij (dP_ij - D_i)
//       dqrot_i = scale sum_j dS_ij krot_j;  dkrot_j = scale sum_i dS_ij qrot_i;  dV_j = sum_i p_ij dO_i
// ONE kernel template, two modes, both "a stationary tile of 128 rows against streamed chunks":
//   MODE 0 (dQ, query-stationary)  rows = queries: A1 = Qrot, A2 = dO tile; chunks = the keys of the
//       tile's window halo: B1 = Krot, B2 = V.            acc1 = dQrot = sum dS  B1
//   MODE 1 (dK/dV, key-stationary) rows = keys:    A1 = Krot, A2 = V tile;  chunks = the queries of
//       the tile's INVERSE halo (B3: the queries whose inward-clamped window holds a key of the tile --
//       not symmetric at the borders): B1 = Qrot, B2 = dO.  acc1 = dKrot = sum dS^T B1,
//       acc2 = dV = sum P^T B2.  The statistics (lse, D) belong to the chunk's COLUMNS here, and a per-column
//       bias is a rank-one term, so the tensor cores add it: S' and dP' get a fifth K step whose A operand is a
//       constant tile (ones in three channels) and whose B operand holds, for column j, -lse_j / scale resp. -D_j
//       split into three bf16 terms (24 significant bits, the sum is exact in the fp32 accumulator).  bwd_stat_kernel
//       writes those 16-byte bias rows per (token, head); one more TMA box per chunk brings them in, unswizzled,
//       which is the K-major core-matrix layout of an UMMA operand as it stands (8 rows x 16 bytes contiguous).
//       (Reading the statistics from shared memory in the elementwise loop cost 28 loads per chunk and thread, each
//       waiting behind the tensor cores' own operand reads; building the bias rows in the producer warp made that
//       warp the bottleneck at ~190 dependent instructions per chunk: profiles/r2_bwd_cfg4.md.)
// Per chunk (CY rows x HX columns of one level plane = N <= 64 columns):
//   S' = A1 B1^T and dP' = A2 B2^T on the tensor cores (M = 128, K = 64) -> TMEM;
//   one row per thread: p = 2^(S' scale log2e - lse log2e) under the window mask, dS = p (dP' - D),
//   written back to TMEM as bf16 over the buffers they came from;
//   acc1 += dS B1 (and acc2 += P B2) with the bf16 matrix as the TMEM A operand and the SAME shared
//   memory chunk re-read as an MN-major B operand.
// No atomics: every output row is owned by exactly one thread; deterministic.
//
// Schedule: ONE persistent CTA per SM runs the chain S'/dP' MMAs -> elementwise pass -> gradient MMAs as a pipeline
// (a one-tile-per-CTA version of round 1 cost ~3100 cycles per chunk in a strictly serial chain that two co-resident
// CTAs only half filled, profiles/r1_bwd_cfg4_and_tile_cfg2.md):
//   * S' / dP' have three buffers in TMEM and TWO elementwise warpgroups split every chunk by columns (the
//     elementwise pass is the longest stage of the ring S' MMA -> elementwise -> gradient MMA: halving its latency
//     shortens the ring; taking alternate chunks instead gave the same throughput bound at twice the latency),
//     so the MMAs of chunks c + 1, c + 2 run under the elementwise pass of chunk c;
//   * the stationary operand tiles are double buffered in shared memory (and the dQ accumulator in TMEM) and the
//     chunk stream runs on across tiles, so the epilogue of tile t (TMEM -> un-rotate -> HBM) and the operand loads
//     of tile t + 1 overlap the MMAs of tile t + 1.
// TMEM (512 columns): accumulators [0, 128) -- MODE 0: acc1 double buffered by tile parity, MODE 1: {acc1, acc2}
// once -- | SD[buf] = {S' -> P, dP' -> dS} at 128 + 128 * buf, buf < 3 (chunk index mod 3).
// Warps (512 threads): 0 TMA producer, 1 S'/dP' MMA issuer + TMEM owner, 2 gradient-MMA issuer, 3 idle,
// 4-7 elementwise group 0, 8-11 group 1 (group g takes columns [32 g, 32 g + 32) of every chunk), 12-15 epilogue
// (acc1 -> dQ or dK, un-rotated; acc2 -> dV in MODE 1).  The epilogue has warps of its own because its table loads
// and stores take about as long as half a tile's elementwise work: done by an elementwise group, it held back that
// group's chunks of the next tile, and with them the MMAs (profiles/r2_bwd_cfg4.md).
#include <type_traits>

#include "tc_common.cuh"
#include "bwd_common.cuh"

namespace strata {
namespace {

using namespace tc;

template <int KL_, int KY_, int KX_>
struct Bwd2Cfg {
  static constexpr int D = 64, KL = KL_, KY = KY_, KX = KX_;
  static constexpr int TL = 2, TY = 8, TX = 8, M = 128;            // stationary tile (tokens)
  static constexpr int HX = TX + KX - 1;                           // chunk width (columns of one row)
  static constexpr int CY = 4;                                     // chunk rows
  static constexpr int NCOL = CY * HX;                             // real columns of a chunk
  static constexpr int N = (NCOL + 15) / 16 * 16;                  // UMMA N (pad columns are masked)
  static constexpr int TILE_BYTES = M * 128, CHUNK_BYTES = N * 128;
  static constexpr int STAGE_BYTES = 2 * CHUNK_BYTES;              // B1 | B2
  static constexpr int NSTAGE = 4;
  static constexpr int BIAS_BYTES = N * 16;                        // bias rows of a chunk: [N columns][8 bf16]
  static constexpr int XTRA_BYTES = TILE_BYTES + NSTAGE * 1024 + 1024;   // MODE 1: ones tile | per-stage bias rows | zeros
  static_assert(BIAS_BYTES <= 1024, "bias rows of a chunk");
  static constexpr int NBUF = 3;                                   // S'/dP' buffers in TMEM
  static constexpr int TMEM_ACC = 0, TMEM_SD = 128, TMEM_COLS = 512;
  static constexpr int NBARS = 4 + 2 * NSTAGE + 3 * NBUF + 4;
  static constexpr int SMEM_BYTES = 1024 + 4 * TILE_BYTES + NSTAGE * STAGE_BYTES + XTRA_BYTES + 8 * NBARS + 16 + 128;
  static_assert(KL % 2 == 1 && KY % 2 == 1 && KX % 2 == 1, "odd windows only");
  static_assert(N <= 64 && HX <= 16 && HX % 2 == 0, "a chunk must fit 64 TMEM columns; column pairs share a row");
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

constexpr int kBwd2Threads = 512;

// Geometry of one stationary tile and of its streamed box.
struct Tile2 {
  int b, h, x0, y0, l0;
  int bx0, by0, bl0, bl1, ncx, ncy, nchunks;
};

// ------------------------------------------------------------------------------------------------
// Kernel
// ------------------------------------------------------------------------------------------------
template <class C, int MODE>
__global__ void __launch_bounds__(kBwd2Threads, 1)
na3d_bwd_tc2_kernel(const __grid_constant__ CUtensorMap tm_a1, const __grid_constant__ CUtensorMap tm_a2,
                    const __grid_constant__ CUtensorMap tm_b1, const __grid_constant__ CUtensorMap tm_b2,
                    const __grid_constant__ CUtensorMap tm_bias, const float2* __restrict__ stat, const float4* __restrict__ rtab,
                    __nv_bfloat16* __restrict__ out1, __nv_bfloat16* __restrict__ out2, const BwdParams p,
                    const int ntiles) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  auto a_smem = [&](int par, int which) { return base + (uint32_t)(2 * par + which) * C::TILE_BYTES; };
  const uint32_t st_smem = base + 4 * C::TILE_BYTES;                       // stages
  const uint32_t xa_smem = st_smem + C::NSTAGE * C::STAGE_BYTES;           // MODE 1: A operand of the bias K step
  auto xb_smem = [&](int s) { return xa_smem + C::TILE_BYTES + (uint32_t)s * 1024; };             // its B operand
  const uint32_t xz_smem = xb_smem(C::NSTAGE);                             // zeros: channels 8-15 of every bias row
  const uint32_t bars = xa_smem + C::XTRA_BYTES;
  auto bar_afull = [&](int par) { return bars + 8u * par; };               // TMA -> MMA: operand tiles of a tile
  auto bar_aempty = [&](int par) { return bars + 8u * (2 + par); };        // last S'/dP' MMA of the tile -> TMA
  auto bar_full = [&](int s) { return bars + 8u * (4 + s); };
  auto bar_empty = [&](int s) { return bars + 8u * (4 + C::NSTAGE + s); };
  auto bar_sfull = [&](int b) { return bars + 8u * (4 + 2 * C::NSTAGE + b); };                  // MMA -> elementwise, buffer b
  auto bar_pfull = [&](int b) { return bars + 8u * (4 + 2 * C::NSTAGE + C::NBUF + b); };        // elementwise -> MMA (4 warps)
  auto bar_sdfree = [&](int b) { return bars + 8u * (4 + 2 * C::NSTAGE + 2 * C::NBUF + b); };   // gradient MMAs have read buffer b
  auto bar_accdone = [&](int a) { return bars + 8u * (4 + 2 * C::NSTAGE + 3 * C::NBUF + a); };  // last gradient MMA of the tile
  auto bar_accfree = [&](int a) { return bars + 8u * (6 + 2 * C::NSTAGE + 3 * C::NBUF + a); };  // epilogue has read acc[a]
  // accumulators: MODE 0 needs acc1 only and double buffers it by tile parity; MODE 1 has {acc1, acc2} once
  constexpr int NACC = MODE == 0 ? 2 : 1, ACC_STRIDE = 64;
  const uint32_t tmem_slot = bars + 8u * C::NBARS;
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  auto tile_of = [&](int t) {
    Tile2 T;
    int bid = t;
    const int tx = bid % p.ntx; bid /= p.ntx;
    const int ty = bid % p.nty; bid /= p.nty;
    const int tl = bid % p.ntl; bid /= p.ntl;
    T.h = bid % p.H;
    T.b = bid / p.H;
    T.x0 = tx * C::TX; T.y0 = ty * C::TY; T.l0 = tl * C::TL;
    const int xl = min(T.x0 + C::TX, p.X) - 1, yl = min(T.y0 + C::TY, p.Y) - 1, ll = min(T.l0 + C::TL, p.L) - 1;
    int bx1, by1, t0, t1;
    row_interval<MODE>(T.x0, C::KX, p.X, T.bx0, t1); row_interval<MODE>(xl, C::KX, p.X, t0, bx1);
    row_interval<MODE>(T.y0, C::KY, p.Y, T.by0, t1); row_interval<MODE>(yl, C::KY, p.Y, t0, by1);
    row_interval<MODE>(T.l0, C::KL, p.L, T.bl0, t1); row_interval<MODE>(ll, C::KL, p.L, t0, T.bl1);
    T.ncx = (bx1 - T.bx0 + C::HX - 1) / C::HX;
    T.ncy = (by1 - T.by0 + C::CY - 1) / C::CY;
    T.nchunks = (T.bl1 - T.bl0) * T.ncy * T.ncx;
    return T;
  };

  // ---- one-time setup
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_a1); tma_prefetch_desc(&tm_a2); tma_prefetch_desc(&tm_b1); tma_prefetch_desc(&tm_b2);
    if (MODE == 1) tma_prefetch_desc(&tm_bias);
    for (int i = 0; i < 2; ++i) {
      mbar_init(bar_afull(i), 1); mbar_init(bar_aempty(i), 1);
      mbar_init(bar_accdone(i), 1); mbar_init(bar_accfree(i), 4);
    }
    for (int i = 0; i < C::NBUF; ++i) { mbar_init(bar_sfull(i), 1); mbar_init(bar_pfull(i), 8); mbar_init(bar_sdfree(i), 1); }
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(bar_full(s), 1); mbar_init(bar_empty(s), 1); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, C::TMEM_COLS);
  // chunk rows the TMA box never writes (pad columns of the UMMA N) must hold finite numbers
  if (C::N > C::NCOL) {
    for (int s = 0; s < C::NSTAGE; ++s)
      for (int u = threadIdx.x; u < 2 * (C::N - C::NCOL) * 8; u += kBwd2Threads) {
        const int which = u / ((C::N - C::NCOL) * 8), off = u % ((C::N - C::NCOL) * 8);
        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(st_smem + s * C::STAGE_BYTES + which * C::CHUNK_BYTES +
                                                                     C::NCOL * 128 + off * 16), "r"(0u) : "memory");
      }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (MODE == 1) {
    // bias K step, A operand (128-byte swizzled rows like the other tiles): row r has ones in channels 0-2 (K step 0:
    // picks the lse terms of a bias row) and in channels 16 + 3..5 (K step 1: picks the D terms); everything else,
    // the zeros block and the pad rows of the bias stages start as zeros
    for (int u = threadIdx.x; u < C::XTRA_BYTES / 16; u += kBwd2Threads) {
      const int r = u >> 3, ch = (u & 7) ^ (r & 7);
      const bool tile = u < C::TILE_BYTES / 16;
      uint32_t w0 = 0u, w1 = 0u, w2 = 0u;
      if (tile && ch == 0) { w0 = 0x3F803F80u; w1 = 0x00003F80u; }
      if (tile && ch == 2) { w1 = 0x3F800000u; w2 = 0x3F803F80u; }
      asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(xa_smem + u * 16), "r"(w0), "r"(w1), "r"(w2), "r"(0u) : "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot_ptr;
  // registers: the kernel is compiled for 128 per thread (512 threads); the control warpgroup (72) hands the rest to
  // the elementwise warpgroups (144) and the epilogue warpgroup (152)
  // (each setmaxnreg sits at the head of its own branch: ptxas budgets the code a setmaxnreg dominates)

  if (warp < 4) {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
  if (warp == 0) {
    // =========================== TMA producer ===========================
    // The control warps walk their loops with all 32 lanes in uniform control flow and elect one lane for the TMA / MMA /
    // commit instructions only: inside `if (lane == 0)` the compiler cannot prove any operand warp-uniform and wraps
    // every tcgen05.mma in a ~10-instruction election / uniformisation sequence (~80 cycles per MMA of 32-48 tensor
    // cycles: the S'/dP' issuer never waited on a barrier, it was the bottleneck).
    {
      int Tn = 0, Cn = 0;
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++Tn) {
        const Tile2 T = tile_of(t);
        const int par = Tn & 1, bl = T.b * p.L;
        mbar_wait_bounded(bar_aempty(par), ((uint32_t)(Tn >> 1) & 1u) ^ 1u);
        if (elect_one()) {
          mbar_expect_tx(bar_afull(par), 2 * C::TILE_BYTES);
          tma_load_5d(a_smem(par, 0), &tm_a1, bar_afull(par), 0, T.h, T.x0, T.y0, bl + T.l0);
          tma_load_5d(a_smem(par, 1), &tm_a2, bar_afull(par), 0, T.h, T.x0, T.y0, bl + T.l0);
        }
        __syncwarp();
        for (int pl = T.bl0; pl < T.bl1; ++pl)
          for (int cy = 0; cy < T.ncy; ++cy)
            for (int cx = 0; cx < T.ncx; ++cx, ++Cn) {
              const int s = Cn % C::NSTAGE;
              const uint32_t ph = (uint32_t)(Cn / C::NSTAGE) & 1u;
              const uint32_t sb = st_smem + s * C::STAGE_BYTES;
              const int gx = T.bx0 + cx * C::HX, gy = T.by0 + cy * C::CY;
              mbar_wait_bounded(bar_empty(s), ph ^ 1u);
              if (elect_one()) {
                mbar_expect_tx(bar_full(s), 2 * C::NCOL * 128 + (MODE == 1 ? C::NCOL * 16 : 0));
                tma_load_5d(sb, &tm_b1, bar_full(s), 0, T.h, gx, gy, bl + pl);
                tma_load_5d(sb + C::CHUNK_BYTES, &tm_b2, bar_full(s), 0, T.h, gx, gy, bl + pl);
                if (MODE == 1) tma_load_5d(xb_smem(s), &tm_bias, bar_full(s), 0, T.h, gx, gy, bl + pl);
              }
              __syncwarp();
            }
      }
    }
  } else if (warp == 1) {
    // =========================== S'/dP' issuer ===========================
    {
      constexpr uint32_t idesc_s = instr_desc(C::M, C::N, false);
      constexpr uint32_t kDescHi = 0x40004040u;            // 8-row groups 1024 bytes apart, version 1, 128-byte swizzle
      auto dlo = [](uint32_t addr) { return ((addr >> 4) & 0x3FFFu) | (1u << 16); };
      auto dsc = [](uint32_t lo) { return ((uint64_t)kDescHi << 32) | lo; };
      const uint32_t lxa = dlo(xa_smem);
      int Tn = 0, Cn = 0;
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++Tn) {
        const int n = tile_of(t).nchunks;
        const int par = Tn & 1;
        mbar_wait<false>(bar_afull(par), (uint32_t)(Tn >> 1) & 1u);
        const uint32_t la1 = dlo(a_smem(par, 0)), la2 = dlo(a_smem(par, 1));
        for (int c = 0; c < n; ++c, ++Cn) {
          const int s = Cn % C::NSTAGE, buf = Cn % C::NBUF;
          mbar_wait<false>(bar_full(s), (uint32_t)(Cn / C::NSTAGE) & 1u);
          mbar_wait<false>(bar_sdfree(buf), ((uint32_t)(Cn / C::NBUF) & 1u) ^ 1u);    // gradient MMAs of chunk Cn - NBUF are done
          tc_fence_after();
          const uint32_t sb = st_smem + s * C::STAGE_BYTES, sd = tmem + C::TMEM_SD + 128 * buf;
          const uint32_t lb1 = dlo(sb), lb2 = dlo(sb + C::CHUNK_BYTES);
          // bias rows: unswizzled K-major operand -- 8 columns x 16 bytes per core matrix, the next 8 columns 128 bytes on
          // (stride offset), channels 8-15 in the zeros block (leading offset)
          const uint64_t dxb = (uint64_t)((xb_smem(s) >> 4) & 0x3FFF) | ((uint64_t)((xz_smem - xb_smem(s)) >> 4) << 16) |
                               ((uint64_t)(128 >> 4) << 32) | (1ull << 46);
          if (elect_one()) {
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) umma_ss(sd, dsc(la1 + 2 * ks), dsc(lb1 + 2 * ks), idesc_s, ks > 0 ? 1u : 0u);
            if (MODE == 1) umma_ss(sd, dsc(lxa), dxb, idesc_s, 1u);                     // S'  -= lse_j / scale
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) umma_ss(sd + 64, dsc(la2 + 2 * ks), dsc(lb2 + 2 * ks), idesc_s, ks > 0 ? 1u : 0u);
            if (MODE == 1) umma_ss(sd + 64, dsc(lxa + 2), dxb, idesc_s, 1u);            // dP' -= D_j
            umma_commit(bar_sfull(buf));
            if (c == n - 1) umma_commit(bar_aempty(par));         // the operand tiles are free after these MMAs
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 2) {
    // =========================== gradient-MMA issuer ===========================
    {
      constexpr uint32_t idesc_acc = instr_desc(C::M, 64, true);
      constexpr uint32_t kDescHi = 0x40004040u;
      auto dlo = [](uint32_t addr) { return ((addr >> 4) & 0x3FFFu) | (1u << 16); };
      auto dsc = [](uint32_t lo) { return ((uint64_t)kDescHi << 32) | lo; };
      int Tn = 0, Cn = 0;
      for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++Tn) {
        const int n = tile_of(t).nchunks;
        const int ai = Tn % NACC, ak = Tn / NACC;
        const uint32_t acc = tmem + C::TMEM_ACC + ACC_STRIDE * ai;
        for (int c = 0; c < n; ++c, ++Cn) {
          const int s = Cn % C::NSTAGE, buf = Cn % C::NBUF;
          mbar_wait<false>(bar_pfull(buf), (uint32_t)(Cn / C::NBUF) & 1u);
          if (c == 0) mbar_wait<false>(bar_accfree(ai), ((uint32_t)ak & 1u) ^ 1u);   // epilogue of the last tile on this accumulator
          tc_fence_after();
          const uint32_t sb = st_smem + s * C::STAGE_BYTES, sd = tmem + C::TMEM_SD + 128 * buf;
          const uint32_t lb1 = dlo(sb), lb2 = dlo(sb + C::CHUNK_BYTES);
          const uint32_t acc_on = c > 0 ? 1u : 0u;
          if (elect_one()) {
#pragma unroll
            for (int ks = 0; ks < C::N / 16; ++ks) {
              // the packed P / dS of key columns [16 ks, 16 ks + 16): written by elementwise group ks / 2 into its own half
              const uint32_t pa = 32u * (ks >> 1) + 8u * (ks & 1);
              umma_ts(acc, sd + 64 + pa, dsc(lb1 + 128 * ks), idesc_acc, ks > 0 ? 1u : acc_on);
              if (MODE == 1) umma_ts(acc + 64, sd + pa, dsc(lb2 + 128 * ks), idesc_acc, ks > 0 ? 1u : acc_on);
            }
            umma_commit(bar_empty(s));
            umma_commit(bar_sdfree(buf));
            if (c == n - 1) umma_commit(bar_accdone(ai));
          }
          __syncwarp();
        }
      }
    }
  }
  } else if (warp < 12) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 144;");
    // =========================== elementwise group g (one row per thread) ===========================
    const int g = (warp - 4) >> 2;                 // group: takes columns [32 g, 32 g + 32) of every chunk
    const int sp = warp & 3;                       // TMEM subpartition of this warp
    const int row = sp * 32 + lane;                // row of the stationary tile == TMEM lane
    const uint32_t tm = tmem + ((uint32_t)(sp * 32) << 16);
    const int rx = row & 7, ry = (row >> 3) & 7, rl = row >> 6;
    const float cs = p.scale_log2e;

    int Tn = 0, Cn = 0;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++Tn) {
      const Tile2 T = tile_of(t);
      const int x0 = T.x0, y0 = T.y0, l0 = T.l0, b = T.b, h = T.h;
      const bool active = (x0 + rx < p.X) && (y0 + ry < p.Y) && (l0 + rl < p.L);
      const int ax = min(x0 + rx, p.X - 1), ay = min(y0 + ry, p.Y - 1), al = min(l0 + rl, p.L - 1);
      const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
      // streamed interval of this row on every axis, relative to the tile's box (planes: absolute)
      int ix0, ix1, iy0, iy1, il0, il1;
      row_interval<MODE>(ax, C::KX, p.X, ix0, ix1); ix0 -= T.bx0; ix1 -= T.bx0;
      row_interval<MODE>(ay, C::KY, p.Y, iy0, iy1); iy0 -= T.by0; iy1 -= T.by0;
      row_interval<MODE>(al, C::KL, p.L, il0, il1);
      if (!active) { ix1 = ix0; iy1 = iy0; il1 = il0; }
      float my_l2 = 0.f, my_d = 0.f;               // MODE 0: the statistics belong to the row
      if (MODE == 0 && active) {
        const float2 st = stat[((long long)b * p.H + h) * p.N + tok];
        my_l2 = st.x; my_d = st.y;
      }

      int c = 0;
      for (int pl = T.bl0; pl < T.bl1; ++pl) {
        const bool plane_ok = pl >= il0 && pl < il1;
        for (int cy = 0; cy < T.ncy; ++cy)
          for (int cx = 0; cx < T.ncx; ++cx, ++c, ++Cn) {
            // validity of this row over the chunk's columns: bit mask (skip test) and additive biases
            const int xa = max(ix0 - cx * C::HX, 0), xb = min(ix1 - cx * C::HX, C::HX);
            const uint32_t xm = xb > xa ? ((1u << xb) - 1u) & ~((1u << xa) - 1u) : 0u;
            bool anyrow = false;
            float nbr[C::CY];
#pragma unroll
            for (int r = 0; r < C::CY; ++r) {
              const int gy = cy * C::CY + r;
              const bool ok = plane_ok && gy >= iy0 && gy < iy1;
              anyrow |= ok;
              nbr[r] = ok ? (MODE == 0 ? -my_l2 : 0.f) : -INFINITY;
            }
            F2 xz2[C::HX / 2];
#pragma unroll
            for (int x = 0; x < C::HX; x += 2) {
              xz2[x >> 1].x = ((xm >> x) & 1u) ? 0.f : -INFINITY;
              xz2[x >> 1].y = ((xm >> (x + 1)) & 1u) ? 0.f : -INFINITY;
            }
            const int buf = Cn % C::NBUF;
            const uint32_t sd = tm + C::TMEM_SD + 128 * buf;
            mbar_wait(bar_sfull(buf), (uint32_t)(Cn / C::NBUF) & 1u);
            tc_fence_after();
            if (__any_sync(0xffffffffu, anyrow && xm != 0u)) {
              // this group's half of the columns, 16 at a time, software pipelined: the TMEM load of batch k + 1 is issued
              // before the arithmetic of batch k (tcgen05.wait::ld waits for every outstanding load: one batch in flight)
              auto half = [&](auto gc) {
                constexpr int NB = 16, KB0 = 2 * decltype(gc)::value, KB1 = (KB0 + 2 < C::N / NB) ? KB0 + 2 : C::N / NB;
                uint32_t svw[2][NB], dpw[2][NB];
                tmem_ld_issue_n<NB>(sd + KB0 * NB, svw[0]);
                tmem_ld_issue_n<NB>(sd + 64 + KB0 * NB, dpw[0]);
#pragma unroll
                for (int kb = KB0; kb < KB1; ++kb) {
                  const int H0 = kb * NB, cur = (kb - KB0) & 1;
                  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                  reg_fence_n<NB>(svw[cur]);
                  reg_fence_n<NB>(dpw[cur]);
                  if (kb + 1 < KB1) {
                    tmem_ld_issue_n<NB>(sd + H0 + NB, svw[cur ^ 1]);
                    tmem_ld_issue_n<NB>(sd + 64 + H0 + NB, dpw[cur ^ 1]);
                  }
                  uint32_t pw[NB / 2], dw[NB / 2];
#pragma unroll
                  for (int u = 0; u < NB; u += 2) {
                    const int col = H0 + u;                            // compile-time
                    if (col < C::NCOL) {
                      const int r = col / C::HX, x = col % C::HX;     // x even: (x, x + 1) are in the same row
                      // MODE 1: the tensor cores have already subtracted the column statistics (bias K step)
                      const F2 nb = {nbr[r], nbr[r]}, dd = {-my_d, -my_d};
                      F2 tt = ffma2(F2{__uint_as_float(svw[cur][u]), __uint_as_float(svw[cur][u + 1])}, F2{cs, cs}, nb);
                      tt = fadd2(tt, xz2[x >> 1]);
                      const F2 e = {ex2(tt.x), ex2(tt.y)};
                      const F2 gq = fmul2(e, fadd2(F2{__uint_as_float(dpw[cur][u]), __uint_as_float(dpw[cur][u + 1])}, dd));
                      pw[u >> 1] = pack_bf16(e.x, e.y);
                      dw[u >> 1] = pack_bf16(gq.x, gq.y);
                    } else {
                      pw[u >> 1] = 0u; dw[u >> 1] = 0u;
                    }
                  }
                  // packed bf16 results go into this group's own half of the buffer (the other half is still being read)
                  constexpr int PK = 32 * (KB0 / 2);
                  if (MODE == 1) tmem_st_n<NB / 2>(sd + PK + (H0 - PK) / 2, pw);
                  tmem_st_n<NB / 2>(sd + 64 + PK + (H0 - PK) / 2, dw);
                }
              };
              if (g == 0) half(std::integral_constant<int, 0>{}); else half(std::integral_constant<int, 1>{});
            } else {
              uint32_t z[8];
#pragma unroll
              for (int u = 0; u < 8; ++u) z[u] = 0u;
#pragma unroll
              for (int j0 = 0; j0 < 16; j0 += 8) {                 // this group's half: 32 columns = 16 packed
                if (32 * g + 2 * j0 < C::N) {
                  if (MODE == 1) tmem_st8(sd + 32 * g + j0, z);
                  tmem_st8(sd + 64 + 32 * g + j0, z);
                }
              }
            }
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_pfull(buf));
          }
      }
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
    // =========================== epilogue warps (one row per thread) ===========================
    // dx = R(-phi) (scale * acc1) -> bf16 (B4 fused); MODE 1 also acc2 -> bf16 dV.  The accumulators are given back
    // as soon as they are in registers; the table loads and the stores of tile t run under the chunks of tile t + 1.
    const int sp = warp & 3, row = sp * 32 + lane;
    const uint32_t tm = tmem + ((uint32_t)(sp * 32) << 16);
    const int rx = row & 7, ry = (row >> 3) & 7, rl = row >> 6;
    int Tn = 0;
    for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++Tn) {
      int bid = t;
      const int x0 = (bid % p.ntx) * C::TX; bid /= p.ntx;
      const int y0 = (bid % p.nty) * C::TY; bid /= p.nty;
      const int l0 = (bid % p.ntl) * C::TL; bid /= p.ntl;
      const int h = bid % p.H, b = bid / p.H;
      const bool active = (x0 + rx < p.X) && (y0 + ry < p.Y) && (l0 + rl < p.L);
      const int ax = min(x0 + rx, p.X - 1), ay = min(y0 + ry, p.Y - 1), al = min(l0 + rl, p.L - 1);
      const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
      const int ai = Tn % NACC, ak = Tn / NACC;
      mbar_wait_bounded(bar_accdone(ai), (uint32_t)ak & 1u);
      tc_fence_after();
      const uint32_t acc = tm + C::TMEM_ACC + ACC_STRIDE * ai;
      uint32_t vw[MODE == 1 ? C::D / 2 : 1];
      if (MODE == 1) {
        float av[C::D];
#pragma unroll
        for (int j = 0; j < C::D; j += 16) tmem_ld16(acc + 64 + j, *reinterpret_cast<float(*)[16]>(&av[j]));
        tmem_wait_ld();
#pragma unroll
        for (int j = 0; j < C::D; j += 2) vw[j >> 1] = pack_bf16(av[j], av[j + 1]);
      }
      float av[C::D];
#pragma unroll
      for (int j = 0; j < C::D; j += 16) tmem_ld16(acc + j, *reinterpret_cast<float(*)[16]>(&av[j]));
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_accfree(ai));              // the accumulators are in registers
      if (MODE == 1 && active) {
        uint4* r2 = reinterpret_cast<uint4*>(out2 + (((long long)b * p.N + tok) * p.H + h) * C::D);
#pragma unroll
        for (int j = 0; j < C::D / 8; ++j) r2[j] = make_uint4(vw[4 * j], vw[4 * j + 1], vw[4 * j + 2], vw[4 * j + 3]);
      }
      if (active) {
        __nv_bfloat16* r1 = out1 + (((long long)b * p.N + tok) * p.H + h) * C::D;
        const float4* trow = rtab ? rtab + ((long long)b * p.N + tok) * (C::D / 4) : nullptr;   // 2 pairs per float4
#pragma unroll
        for (int j = 0; j < C::D; ++j) av[j] *= p.scale;
        if (trow) {
          auto rot = [&](auto half_pairing) {
            constexpr bool HP = decltype(half_pairing)::value;
#pragma unroll
            for (int m = 0; m < C::D / 2; m += 2) {               // pairs m, m + 1
              const float4 tq = __ldg(trow + (m >> 1));           // (cos m, sin m, cos m+1, sin m+1)
              const int a0 = HP ? m : 2 * m, b0 = HP ? m + C::D / 2 : 2 * m + 1;
              const int a1 = HP ? m + 1 : 2 * m + 2, b1 = HP ? m + 1 + C::D / 2 : 2 * m + 3;
              const float xa0 = av[a0], xb0 = av[b0], xa1 = av[a1], xb1 = av[b1];
              av[a0] = fmaf(xb0, tq.y, xa0 * tq.x); av[b0] = fmaf(-xa0, tq.y, xb0 * tq.x);
              av[a1] = fmaf(xb1, tq.w, xa1 * tq.z); av[b1] = fmaf(-xa1, tq.w, xb1 * tq.z);
            }
          };
          if (p.pairing) rot(std::true_type{}); else rot(std::false_type{});
        }
#pragma unroll
        for (int j = 0; j < C::D; j += 8) {
          uint4 w;
          w.x = pack_bf16(av[j], av[j + 1]);     w.y = pack_bf16(av[j + 2], av[j + 3]);
          w.z = pack_bf16(av[j + 4], av[j + 5]); w.w = pack_bf16(av[j + 6], av[j + 7]);
          reinterpret_cast<uint4*>(r1)[j >> 3] = w;
        }
      }
    }
  }

  // ---- teardown
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem, C::TMEM_COLS);
  }
}

DeviceState g_states[64];
std::mutex g_mu;

template <class C>
cudaError_t launch_bwd2_cfg(int slot, const Problem& p, const void* qr, const void* kr, const void* v, const void* d_o,
                            const float2* stat, const void* bias, const void* rtab, void* dq, void* dk, void* dv,
                            cudaStream_t stream, int* launches) {
  // bias rows [B*L, Y, X, H, 8] bf16, unswizzled boxes of one head x (HX, CY) tokens
  CUtensorMap t_bias;
  {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorInvalidValue;
    const cuuint64_t dims[5] = {8, (cuuint64_t)p.H, (cuuint64_t)p.X, (cuuint64_t)p.Y, (cuuint64_t)p.B * (cuuint64_t)p.L};
    const cuuint64_t strides[4] = {16, (cuuint64_t)p.H * 16, (cuuint64_t)p.X * p.H * 16, (cuuint64_t)p.Y * p.X * p.H * 16};
    const cuuint32_t box[5] = {8, 1, (cuuint32_t)C::HX, (cuuint32_t)C::CY, 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    if (fn(&t_bias, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(bias), dims, strides, box, estr,
           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  CUtensorMap tq_t, tdo_t, tk_c, tv_c, tk_t, tv_t, tq_c, tdo_c;
  if (!make_map(&tq_t, qr, p, C::TX, C::TY, C::TL) || !make_map(&tdo_t, d_o, p, C::TX, C::TY, C::TL) ||
      !make_map(&tk_c, kr, p, C::HX, C::CY, 1) || !make_map(&tv_c, v, p, C::HX, C::CY, 1) ||
      !make_map(&tk_t, kr, p, C::TX, C::TY, C::TL) || !make_map(&tv_t, v, p, C::TX, C::TY, C::TL) ||
      !make_map(&tq_c, qr, p, C::HX, C::CY, 1) || !make_map(&tdo_c, d_o, p, C::HX, C::CY, 1))
    return cudaErrorInvalidValue;
  BwdParams bp;
  bp.B = p.B; bp.H = p.H; bp.L = p.L; bp.Y = p.Y; bp.X = p.X; bp.N = p.N;
  bp.ntl = (p.L + C::TL - 1) / C::TL; bp.nty = (p.Y + C::TY - 1) / C::TY; bp.ntx = (p.X + C::TX - 1) / C::TX;
  bp.scale = p.scale; bp.scale_log2e = p.scale * 1.4426950408889634f; bp.pairing = p.pairing;
  const long long ntiles = (long long)p.B * p.H * bp.ntl * bp.nty * bp.ntx;
  if (ntiles > 0x7fffffffLL) return cudaErrorInvalidValue;
  DeviceState* ds = device_state(g_states, g_mu);
  if (!ds) return cudaErrorInvalidDevice;
  const unsigned grid = (unsigned)(ntiles < ds->sm_count ? ntiles : ds->sm_count);
  cudaError_t e = ensure_smem_attr(ds, g_mu, 2 * slot, na3d_bwd_tc2_kernel<C, 0>, C::SMEM_BYTES);
  if (e == cudaSuccess) e = ensure_smem_attr(ds, g_mu, 2 * slot + 1, na3d_bwd_tc2_kernel<C, 1>, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  prof_begin("na3d_bwd_dq_tcgen05", stream);
  na3d_bwd_tc2_kernel<C, 0><<<grid, kBwd2Threads, C::SMEM_BYTES, stream>>>(tq_t, tdo_t, tk_c, tv_c, t_bias, stat, (const float4*)rtab,
                                                                          (__nv_bfloat16*)dq, nullptr, bp, (int)ntiles);
  prof_end(stream);
  prof_begin("na3d_bwd_dkdv_tcgen05", stream);
  na3d_bwd_tc2_kernel<C, 1><<<grid, kBwd2Threads, C::SMEM_BYTES, stream>>>(tk_t, tv_t, tq_c, tdo_c, t_bias, stat, (const float4*)rtab,
                                                                          (__nv_bfloat16*)dk, (__nv_bfloat16*)dv, bp, (int)ntiles);
  prof_end(stream);
  if (launches) *launches += 2;
  return cudaGetLastError();
}

}  // namespace

// The two main kernels of the backward in their persistent form; false if the window is not instantiated.
cudaError_t launch_bwd_tc2_main(const Problem& p, const void* qr, const void* kr, const void* v, const void* d_o,
                                const void* stat, const void* bias, const void* rtab, void* dq, void* dk, void* dv,
                                cudaStream_t stream, int* launches) {
#define X(I_, KL_, KY_, KX_)                                   \
  if (p.kL == KL_ && p.kY == KY_ && p.kX == KX_)                \
    return launch_bwd2_cfg<Bwd2Cfg<KL_, KY_, KX_>>(I_, p, qr, kr, v, d_o, (const float2*)stat, bias, rtab, dq, dk, dv, stream, launches);
  X(0, 3, 7, 7)
  X(1, 3, 5, 5)
  X(2, 3, 3, 3)
  X(3, 9, 9, 9)
#undef X
  return cudaErrorNotSupported;
}

}  // namespace strata
