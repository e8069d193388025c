// na3d_bwd_tc.cu -- tcgen05 / TMEM / TMA backward kernels for 3D neighbourhood attention (sm_100a).
//
// Steps B1-B4 of DESIGN.md on pre-rotated bf16 operands (rope.cu rotates Q, K before; the transpose
// rotation B4 of dQrot, dKrot is fused into the epilogues, from an fp32 cos/sin table).  PAPER.md gives no backward; BASELINE.json config 4 and SURVEY.md §8(a)
// rows B1-B4 define it:
//   B1  D_i    = sum_c dO_ic O_ic                       (bwd_stat_kernel, stored with lse * log2 e)
//   B2  p_ij   = exp(scale qrot_i . krot_j - lse_i),  dP_ij = dO_i . v_j,  dS_ij = p_ij (dP_ij - D_i)
//       dqrot_i = scale sum_j dS_ij krot_j;  dkrot_j = scale sum_i dS_ij qrot_i;  dV_j = sum_i p_ij dO_i
//
// ONE kernel template, two modes, both "a stationary tile of 128 rows against streamed chunks":
//   MODE 0 (dQ, query-stationary)  rows = queries: A1 = Qrot, A2 = dO tile; chunks = the keys of the
//       tile's window halo: B1 = Krot, B2 = V.            acc1 = dQrot = sum dS  B1
//   MODE 1 (dK/dV, key-stationary) rows = keys:    A1 = Krot, A2 = V tile;  chunks = the queries of
//       the tile's INVERSE halo (B3: the queries whose inward-clamped window holds a key of the tile --
//       not symmetric at the borders): B1 = Qrot, B2 = dO.  acc1 = dKrot = sum dS^T B1,
//       acc2 = dV = sum P^T B2.  Row statistics (lse, D) belong to the chunk's columns here: the
//       elementwise threads fetch them one chunk ahead and publish them in shared memory.
// Per chunk (CY rows x HX columns of one level plane = N <= 64 columns):
//   S' = A1 B1^T and dP' = A2 B2^T on the tensor cores (M = 128, K = 64) -> TMEM;
//   one row per thread: p = 2^(S' scale log2e - lse log2e) under the window mask, dS = p (dP' - D),
//   written back to TMEM as bf16 over the buffers they came from;
//   acc1 += dS B1 (and acc2 += P B2) with the bf16 matrix as the TMEM A operand and the SAME shared
//   memory chunk re-read as an MN-major B operand.
// No atomics: every output row is owned by exactly one thread; deterministic.
//
// Warp roles (192 threads, 2 CTAs / SM -- the other CTA fills this one's MMA <-> elementwise bubbles):
// warp 0 = TMA producer, warp 1 = MMA issuer + TMEM owner, warps 2-5 = elementwise + epilogue.
// TMEM (256 columns): acc1 [0,64) | acc2 [64,128) | S' -> P [128,192) | dP' -> dS [192,256).
#include <cstdio>
#include <cstdlib>
#include <type_traits>

#include "tc_common.cuh"
#include "bwd_common.cuh"

namespace strata {
namespace {

using namespace tc;

template <int KL_, int KY_, int KX_>
struct BwdCfg {
  static constexpr int D = 64, KL = KL_, KY = KY_, KX = KX_;
  static constexpr int TL = 2, TY = 8, TX = 8, M = 128;            // stationary tile (tokens)
  static constexpr int HX = TX + KX - 1;                           // chunk width (columns of one row)
  static constexpr int CY = 4;                                     // chunk rows
  static constexpr int NCOL = CY * HX;                             // real columns of a chunk
  static constexpr int N = (NCOL + 15) / 16 * 16;                  // UMMA N (pad columns are masked)
  static constexpr int TILE_BYTES = M * 128, CHUNK_BYTES = N * 128;
  static constexpr int STAT_BYTES = CY * 128;                      // [CY][16 tokens] float2 (MODE 1)
  static constexpr int STAGE_BYTES = 2 * CHUNK_BYTES;              // B1 | B2
  static constexpr int NSTAGE = 3;
  static constexpr int TMEM_ACC1 = 0, TMEM_ACC2 = 64, TMEM_S = 128, TMEM_DP = 192, TMEM_COLS = 256;
  static constexpr int BAR_BYTES = 128 + 2 * STAT_BYTES;           // barriers | two statistics buffers
  static constexpr int SMEM_BYTES = 1024 + 2 * TILE_BYTES + NSTAGE * STAGE_BYTES + BAR_BYTES;
  static_assert(KL % 2 == 1 && KY % 2 == 1 && KX % 2 == 1, "odd windows only");
  static_assert(N <= 64 && HX <= 16 && HX % 2 == 0, "a chunk must fit 64 TMEM columns; column pairs share a row");
  static_assert(2 * SMEM_BYTES <= 227 * 1024, "two CTAs per SM");
};

constexpr int kBwdThreads = 192;

// ------------------------------------------------------------------------------------------------
// Kernel
// ------------------------------------------------------------------------------------------------
template <class C, int MODE>
__global__ void __launch_bounds__(kBwdThreads, 2)
na3d_bwd_tc_kernel(const __grid_constant__ CUtensorMap tm_a1, const __grid_constant__ CUtensorMap tm_a2,
                   const __grid_constant__ CUtensorMap tm_b1, const __grid_constant__ CUtensorMap tm_b2,
                   const float2* __restrict__ stat, const float4* __restrict__ rtab,
                   __nv_bfloat16* __restrict__ out1, __nv_bfloat16* __restrict__ out2, const BwdParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t a1_smem = base, a2_smem = base + C::TILE_BYTES;
  const uint32_t st_smem = a2_smem + C::TILE_BYTES;                       // stages
  const uint32_t bars = st_smem + C::NSTAGE * C::STAGE_BYTES;
  const uint32_t bar_a = bars;
  auto bar_full = [&](int s) { return bars + 8u * (1 + s); };
  auto bar_empty = [&](int s) { return bars + 8u * (1 + C::NSTAGE + s); };
  const uint32_t bar_sfull = bars + 8u * (1 + 2 * C::NSTAGE);
  const uint32_t bar_pfull = bar_sfull + 8, bar_done = bar_sfull + 16, tmem_slot = bar_sfull + 24;
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- stationary tile of this CTA: x fastest, then y, level, head, sample
  int bid = blockIdx.x;
  const int tx = bid % p.ntx; bid /= p.ntx;
  const int ty = bid % p.nty; bid /= p.nty;
  const int tl = bid % p.ntl; bid /= p.ntl;
  const int h = bid % p.H;
  const int b = bid / p.H;
  const int x0 = tx * C::TX, y0 = ty * C::TY, l0 = tl * C::TL;
  const int xl = min(x0 + C::TX, p.X) - 1, yl = min(y0 + C::TY, p.Y) - 1, ll = min(l0 + C::TL, p.L) - 1;
  // streamed box of the tile: union of its rows' intervals (both interval ends are monotone in the row index)
  int bx0, bx1, by0, by1, bl0, bl1, t0, t1;
  row_interval<MODE>(x0, C::KX, p.X, bx0, t1); row_interval<MODE>(xl, C::KX, p.X, t0, bx1);
  row_interval<MODE>(y0, C::KY, p.Y, by0, t1); row_interval<MODE>(yl, C::KY, p.Y, t0, by1);
  row_interval<MODE>(l0, C::KL, p.L, bl0, t1); row_interval<MODE>(ll, C::KL, p.L, t0, bl1);
  const int ncx = (bx1 - bx0 + C::HX - 1) / C::HX;          // 1 except at clamped borders of ragged grids (MODE 1)
  const int ncy = (by1 - by0 + C::CY - 1) / C::CY;
  const int nchunks = (bl1 - bl0) * ncy * ncx;

  // ---- one-time setup
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_a1); tma_prefetch_desc(&tm_a2); tma_prefetch_desc(&tm_b1); tma_prefetch_desc(&tm_b2);
    mbar_init(bar_a, 1);
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(bar_full(s), 1); mbar_init(bar_empty(s), 1); }
    mbar_init(bar_sfull, 1);
    mbar_init(bar_pfull, 128);
    mbar_init(bar_done, 1);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, C::TMEM_COLS);
  // chunk rows the TMA box never writes (pad columns of the UMMA N) must hold finite numbers
  if (C::N > C::NCOL) {
    for (int s = 0; s < C::NSTAGE; ++s)
      for (int u = threadIdx.x; u < 2 * (C::N - C::NCOL) * 8; u += kBwdThreads) {
        const int which = u / ((C::N - C::NCOL) * 8), off = u % ((C::N - C::NCOL) * 8);
        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(st_smem + s * C::STAGE_BYTES + which * C::CHUNK_BYTES +
                                                                     C::NCOL * 128 + off * 16), "r"(0u) : "memory");
      }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot_ptr;

  if (warp == 0) {
    // =========================== TMA producer ===========================
    if (lane == 0) {
      const int bl = b * p.L;
      mbar_expect_tx(bar_a, 2 * C::TILE_BYTES);
      tma_load_5d(a1_smem, &tm_a1, bar_a, 0, h, x0, y0, bl + l0);
      tma_load_5d(a2_smem, &tm_a2, bar_a, 0, h, x0, y0, bl + l0);
      int c = 0;
      for (int pl = bl0; pl < bl1; ++pl)
        for (int cy = 0; cy < ncy; ++cy)
          for (int cx = 0; cx < ncx; ++cx, ++c) {
            const int s = c % C::NSTAGE;
            const uint32_t ph = (uint32_t)(c / C::NSTAGE) & 1u;
            const uint32_t sb = st_smem + s * C::STAGE_BYTES;
            const int gx = bx0 + cx * C::HX, gy = by0 + cy * C::CY;
            mbar_wait(bar_empty(s), ph ^ 1u);
            mbar_expect_tx(bar_full(s), 2 * C::NCOL * 128);
            tma_load_5d(sb, &tm_b1, bar_full(s), 0, h, gx, gy, bl + pl);
            tma_load_5d(sb + C::CHUNK_BYTES, &tm_b2, bar_full(s), 0, h, gx, gy, bl + pl);
          }
    }
  } else if (warp == 1) {
    // =========================== MMA issuer ===========================
    if (lane == 0) {
      constexpr uint32_t idesc_s = instr_desc(C::M, C::N, false);
      constexpr uint32_t idesc_acc = instr_desc(C::M, 64, true);
      mbar_wait(bar_a, 0);
      tc_fence_after();
      const uint64_t da1 = smem_desc(a1_smem), da2 = smem_desc(a2_smem);
      for (int c = 0; c < nchunks; ++c) {
        const int s = c % C::NSTAGE;
        const uint32_t ph = (uint32_t)(c / C::NSTAGE) & 1u;
        const uint32_t sb = st_smem + s * C::STAGE_BYTES;
        mbar_wait(bar_full(s), ph);
        BTRACE(0, c);
        tc_fence_after();
        // ---- S' = A1 B1^T, dP' = A2 B2^T  (M = 128, N, K = 64 in steps of 16).  The descriptors of the K steps
        // differ by a constant in their address field: one base per operand, then additions.
        const uint64_t db1 = smem_desc(sb), db2 = smem_desc(sb + C::CHUNK_BYTES);
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          umma_ss(tmem + C::TMEM_S, da1 + 2 * ks, db1 + 2 * ks, idesc_s, ks > 0 ? 1u : 0u);
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          umma_ss(tmem + C::TMEM_DP, da2 + 2 * ks, db2 + 2 * ks, idesc_s, ks > 0 ? 1u : 0u);
        umma_commit(bar_sfull);
        BTRACE(1, c);
        // ---- acc1 += dS B1, acc2 += P B2  (A from TMEM, K = N columns in steps of 16)
        mbar_wait(bar_pfull, (uint32_t)c & 1u);
        BTRACE(2, c);
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < C::N / 16; ++ks) {
          umma_ts(tmem + C::TMEM_ACC1, tmem + C::TMEM_DP + 8 * ks, db1 + 128 * ks, idesc_acc, (c > 0 || ks > 0) ? 1u : 0u);
          if (MODE == 1)
            umma_ts(tmem + C::TMEM_ACC2, tmem + C::TMEM_S + 8 * ks, db2 + 128 * ks, idesc_acc, (c > 0 || ks > 0) ? 1u : 0u);
        }
        umma_commit(bar_empty(s));
        BTRACE(3, c);
        if (c == nchunks - 1) umma_commit(bar_done);
      }
    }
  } else {
    // =========================== elementwise (one row per thread) + epilogue ===========================
    const int sp = warp & 3;                       // TMEM subpartition of this warp
    const int row = sp * 32 + lane;                // row of the stationary tile == TMEM lane
    const uint32_t tm = tmem + ((uint32_t)(sp * 32) << 16);
    const int rx = row & 7, ry = (row >> 3) & 7, rl = row >> 6;
    const bool active = (x0 + rx < p.X) && (y0 + ry < p.Y) && (l0 + rl < p.L);
    const int ax = min(x0 + rx, p.X - 1), ay = min(y0 + ry, p.Y - 1), al = min(l0 + rl, p.L - 1);
    const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
    // streamed interval of this row on every axis, relative to the tile's box (planes: absolute)
    int ix0, ix1, iy0, iy1, il0, il1;
    row_interval<MODE>(ax, C::KX, p.X, ix0, ix1); ix0 -= bx0; ix1 -= bx0;
    row_interval<MODE>(ay, C::KY, p.Y, iy0, iy1); iy0 -= by0; iy1 -= by0;
    row_interval<MODE>(al, C::KL, p.L, il0, il1);
    if (!active) { ix1 = ix0; iy1 = iy0; il1 = il0; }
    float my_l2 = 0.f, my_d = 0.f;                 // MODE 0: the statistics belong to the row
    if (MODE == 0 && active) {
      const float2 st = stat[((long long)b * p.H + h) * p.N + tok];
      my_l2 = st.x; my_d = st.y;
    }
    const float cs = p.scale_log2e;
    // MODE 1: the statistics belong to the chunk's columns (queries).  Thread t < NCOL fetches the pair of
    // column t one chunk ahead (registers), publishes it in shared memory [chunk & 1][r][16 tokens] at the
    // start of the chunk; a named barrier of the 128 elementwise threads orders write -> reads.
    const int et = threadIdx.x - 64;
    const int sr = et / C::HX, sx = et % C::HX;
    auto fetch_stat = [&](int cc) -> float2 {
      if (MODE != 1 || et >= C::NCOL || cc >= nchunks) return make_float2(0.f, 0.f);
      const int ccx = cc % ncx, t2 = cc / ncx, ccy = t2 % ncy, cpl = bl0 + t2 / ncy;
      const int gy = by0 + ccy * C::CY + sr, gx = bx0 + ccx * C::HX + sx;
      if (gy >= p.Y || gx >= p.X) return make_float2(0.f, 0.f);
      return __ldg(&stat[((long long)b * p.H + h) * p.N + ((long long)cpl * p.Y + gy) * p.X + gx]);
    };
    float2 next_stat = fetch_stat(0);

    int c = 0;
    for (int pl = bl0; pl < bl1; ++pl) {
      const bool plane_ok = pl >= il0 && pl < il1;
      for (int cy = 0; cy < ncy; ++cy)
        for (int cx = 0; cx < ncx; ++cx, ++c) {
          // validity mask of this row over the chunk's columns, column r * HX + x <-> bit
          const int xa = max(ix0 - cx * C::HX, 0), xb = min(ix1 - cx * C::HX, C::HX);
          const uint32_t xm = xb > xa ? ((1u << xb) - 1u) & ~((1u << xa) - 1u) : 0u;
          unsigned long long vm = 0ull;
#pragma unroll
          for (int r = 0; r < C::CY; ++r) {
            const int gy = cy * C::CY + r;
            if (plane_ok && gy >= iy0 && gy < iy1) vm |= (unsigned long long)xm << (r * C::HX);
          }
          // the same mask as additive biases: nbr[r] = -lse (MODE 0) or 0 (MODE 1) for a valid chunk row, -inf else;
          // xz2[x / 2] = 0 / -inf per column of the pair
          float nbr[C::CY];
          F2 xz2[C::HX / 2];
#pragma unroll
          for (int r = 0; r < C::CY; ++r) {
            const int gy = cy * C::CY + r;
            nbr[r] = (plane_ok && gy >= iy0 && gy < iy1) ? (MODE == 0 ? -my_l2 : 0.f) : -INFINITY;
          }
#pragma unroll
          for (int x = 0; x < C::HX; x += 2) {
            xz2[x >> 1].x = ((xm >> x) & 1u) ? 0.f : -INFINITY;
            xz2[x >> 1].y = ((xm >> (x + 1)) & 1u) ? 0.f : -INFINITY;
          }
          const uint32_t stat_smem = bars + 128 + (uint32_t)(c & 1) * C::STAT_BYTES;
          if (MODE == 1) {
            if (et < C::NCOL)
              asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(stat_smem + (sr * 16 + sx) * 8), "f"(next_stat.x), "f"(next_stat.y) : "memory");
            next_stat = fetch_stat(c + 1);
            asm volatile("bar.sync 1, 128;" ::: "memory");
          }
          mbar_wait(bar_sfull, (uint32_t)c & 1u);
          if (et == 0) BTRACE(4, c);
          tc_fence_after();
          if (__any_sync(0xffffffffu, vm != 0ull)) {
            // S' and dP' in batches of 32 columns: one wait per batch, branch-free arithmetic in between
            auto batch = [&](auto h0c, auto nbc) {
              constexpr int H0 = decltype(h0c)::value, NB = decltype(nbc)::value;
              uint32_t svw[NB], dpw[NB];
              tmem_ld_issue_n<NB>(tm + C::TMEM_S + H0, svw);
              tmem_ld_issue_n<NB>(tm + C::TMEM_DP + H0, dpw);
              asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
              reg_fence_n<NB>(svw);
              reg_fence_n<NB>(dpw);
              uint32_t pw[NB / 2], dw[NB / 2];
#pragma unroll
              for (int u = 0; u < NB; u += 2) {
                const int col = H0 + u;                            // compile-time
                if (col < C::NCOL) {
                  const int r = col / C::HX, x = col % C::HX;     // x even: (x, x + 1) are in the same row
                  // window mask as an additive bias: 0 or -inf per chunk row (nbr) and per column pair (xz2)
                  F2 nb = {nbr[r], nbr[r]}, dd = {-my_d, -my_d};
                  if (MODE == 1) {
                    float4 st;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                 : "=f"(st.x), "=f"(st.y), "=f"(st.z), "=f"(st.w) : "r"(stat_smem + (r * 32 + 2 * x) * 4));
                    nb = ffma2(F2{st.x, st.z}, F2{-1.f, -1.f}, nb);
                    dd = F2{-st.y, -st.w};
                  }
                  F2 t = ffma2(F2{__uint_as_float(svw[u]), __uint_as_float(svw[u + 1])}, F2{cs, cs}, nb);
                  t = fadd2(t, xz2[x >> 1]);
                  const F2 e = {ex2(t.x), ex2(t.y)};
                  const F2 g = fmul2(e, fadd2(F2{__uint_as_float(dpw[u]), __uint_as_float(dpw[u + 1])}, dd));
                  pw[u >> 1] = pack_bf16(e.x, e.y);
                  dw[u >> 1] = pack_bf16(g.x, g.y);
                } else {
                  pw[u >> 1] = 0u; dw[u >> 1] = 0u;
                }
              }
              if (MODE == 1) tmem_st_n<NB / 2>(tm + C::TMEM_S + H0 / 2, pw);
              tmem_st_n<NB / 2>(tm + C::TMEM_DP + H0 / 2, dw);
            };
            batch(std::integral_constant<int, 0>{}, std::integral_constant<int, (C::N < 32 ? C::N : 32)>{});
            if constexpr (C::N > 32) batch(std::integral_constant<int, 32>{}, std::integral_constant<int, C::N - 32>{});
          } else {
            uint32_t z[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) z[u] = 0u;
#pragma unroll
            for (int j0 = 0; j0 < C::N / 2; j0 += 8) {
              if (MODE == 1) tmem_st8(tm + C::TMEM_S + j0, z);
              tmem_st8(tm + C::TMEM_DP + j0, z);
            }
          }
          if (et == 0) BTRACE(5, c);
          tmem_wait_st();
          tc_fence_before();
          if (et == 0) BTRACE(6, c);
          mbar_arrive(bar_pfull);
        }
    }
    // ---- epilogue: B4 fused -- dx = R(-phi) (scale * acc1), (a, b) -> (a cos + b sin, b cos - a sin) on every
    // rotary pair of the row, rounded to bf16; acc2 -> bf16 dV
    mbar_wait(bar_done, 0);
    tc_fence_after();
    {
      __nv_bfloat16* r1 = out1 + (((long long)b * p.N + tok) * p.H + h) * C::D;
      const float4* trow = rtab ? rtab + ((long long)b * p.N + tok) * (C::D / 4) : nullptr;   // 2 pairs per float4
      float av[C::D];
#pragma unroll
      for (int j = 0; j < C::D; j += 16) tmem_ld16(tm + C::TMEM_ACC1 + j, *reinterpret_cast<float(*)[16]>(&av[j]));
      tmem_wait_ld();
#pragma unroll
      for (int j = 0; j < C::D; ++j) av[j] *= p.scale;
      if (active) {
        if (trow) {
          auto rot = [&](auto half_pairing) {
            constexpr bool HP = decltype(half_pairing)::value;
#pragma unroll
            for (int m = 0; m < C::D / 2; m += 2) {               // pairs m, m + 1
              const float4 t = __ldg(trow + (m >> 1));            // (cos m, sin m, cos m+1, sin m+1)
              constexpr int dummy = 0; (void)dummy;
              const int a0 = HP ? m : 2 * m, b0 = HP ? m + C::D / 2 : 2 * m + 1;
              const int a1 = HP ? m + 1 : 2 * m + 2, b1 = HP ? m + 1 + C::D / 2 : 2 * m + 3;
              const float xa0 = av[a0], xb0 = av[b0], xa1 = av[a1], xb1 = av[b1];
              av[a0] = fmaf(xb0, t.y, xa0 * t.x); av[b0] = fmaf(-xa0, t.y, xb0 * t.x);
              av[a1] = fmaf(xb1, t.w, xa1 * t.z); av[b1] = fmaf(-xa1, t.w, xb1 * t.z);
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
    if (MODE == 1) {
      __nv_bfloat16* r2 = out2 + (((long long)b * p.N + tok) * p.H + h) * C::D;
#pragma unroll
      for (int j = 0; j < C::D; j += 16) {
        float av[16];
        tmem_ld16(tm + C::TMEM_ACC2 + j, av);
        tmem_wait_ld();
        if (active) {
          uint4 w0, w1;
          w0.x = pack_bf16(av[0], av[1]);   w0.y = pack_bf16(av[2], av[3]);
          w0.z = pack_bf16(av[4], av[5]);   w0.w = pack_bf16(av[6], av[7]);
          w1.x = pack_bf16(av[8], av[9]);   w1.y = pack_bf16(av[10], av[11]);
          w1.z = pack_bf16(av[12], av[13]); w1.w = pack_bf16(av[14], av[15]);
          reinterpret_cast<uint4*>(r2 + j)[0] = w0;
          reinterpret_cast<uint4*>(r2 + j)[1] = w1;
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

// B1 (+ the row statistics in the form the kernels above consume): stat[b][h][t] = (lse * log2 e, D),
// D = sum_c dO_c O_c.  8 lanes per (b, token, h) row of 64 channels, rows in memory order.
__global__ void __launch_bounds__(256)
bwd_stat_kernel(const __nv_bfloat16* __restrict__ o, const __nv_bfloat16* __restrict__ d_o,
                const float* __restrict__ lse, float2* __restrict__ stat, long long rows, long long N, int H) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long r = gid >> 3;
  const int sub = (int)(gid & 7);
  float part = 0.f;
  if (r < rows) {
    const uint4 a = reinterpret_cast<const uint4*>(o + r * 64)[sub], g = reinterpret_cast<const uint4*>(d_o + r * 64)[sub];
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
  if (r < rows && sub == 0) {
    const int h = (int)(r % H);
    const long long bt = r / H, b = bt / N, t = bt - b * N;
    const long long idx = (b * H + h) * N + t;
    stat[idx] = make_float2(lse[idx] * 1.4426950408889634f, part);
  }
}

}  // namespace
cudaError_t launch_bwd_tc2_main(const Problem& p, const void* qr, const void* kr, const void* v, const void* d_o,
                                const void* stat, const void* rtab, void* dq, void* dk, void* dv,
                                cudaStream_t stream, int* launches);
namespace {

template <class C>
cudaError_t launch_bwd_cfg(const Problem& p, const void* qr, const void* kr, const void* v, const void* o,
                           const void* d_o, const float* lse, float2* stat, const void* rtab, void* dq, void* dk, void* dv,
                           cudaStream_t stream, int* launches) {
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
#ifdef STRATA_TRACE
  {
    const char* e = getenv("STRATA_TRACE_PTR");
    bp.trace = e ? (unsigned long long*)strtoull(e, nullptr, 0) : nullptr;
    const char* cc = getenv("STRATA_TRACE_CTA");
    bp.trace_cta = cc ? atoi(cc) : 0;
  }
#endif
  const long long grid = (long long)p.B * p.H * bp.ntl * bp.nty * bp.ntx;
  const long long rows = p.rows(), sgrid = (rows * 8 + 255) / 256;
  if (grid > 0x7fffffffLL || sgrid > 0x7fffffffLL) return cudaErrorInvalidValue;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(na3d_bwd_tc_kernel<C, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(na3d_bwd_tc_kernel<C, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
#ifdef STRATA_DEBUG_SYNC
#define STRATA_DBG(what) do { cudaError_t de = cudaStreamSynchronize(stream); fprintf(stderr, "[bwd_tc] %s: %s\n", what, cudaGetErrorString(de)); } while (0)
#else
#define STRATA_DBG(what) do {} while (0)
#endif
  STRATA_DBG("before");
  prof_begin("na3d_bwd_stat", stream);
  bwd_stat_kernel<<<(unsigned)sgrid, 256, 0, stream>>>((const __nv_bfloat16*)o, (const __nv_bfloat16*)d_o, lse, stat, rows, p.N, p.H);
  prof_end(stream);
  STRATA_DBG("stat");
  static const bool use_v2 = getenv("STRATA_BWD2") ? atoi(getenv("STRATA_BWD2")) != 0 : true;
  if (use_v2) {
    if (launches) *launches += 1;
    return launch_bwd_tc2_main(p, qr, kr, v, d_o, stat, rtab, dq, dk, dv, stream, launches);
  }
  prof_begin("na3d_bwd_dq_tcgen05", stream);
  na3d_bwd_tc_kernel<C, 0><<<(unsigned)grid, kBwdThreads, C::SMEM_BYTES, stream>>>(tq_t, tdo_t, tk_c, tv_c, stat, (const float4*)rtab, (__nv_bfloat16*)dq,
                                                                                  nullptr, bp);
  prof_end(stream);
  STRATA_DBG("dq");
  prof_begin("na3d_bwd_dkdv_tcgen05", stream);
  na3d_bwd_tc_kernel<C, 1><<<(unsigned)grid, kBwdThreads, C::SMEM_BYTES, stream>>>(tk_t, tv_t, tq_c, tdo_c, stat, (const float4*)rtab, (__nv_bfloat16*)dk,
                                                                                  (__nv_bfloat16*)dv, bp);
  prof_end(stream);
  STRATA_DBG("dkdv");
  if (launches) *launches += 3;
  return cudaGetLastError();
}
#undef STRATA_DBG

}  // namespace

// Shapes the tensor-core backward covers: bf16, head_dim 64, the windows below.
#define STRATA_BWD_CONFIGS(X) \
  X(3, 7, 7)                  \
  X(3, 5, 5)                  \
  X(3, 3, 3)

bool tc_bwd_supported(const Problem& p) {
  if (p.dtype != 1 || p.D != 64) return false;
#define X(KL_, KY_, KX_) \
  if (p.kL == KL_ && p.kY == KY_ && p.kX == KX_) return true;
  STRATA_BWD_CONFIGS(X)
#undef X
  return false;
}

cudaError_t launch_bwd_tc(const Problem& p, const void* qr, const void* kr, const void* v, const void* o,
                          const void* d_o, const float* lse, void* stat, const void* rtab, void* dq, void* dk,
                          void* dv, cudaStream_t stream, int* launches) {
#define X(KL_, KY_, KX_)                                        \
  if (p.kL == KL_ && p.kY == KY_ && p.kX == KX_)                \
    return launch_bwd_cfg<BwdCfg<KL_, KY_, KX_>>(p, qr, kr, v, o, d_o, lse, (float2*)stat, rtab, dq, dk, dv, stream, launches);
  STRATA_BWD_CONFIGS(X)
#undef X
  return cudaErrorNotSupported;
}

}  // namespace strata
