// na3d_tc_fwd.cu -- tcgen05 / TMEM / TMA forward kernel for 3D neighbourhood attention (sm_100a).
//
// Steps A3-A6 of DESIGN.md on pre-rotated bf16 operands (A1, A2 are done by rope.cu):
//   one CTA owns a 3D query tile of TL x TY x TX = 2 x 8 x 8 = 128 queries of one (sample, head);
//   the union of its neighbours' keys -- the halo box of (TL+kL-1) x (TY+kY-1) x (TX+kX-1) keys,
//   trimmed to what the inward-clamped windows (R1) really reach -- is
//   streamed through shared memory by TMA in chunks of CY = 8 key rows of one level plane;
//   S = Qrot Krot^T and O += P V run on the 5th-gen tensor cores (tcgen05.mma, M = 128,
//   accumulators in TMEM); one query row per thread, the window mask applied as an additive -inf bias and whole key
//   rows / planes skipped per warp.  As in the fused forward there is no running maximum and no rescale of O
//   (R19): P = 2^(s scale log2 e); a row whose sum leaves 2^-80 .. 2^100 is listed in `fix` and recomputed
//   by na3d_fix_rows_kernel (two-pass softmax from the raw Q, K) right after this kernel.  Dropping the maximum, the
//   optimistic-pass / redo logic and the O rescale took 6 % off config 2 and 12 % off the 9 x 9 x 9 shape.
//
// Warp roles (192 threads): warp 0 = TMA producer, warp 1 = MMA issuer + TMEM owner,
// warps 2-5 = softmax + epilogue (TMEM subpartition = warp index mod 4).
// Pipelines (mbarriers): K/V stage full/empty (TMA <-> MMA), s_full (MMA1 -> softmax),
// p_full (softmax -> MMA2), pv_done (MMA2 -> epilogue).
//
// TMEM columns: O [0, D) fp32 | S [D, D+NKEY) fp32, overwritten by P (bf16x2, A operand of MMA2).
#include "tc_common.cuh"

namespace strata {
namespace {

using namespace tc;

// ------------------------------------------------------------------------------------------------
// Configuration
// ------------------------------------------------------------------------------------------------
template <int D_, int KL_, int KY_, int KX_>
struct Cfg {
  static constexpr int D = D_, KL = KL_, KY = KY_, KX = KX_;
  static constexpr int TL = 2, TY = 8, TX = 8, M = 128;            // query tile
  static constexpr int HL = TL + KL - 1, HY = TY + KY - 1, HX = TX + KX - 1;   // halo box
  static constexpr int CY = (D == 128 || HX == 16) ? 4 : 8;        // key rows per chunk (d = 128 / 16-wide halos: 64 keys, so that two S buffers and two CTAs per SM fit)
  static constexpr int NKEY = CY * HX;                             // keys per chunk (UMMA N of S)
  static constexpr int DSUB = D / 64;                              // 128-byte sub-tiles per row
  static constexpr int SUB_Q = M * 128, SUB_KV = NKEY * 128;       // bytes of one sub-tile
  static constexpr int Q_BYTES = DSUB * SUB_Q, STAGE_BYTES = DSUB * SUB_KV;
  static constexpr int NSTAGE = (2 * 3 * STAGE_BYTES + Q_BYTES <= 110 * 1024) ? 3 : 2;
  // P (bf16 pairs) overlays the front of S: every S column of a chunk is in registers before P is stored
  static constexpr int TMEM_O = 0, TMEM_S = D, TMEM_P = D;
  static constexpr int TMEM_COLS = (D + NKEY <= 256) ? 256 : 512;
  // Two S buffers where they fit the same allocation (d = 128: 128 + 2 x 64): Q K^T of chunk c + 1 runs under the
  // softmax of chunk c.
  static constexpr int NSBUF = (D + 2 * NKEY <= TMEM_COLS) ? 2 : 1;
  static constexpr int BAR_BYTES = 256;
  static constexpr int SMEM_BYTES = 1024 + Q_BYTES + 2 * NSTAGE * STAGE_BYTES + BAR_BYTES;
  static constexpr int CTAS_PER_SM = (2 * SMEM_BYTES <= 227 * 1024 && TMEM_COLS == 256) ? 2 : 1;
  static_assert(KL % 2 == 1 && KY % 2 == 1 && KX % 2 == 1, "odd windows only (HX even, no pad keys)");
  static_assert(NKEY % 16 == 0 && NKEY <= 128 && HX <= 16, "chunk must fit one UMMA N <= 128");
  static_assert(D == 64 || D == 128, "head_dim 64 or 128");
};

struct TcParams {
  int B, H, L, Y, X;
  int ntl, nty, ntx;
  long long N;
  float scale_log2e;
  unsigned long long* fix;   // fix-up list (common.cuh): rows whose sum left the safe range
};

constexpr int kThreads = 192;

// ------------------------------------------------------------------------------------------------
// Kernel
// ------------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(kThreads, C::CTAS_PER_SM)
na3d_fwd_tc_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                   const __grid_constant__ CUtensorMap tm_v, __nv_bfloat16* __restrict__ o,
                   float* __restrict__ lse, const TcParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t q_smem = base;
  const uint32_t k_smem = q_smem + C::Q_BYTES;
  const uint32_t v_smem = k_smem + C::NSTAGE * C::STAGE_BYTES;
  const uint32_t bars = v_smem + C::NSTAGE * C::STAGE_BYTES;
  // barrier slots (8 bytes each)
  const uint32_t bar_q = bars;
  auto bar_kfull = [&](int s) { return bars + 8u * (1 + s); };
  auto bar_kempty = [&](int s) { return bars + 8u * (1 + C::NSTAGE + s); };
  auto bar_vfull = [&](int s) { return bars + 8u * (1 + 2 * C::NSTAGE + s); };
  auto bar_vempty = [&](int s) { return bars + 8u * (1 + 3 * C::NSTAGE + s); };
  const uint32_t bar_sfull = bars + 8u * (1 + 4 * C::NSTAGE);      // [2] by S buffer
  const uint32_t bar_pfull = bar_sfull + 16;                        // [2]
  // [2] by chunk parity: a softmax warp can be two P V ahead of the last completed one when Q K^T runs a chunk ahead,
  // and one barrier's parity cannot tell phase c - 1 from phase c - 3
  const uint32_t bar_pvdone = bar_sfull + 32;
  const uint32_t tmem_slot = bar_sfull + 48;
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- tile of this CTA: x fastest, then y, level, head, sample (spatial neighbours co-resident)
  int bid = blockIdx.x;
  const int tx = bid % p.ntx; bid /= p.ntx;
  const int ty = bid % p.nty; bid /= p.nty;
  const int tl = bid % p.ntl; bid /= p.ntl;
  const int h = bid % p.H;
  const int b = bid / p.H;
  const int x0 = tx * C::TX, y0 = ty * C::TY, l0 = tl * C::TL;
  // halo box actually reached by the in-grid queries of the tile (A3, inward clamp)
  const int xl = min(x0 + C::TX, p.X) - 1, yl = min(y0 + C::TY, p.Y) - 1, ll = min(l0 + C::TL, p.L) - 1;
  const int hs_x = window_start(x0, C::KX, p.X), hs_y = window_start(y0, C::KY, p.Y), hs_l = window_start(l0, C::KL, p.L);
  const int hy = window_start(yl, C::KY, p.Y) + C::KY - hs_y;      // <= HY
  const int hl = window_start(ll, C::KL, p.L) + C::KL - hs_l;      // <= HL
  (void)xl;
  const int ncy = (hy + C::CY - 1) / C::CY;
  const int nchunks = hl * ncy;

  // ---- one-time setup
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_q); tma_prefetch_desc(&tm_k); tma_prefetch_desc(&tm_v);
    mbar_init(bar_q, 1);
    for (int s = 0; s < C::NSTAGE; ++s) {
      mbar_init(bar_kfull(s), 1); mbar_init(bar_kempty(s), 1);
      mbar_init(bar_vfull(s), 1); mbar_init(bar_vempty(s), 1);
    }
    mbar_init(bar_sfull, 1); mbar_init(bar_sfull + 8, 1);
    mbar_init(bar_pfull, 128); mbar_init(bar_pfull + 8, 128);
    mbar_init(bar_pvdone, 1); mbar_init(bar_pvdone + 8, 1);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, C::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot_ptr;

  if (warp == 0) {
    // =========================== TMA producer ===========================
    // Both control warps run their loops with all 32 lanes in uniform control flow and elect one lane for the TMA /
    // MMA / commit instructions: under `if (lane == 0)` the compiler cannot prove the operands warp-uniform and wraps
    // every tcgen05.mma in an election / uniformisation sequence of ~10 instructions.
    {
      const int bl = b * p.L;
      if (elect_one()) {
        mbar_expect_tx(bar_q, C::Q_BYTES);
        for (int j = 0; j < C::DSUB; ++j) tma_load_5d(q_smem + j * C::SUB_Q, &tm_q, bar_q, 64 * j, h, x0, y0, bl + l0);
      }
      __syncwarp();
      // K loads run one chunk ahead of the V loads: a K stage is released by the QK^T MMA, a V stage only by
      // the PV MMA after the softmax; waiting for V first would hold back the next K chunk
      auto load_v = [&](int c, int pl, int cy) {
        const int s = c % C::NSTAGE;
        const uint32_t ph = (uint32_t)(c / C::NSTAGE) & 1u;
        mbar_wait_bounded(bar_vempty(s), ph ^ 1u);
        if (elect_one()) {
          mbar_expect_tx(bar_vfull(s), C::STAGE_BYTES);
          for (int j = 0; j < C::DSUB; ++j)
            tma_load_5d(v_smem + s * C::STAGE_BYTES + j * C::SUB_KV, &tm_v, bar_vfull(s), 64 * j, h, hs_x,
                        hs_y + cy * C::CY, bl + hs_l + pl);
        }
        __syncwarp();
      };
      int c = 0, ppl = -1, pcy = 0;
      for (int pl = 0; pl < hl; ++pl)
        for (int cy = 0; cy < ncy; ++cy, ++c) {
          const int s = c % C::NSTAGE;
          const uint32_t ph = (uint32_t)(c / C::NSTAGE) & 1u;
          mbar_wait_bounded(bar_kempty(s), ph ^ 1u);
          if (elect_one()) {
            mbar_expect_tx(bar_kfull(s), C::STAGE_BYTES);
            for (int j = 0; j < C::DSUB; ++j)
              tma_load_5d(k_smem + s * C::STAGE_BYTES + j * C::SUB_KV, &tm_k, bar_kfull(s), 64 * j, h, hs_x,
                          hs_y + cy * C::CY, bl + hs_l + pl);
          }
          __syncwarp();
          if (ppl >= 0) load_v(c - 1, ppl, pcy);
          ppl = pl; pcy = cy;
        }
      if (ppl >= 0) load_v(c - 1, ppl, pcy);
    }
  } else if (warp == 1) {
    // =========================== MMA issuer ===========================
    {
      constexpr uint32_t idesc_qk = instr_desc(C::M, C::NKEY, false);
      constexpr uint32_t idesc_pv = instr_desc(C::M, 64, true);
      mbar_wait(bar_q, 0);
      tc_fence_after();
      // chunk c uses S buffer c % NSBUF; barrier phases of a buffer count its uses
      auto issue_qk = [&](int c) {
        const int s = c % C::NSTAGE, sb = c % C::NSBUF;
        const uint32_t ph = (uint32_t)(c / C::NSTAGE) & 1u;
        // ---- S = Qrot Krot^T  (M = 128, N = NKEY, K = D in steps of 16)
        mbar_wait(bar_kfull(s), ph);
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < C::D / 16; ++ks) {
            const uint32_t off = (ks >> 2) * 1u, kin = (ks & 3) * 32u;      // sub-tile, byte offset in the row
            const uint64_t ad = smem_desc(q_smem + off * C::SUB_Q + kin);
            const uint64_t bd = smem_desc(k_smem + s * C::STAGE_BYTES + off * C::SUB_KV + kin);
            umma_ss(tmem + C::TMEM_S + sb * C::NKEY, ad, bd, idesc_qk, ks > 0 ? 1u : 0u);
          }
          umma_commit(bar_kempty(s));
          umma_commit(bar_sfull + 8u * sb);
        }
        __syncwarp();
      };
      // With two buffers Q K^T runs one chunk ahead: buffer (c + 1) % 2 is free once P V of chunk c - 1 (which read
      // its P) has been issued -- the tensor pipe executes in issue order.
      if (nchunks > 0) issue_qk(0);
      for (int c = 0; c < nchunks; ++c) {
        const int s = c % C::NSTAGE, sb = c % C::NSBUF;
        const uint32_t ph = (uint32_t)(c / C::NSTAGE) & 1u;
        if (C::NSBUF == 2 && c + 1 < nchunks) issue_qk(c + 1);
        // ---- O += P V  (M = 128, N = 64 per sub-tile, K = NKEY in steps of 16 keys)
        mbar_wait(bar_pfull + 8u * sb, (uint32_t)(c / C::NSBUF) & 1u);
        mbar_wait(bar_vfull(s), ph);
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < C::NKEY / 16; ++ks) {
#pragma unroll
            for (int j = 0; j < C::DSUB; ++j) {
              const uint64_t bd = smem_desc(v_smem + s * C::STAGE_BYTES + j * C::SUB_KV + ks * 16 * 128);
              umma_ts(tmem + C::TMEM_O + 64 * j, tmem + C::TMEM_P + sb * C::NKEY + 8 * ks, bd, idesc_pv, (c > 0 || ks > 0) ? 1u : 0u);
            }
          }
          umma_commit(bar_vempty(s));
          umma_commit(bar_pvdone + 8u * (c & 1));
        }
        __syncwarp();
        if (C::NSBUF == 1 && c + 1 < nchunks) issue_qk(c + 1);
      }
    }
  } else {
    // =========================== softmax + epilogue ===========================
    const int sp = warp & 3;                       // TMEM subpartition of this warp
    const int row = sp * 32 + lane;                // query row of the tile == TMEM lane
    const uint32_t lane_addr = (uint32_t)(sp * 32) << 16;
    const int qx = row & 7, qy = (row >> 3) & 7, ql = row >> 6;
    const bool active = (x0 + qx < p.X) && (y0 + qy < p.Y) && (l0 + ql < p.L);
    const int ax = min(x0 + qx, p.X - 1), ay = min(y0 + qy, p.Y - 1), al = min(l0 + ql, p.L - 1);
    // window of this query relative to the halo box
    const int lo_x = window_start(ax, C::KX, p.X) - hs_x;
    const int lo_y = window_start(ay, C::KY, p.Y) - hs_y;
    const int lo_l = window_start(al, C::KL, p.L) - hs_l;
    float xbias[C::HX];
#pragma unroll
    for (int j = 0; j < C::HX; ++j) xbias[j] = (j >= lo_x && j < lo_x + C::KX) ? 0.f : -INFINITY;
    // key rows / planes any query of this warp needs (warp-uniform skip ranges)
    const int wy_lo = __reduce_min_sync(0xffffffffu, lo_y), wy_hi = __reduce_max_sync(0xffffffffu, lo_y + C::KY);
    const int wl_lo = __reduce_min_sync(0xffffffffu, lo_l), wl_hi = __reduce_max_sync(0xffffffffu, lo_l + C::KL);

    float lsum = 0.f;
    const float cs = p.scale_log2e;
    int c = 0;
    for (int pl = 0; pl < hl; ++pl) {
      const bool plane_needed = pl >= wl_lo && pl < wl_hi;
      const bool plane_ok = pl >= lo_l && pl < lo_l + C::KL;
      for (int cy = 0; cy < ncy; ++cy, ++c) {
        const int sb = c % C::NSBUF;
        const uint32_t s_tm = tmem + lane_addr + C::TMEM_S + sb * C::NKEY;       // S of the chunk; P goes over its front
        mbar_wait(bar_sfull + 8u * sb, (uint32_t)(c / C::NSBUF) & 1u);
        tc_fence_after();
        uint32_t pw[C::NKEY / 2];
        float csum = 0.f;
        // No running maximum and no rescale of O: P = 2^(s scale log2 e) as in the fused forward (R19).  The epilogue
        // checks the row sum and lists the row for the two-pass fix-up kernel if it left the safe range.
#pragma unroll
        for (int r = 0; r < C::CY; ++r) {
          const int py = cy * C::CY + r;
          if (plane_needed && py >= wy_lo && py < wy_hi) {
            float sv[16];
            tmem_ld16(s_tm + r * C::HX, sv);
            tmem_wait_ld();
            const bool rowok = plane_ok && py >= lo_y && py < lo_y + C::KY;
            const float nb = rowok ? 0.f : -INFINITY;
            float rsum = 0.f;
#pragma unroll
            for (int j = 0; j < C::HX; j += 2) {
              const float p0 = ex2(fmaf(sv[j], cs, xbias[j]) + nb), p1 = ex2(fmaf(sv[j + 1], cs, xbias[j + 1]) + nb);
              rsum += p0 + p1;
              pw[(r * C::HX + j) >> 1] = pack_bf16(p0, p1);
            }
            csum += rsum;
          } else {
#pragma unroll
            for (int j = 0; j < C::HX; j += 2) pw[(r * C::HX + j) >> 1] = 0u;
          }
        }
        lsum += csum;
        // P (bf16 pairs) -> TMEM, then hand the chunk to MMA2
#pragma unroll
        for (int j = 0; j < C::NKEY / 2; j += 8) tmem_st8(s_tm + j, &pw[j]);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bar_pfull + 8u * sb);
      }
    }
    // ---- epilogue: O / l -> bf16 -> global, LSE
    mbar_wait_bounded(bar_pvdone + 8u * ((nchunks - 1) & 1), (uint32_t)((nchunks - 1) >> 1) & 1u);
    tc_fence_after();
    const float inv = 1.f / lsum;
    const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
    __nv_bfloat16* orow = o + (((long long)b * p.N + tok) * p.H + h) * C::D;
#pragma unroll
    for (int j = 0; j < C::D; j += 16) {
      float ov[16];
      tmem_ld16(tmem + lane_addr + C::TMEM_O + j, ov);
      tmem_wait_ld();
      if (active) {
        uint4 w0, w1;
        w0.x = pack_bf16(ov[0] * inv, ov[1] * inv);   w0.y = pack_bf16(ov[2] * inv, ov[3] * inv);
        w0.z = pack_bf16(ov[4] * inv, ov[5] * inv);   w0.w = pack_bf16(ov[6] * inv, ov[7] * inv);
        w1.x = pack_bf16(ov[8] * inv, ov[9] * inv);   w1.y = pack_bf16(ov[10] * inv, ov[11] * inv);
        w1.z = pack_bf16(ov[12] * inv, ov[13] * inv); w1.w = pack_bf16(ov[14] * inv, ov[15] * inv);
        reinterpret_cast<uint4*>(orow + j)[0] = w0;
        reinterpret_cast<uint4*>(orow + j)[1] = w1;
      }
    }
    if (active) {
      const long long rid = ((long long)b * p.H + h) * p.N + tok;
      lse[rid] = log2f(lsum) * 0.69314718055994531f;
      if (!(lsum < kRowSumMax && lsum > kRowSumMin)) {        // out of the safe range (or NaN): the fix-up kernel recomputes the row
        const unsigned long long idx = atomicAdd(p.fix, 1ull);
        if (idx < kFixCap) p.fix[2 + idx] = (unsigned long long)rid;
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

// ------------------------------------------------------------------------------------------------
// Host side: tensor maps + launch
// ------------------------------------------------------------------------------------------------
DeviceState g_states[64];
std::mutex g_mu;

template <class C>
cudaError_t launch_cfg(int slot, const Problem& p, const void* qr, const void* kr, const void* v, void* o, float* lse,
                       void* fix, cudaStream_t stream, int* launches) {
  CUtensorMap tq, tk, tv;
  if (!make_map(&tq, qr, p, C::TX, C::TY, C::TL) || !make_map(&tk, kr, p, C::HX, C::CY, 1) ||
      !make_map(&tv, v, p, C::HX, C::CY, 1))
    return cudaErrorInvalidValue;
  TcParams tp;
  tp.B = p.B; tp.H = p.H; tp.L = p.L; tp.Y = p.Y; tp.X = p.X; tp.N = p.N;
  tp.ntl = (p.L + C::TL - 1) / C::TL; tp.nty = (p.Y + C::TY - 1) / C::TY; tp.ntx = (p.X + C::TX - 1) / C::TX;
  tp.scale_log2e = p.scale * 1.4426950408889634f;
  tp.fix = reinterpret_cast<unsigned long long*>(fix);
  const long long grid = (long long)p.B * p.H * tp.ntl * tp.nty * tp.ntx;
  if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  DeviceState* ds = device_state(g_states, g_mu);
  if (!ds) return cudaErrorInvalidDevice;
  cudaError_t e = ensure_smem_attr(ds, g_mu, slot, na3d_fwd_tc_kernel<C>, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(fix, 0, 16, stream);
  if (e != cudaSuccess) return e;
  prof_begin("na3d_fwd_tcgen05", stream);
  na3d_fwd_tc_kernel<C><<<(unsigned)grid, kThreads, C::SMEM_BYTES, stream>>>(tq, tk, tv, (__nv_bfloat16*)o, lse, tp);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace

// Shapes the tensor-core path covers: bf16, head_dim 64 / 128, the window sizes instantiated below.
#define STRATA_TC_CONFIGS(X) \
  X(0, 64, 3, 7, 7)          \
  X(1, 128, 5, 9, 9)         \
  X(2, 64, 3, 5, 5)          \
  X(3, 64, 3, 3, 3)          \
  X(4, 64, 9, 9, 9)         \
  X(5, 128, 9, 9, 9)

bool tc_fwd_supported(const Problem& p) {
  if (p.dtype != 1) return false;
#define X(I_, D_, KL_, KY_, KX_) \
  if (p.D == D_ && p.kL == KL_ && p.kY == KY_ && p.kX == KX_) return true;
  STRATA_TC_CONFIGS(X)
#undef X
  return false;
}

cudaError_t launch_fwd_tc(const Problem& p, const void* qr, const void* kr, const void* v, void* o,
                          float* lse, void* fix, cudaStream_t stream, int* launches) {
#define X(I_, D_, KL_, KY_, KX_)                                           \
  if (p.D == D_ && p.kL == KL_ && p.kY == KY_ && p.kX == KX_)               \
    return launch_cfg<Cfg<D_, KL_, KY_, KX_>>(I_, p, qr, kr, v, o, lse, fix, stream, launches);
  STRATA_TC_CONFIGS(X)
#undef X
  return cudaErrorNotSupported;
}

}  // namespace strata
