// na3d_tc_fwd_sweep.cu -- "L-sweep" tcgen05 forward for head_dim 64 and level window k_L = 3.
//
// Steps A3-A6 of DESIGN.md on pre-rotated bf16 operands.  One CTA owns a whole level COLUMN of the
// token grid: the 8 x 8 (y, x) patch of every level, i.e. ceil(L/2) query tiles of 2 x 8 x 8 = 128
// queries.  The key/value planes of the column's halo ((8+kY-1) x (8+kX-1) keys per level) are
// streamed through shared memory ONCE, level by level, in parts of CY key rows; each part is
// multiplied against the (at most two) query tiles whose clamped level windows reach that plane.
// Compared with one tile per CTA this halves the L2 -> SM traffic of K and V.
//
// Two independent tile pipelines ("slots") run inside the CTA: slot s owns tiles s, s+2, ...
// Each slot has its own MMA issuer thread, its own softmax warpgroup (128 threads = 128 query
// rows) and its own 256 TMEM columns: O [0,64) fp32 | S0 [64,160) | S1 [160,256) -- S is double
// buffered (QK^T of item i+1 runs while the softmax of item i is in flight) and P (bf16) is
// written over the front of the S buffer it came from (A operand of the PV MMA, read from TMEM).
// The slots share only the K/V stage ring (each stage is released by both slots).
//
// Warps (384 threads): 0 = K/V TMA producer, 1 / 2 = MMA issuer of slot 0 / 1 (they also issue the
// TMA loads of their Q tiles), 3 = TMEM owner, 4-7 = softmax of slot 0, 8-11 = softmax of slot 1.
#include "tc_common.cuh"

namespace strata {
namespace {

using namespace tc;

template <int KY_, int KX_, int CY_>
struct SweepCfg {
  static constexpr int D = 64, KL = 3, KY = KY_, KX = KX_;
  static constexpr int TL = 2, TY = 8, TX = 8, M = 128;
  static constexpr int HY = TY + KY - 1, HX = TX + KX - 1;
  static constexpr int CY = CY_;                                   // key rows per part
  static constexpr int NPARTS = (HY + CY - 1) / CY;
  static constexpr int TAIL = HY - (NPARTS - 1) * CY;              // rows of the last part
  static constexpr int NMAX = (CY * HX + 15) / 16 * 16;            // UMMA N of a full part
  static constexpr int STAGE_BYTES = NMAX * 128;
  static constexpr int NSTAGE = 5;
  static constexpr int Q_BYTES = M * 128;
  static constexpr int TMEM_SLOT = 256, TMEM_O = 0, TMEM_S = 64, TMEM_SSTRIDE = 96;
  static constexpr int NBARS = 4 * NSTAGE + 2 * 8;
  static constexpr int SMEM_BYTES = 1024 + 4 * Q_BYTES + 2 * NSTAGE * STAGE_BYTES + 8 * NBARS + 16;
  static_assert(KY % 2 == 1 && KX % 2 == 1, "odd windows only (HX even)");
  static_assert(NMAX <= 96 && HX <= 16, "a part must fit one S buffer");
  static_assert((CY - 1) * HX + 16 <= TMEM_SSTRIDE, "row loads stay inside the S buffer");
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct SweepParams {
  int B, H, L, Y, X;
  int nty, ntx;
  long long N;
  float scale_log2e;
};

constexpr int kSweepThreads = 384;
constexpr float kUp = 8.f, kDown = 16.f;   // lazy reference-maximum update thresholds (log2 units)

__device__ __forceinline__ void tmem_ld16_issue(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr) : "memory");
}
// wait::ld with the loaded registers as in/out operands: no use of them can be scheduled above it.
__device__ __forceinline__ void tmem_ld16_wait(uint32_t (&r)[16]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                 "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
               :: "memory");
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
  float d;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}

// Level planes [lo, hi) the windows of tile t (levels 2t, 2t+1) reach (A3 with k_L = 3).
__device__ __host__ inline int tile_plo(int t, int L) { return window_start(2 * t, 3, L); }
__device__ __host__ inline int tile_phi(int t, int L) { return window_start(min(2 * t + 1, L - 1), 3, L) + 3; }

// Position of one slot in the global chunk stream (plane-major, part-minor).
struct SlotWalk {
  int t;   // current tile of the slot
  __device__ __forceinline__ void classify(int plane, int part, int nparts, int ntl, int L, bool& needed,
                                           bool& first, bool& last) {
    while (t < ntl && plane >= tile_phi(t, L)) t += 2;
    needed = t < ntl && plane >= tile_plo(t, L);
    first = needed && plane == tile_plo(t, L) && part == 0;
    last = needed && plane == tile_phi(t, L) - 1 && part == nparts - 1;
  }
};

template <class C>
__global__ void __launch_bounds__(kSweepThreads, 1)
na3d_fwd_sweep_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                      const __grid_constant__ CUtensorMap tm_kt, const __grid_constant__ CUtensorMap tm_v,
                      const __grid_constant__ CUtensorMap tm_vt, __nv_bfloat16* __restrict__ o,
                      float* __restrict__ lse, const SweepParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t q_smem = base;                                   // [slot][buf] x Q_BYTES
  const uint32_t k_smem = q_smem + 4 * C::Q_BYTES;
  const uint32_t v_smem = k_smem + C::NSTAGE * C::STAGE_BYTES;
  const uint32_t bars = v_smem + C::NSTAGE * C::STAGE_BYTES;
  auto bar_kfull = [&](int s) { return bars + 8u * s; };
  auto bar_kempty = [&](int s) { return bars + 8u * (C::NSTAGE + s); };
  auto bar_vfull = [&](int s) { return bars + 8u * (2 * C::NSTAGE + s); };
  auto bar_vempty = [&](int s) { return bars + 8u * (3 * C::NSTAGE + s); };
  auto bar_slot = [&](int slot, int which) { return bars + 8u * (4 * C::NSTAGE + 8 * slot + which); };
  // per slot: 0,1 = qfull[buf]   2,3 = sfull[buf]   4,5 = pfull[buf]   6,7 = pvdone[buf]
  // Every barrier that is not waited on in every phase is split by item parity: a waiter may only
  // test the parity of a phase when the barrier is known to be in that phase or the next one.
  const uint32_t tmem_word = bars + 8u * C::NBARS;
  uint32_t* tmem_word_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_word - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- the level column of this CTA: x fastest, then y, head, sample
  int bid = blockIdx.x;
  const int tx = bid % p.ntx; bid /= p.ntx;
  const int ty = bid % p.nty; bid /= p.nty;
  const int h = bid % p.H;
  const int b = bid / p.H;
  const int x0 = tx * C::TX, y0 = ty * C::TY;
  const int yl = min(y0 + C::TY, p.Y) - 1;
  const int hs_x = window_start(x0, C::KX, p.X), hs_y = window_start(y0, C::KY, p.Y);
  const int hy = window_start(yl, C::KY, p.Y) + C::KY - hs_y;     // key rows of the halo, <= HY
  const int nparts = (hy + C::CY - 1) / C::CY;
  const int ntl = (p.L + 1) / 2;
  const int nchunks = p.L * nparts;
  const int bl = b * p.L;

  // ---- one-time setup
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_q); tma_prefetch_desc(&tm_k); tma_prefetch_desc(&tm_kt);
    tma_prefetch_desc(&tm_v); tma_prefetch_desc(&tm_vt);
    for (int s = 0; s < C::NSTAGE; ++s) {
      mbar_init(bar_kfull(s), 1); mbar_init(bar_kempty(s), 2);
      mbar_init(bar_vfull(s), 1); mbar_init(bar_vempty(s), 2);
    }
    for (int slot = 0; slot < 2; ++slot) {
      mbar_init(bar_slot(slot, 0), 1); mbar_init(bar_slot(slot, 1), 1);
      mbar_init(bar_slot(slot, 2), 1); mbar_init(bar_slot(slot, 3), 1);
      mbar_init(bar_slot(slot, 4), 128); mbar_init(bar_slot(slot, 5), 128);
      mbar_init(bar_slot(slot, 6), 1); mbar_init(bar_slot(slot, 7), 1);
    }
    fence_barrier_init();
  }
  if (warp == 3) tmem_alloc(tmem_word, 512);
  // V stages start as zeros: rows of a stage that a (shorter) part does not overwrite are multiplied
  // by P = 0 in the PV MMA and must therefore hold finite numbers.
  for (uint32_t off = threadIdx.x * 16u; off < (uint32_t)(C::NSTAGE * C::STAGE_BYTES); off += kSweepThreads * 16u)
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(v_smem + off), "r"(0u) : "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_word_ptr;

  if (warp == 0) {
    // =========================== K/V TMA producer ===========================
    if (lane == 0) {
      int g = 0;
      for (int plane = 0; plane < p.L; ++plane)
        for (int part = 0; part < nparts; ++part, ++g) {
          const int s = g % C::NSTAGE;
          const uint32_t ph = (uint32_t)(g / C::NSTAGE) & 1u;
          const int nrows = min(C::CY, hy - part * C::CY);
          const bool tail = (C::TAIL < C::CY) && nrows <= C::TAIL;
          const uint32_t bytes = (uint32_t)((tail ? C::TAIL : C::CY) * C::HX * 128);
          mbar_wait(bar_kempty(s), ph ^ 1u);
          mbar_expect_tx(bar_kfull(s), bytes);
          tma_load_5d(k_smem + s * C::STAGE_BYTES, tail ? &tm_kt : &tm_k, bar_kfull(s), 0, h, hs_x, hs_y + part * C::CY, bl + plane);
          mbar_wait(bar_vempty(s), ph ^ 1u);
          mbar_expect_tx(bar_vfull(s), bytes);
          tma_load_5d(v_smem + s * C::STAGE_BYTES, tail ? &tm_vt : &tm_v, bar_vfull(s), 0, h, hs_x, hs_y + part * C::CY, bl + plane);
        }
    }
  } else if (warp == 1 || warp == 2) {
    // =========================== MMA issuer of one slot ===========================
    if (lane == 0) {
      const int slot = warp - 1;
      const uint32_t tm = tmem + slot * C::TMEM_SLOT;
      constexpr uint32_t idesc_pv = instr_desc(C::M, 64, true);
      auto issue_q = [&](int nseq, int tile) {
        const uint32_t bar = bar_slot(slot, nseq & 1);
        mbar_expect_tx(bar, C::Q_BYTES);
        tma_load_5d(q_smem + (slot * 2 + (nseq & 1)) * C::Q_BYTES, &tm_q, bar, 0, h, x0, y0, bl + 2 * tile);
      };
      for (int n = 0; n < 2; ++n)
        if (slot + 2 * n < ntl) issue_q(n, slot + 2 * n);

      struct Pending { int i, g, stage, n, nseq, tile; uint32_t ph; bool first, last; };
      Pending prev{};
      bool have_prev = false;
      auto issue_mma2 = [&](const Pending& it) {
        mbar_wait(bar_slot(slot, 4 + (it.i & 1)), (uint32_t)(it.i >> 1) & 1u);   // P of item i is in TMEM
        mbar_wait(bar_vfull(it.stage), it.ph);
        tc_fence_after();
        const uint32_t a_tmem = tm + C::TMEM_S + (it.i & 1) * C::TMEM_SSTRIDE;
        for (int ks = 0; ks < it.n / 16; ++ks) {
          const uint64_t bd = smem_desc(v_smem + it.stage * C::STAGE_BYTES + ks * 16 * 128);
          umma_ts(tm + C::TMEM_O, a_tmem + 8 * ks, bd, idesc_pv, (!it.first || ks > 0) ? 1u : 0u);
        }
        umma_commit(bar_vempty(it.stage));
        umma_commit(bar_slot(slot, 6 + (it.i & 1)));
        // all QK^T MMAs of this tile have completed (its last softmax ran): its Q buffer is free
        if (it.last && it.tile + 4 < ntl) issue_q(it.nseq + 2, it.tile + 4);
      };

      SlotWalk walk{slot};
      int i = 0, g = 0;
      for (int plane = 0; plane < p.L; ++plane)
        for (int part = 0; part < nparts; ++part, ++g) {
          bool needed, first, last;
          walk.classify(plane, part, nparts, ntl, p.L, needed, first, last);
          const int s = g % C::NSTAGE;
          const uint32_t ph = (uint32_t)(g / C::NSTAGE) & 1u;
          if (!needed) {       // this slot does not use the chunk: release it once it has landed (one
            mbar_wait(bar_kfull(s), ph);      // arrival per slot and phase, never ahead of the producer)
            mbar_arrive(bar_kempty(s));
            mbar_wait(bar_vfull(s), ph);
            mbar_arrive(bar_vempty(s));
            continue;
          }
          // never hold a V stage across a gap that could stall the producer (deadlock guard)
          if (have_prev && g - prev.g >= C::NSTAGE - 1) { issue_mma2(prev); have_prev = false; }
          const int nseq = (walk.t - slot) >> 1;
          if (first) mbar_wait(bar_slot(slot, nseq & 1), (uint32_t)(nseq >> 1) & 1u);
          mbar_wait(bar_kfull(s), ph);
          tc_fence_after();
          const int nrows = min(C::CY, hy - part * C::CY);
          const int n = (nrows * C::HX + 15) / 16 * 16;
          const uint32_t idesc_qk = instr_desc(C::M, n, false);
          const uint32_t qb = q_smem + (slot * 2 + (nseq & 1)) * C::Q_BYTES;
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            umma_ss(tm + C::TMEM_S + (i & 1) * C::TMEM_SSTRIDE, smem_desc(qb + ks * 32),
                    smem_desc(k_smem + s * C::STAGE_BYTES + ks * 32), idesc_qk, ks > 0 ? 1u : 0u);
          umma_commit(bar_kempty(s));
          umma_commit(bar_slot(slot, 2 + (i & 1)));
          if (have_prev) issue_mma2(prev);
          prev = Pending{i, g, s, n, nseq, walk.t, ph, first, last};
          have_prev = true;
          ++i;
        }
      if (have_prev) issue_mma2(prev);
    }
  } else if (warp >= 4) {
    // =========================== softmax + epilogue of one slot ===========================
    const int slot = (warp - 4) >> 2;
    const int sp = warp & 3;                       // TMEM subpartition
    const int row = sp * 32 + lane;                // query row of the tile == TMEM lane
    const uint32_t tm = tmem + slot * C::TMEM_SLOT + ((uint32_t)(sp * 32) << 16);
    const int qx = row & 7, qy = (row >> 3) & 7, ql = row >> 6;
    const int ax = min(x0 + qx, p.X - 1), ay = min(y0 + qy, p.Y - 1);
    const bool active_xy = (x0 + qx < p.X) && (y0 + qy < p.Y);
    const int lo_x = window_start(ax, C::KX, p.X) - hs_x;
    const int lo_y = window_start(ay, C::KY, p.Y) - hs_y;
    float xbias[C::HX], xb[C::HX];
#pragma unroll
    for (int j = 0; j < C::HX; ++j) xbias[j] = (j >= lo_x && j < lo_x + C::KX) ? 0.f : -INFINITY;
    const int wy_lo = __reduce_min_sync(0xffffffffu, lo_y), wy_hi = __reduce_max_sync(0xffffffffu, lo_y + C::KY);
    const float cs = p.scale_log2e;

    int i = 0;
    for (int tile = slot; tile < ntl; tile += 2) {
      const int al = min(2 * tile + ql, p.L - 1);
      const bool active = active_xy && (2 * tile + ql < p.L);
      const int pw_lo = window_start(al, 3, p.L);                  // planes of this query: [pw_lo, pw_lo+3)
      const int wl_lo = __reduce_min_sync(0xffffffffu, pw_lo), wl_hi = __reduce_max_sync(0xffffffffu, pw_lo + 3);
      float m_ref = 0.f, lsum = 0.f, run_max = -INFINITY;
#pragma unroll
      for (int j = 0; j < C::HX; ++j) xb[j] = xbias[j];
      const int plo = tile_plo(tile, p.L), phi = tile_phi(tile, p.L);
      for (int plane = plo; plane < phi; ++plane) {
        const bool plane_needed = plane >= wl_lo && plane < wl_hi;
        const bool plane_ok = plane >= pw_lo && plane < pw_lo + 3;
        for (int part = 0; part < nparts; ++part, ++i) {
          const int nrows = min(C::CY, hy - part * C::CY);
          const int nwords = ((nrows * C::HX + 15) / 16 * 16) / 2;
          const int r_base = part * C::CY;
          const uint32_t s_addr = tm + C::TMEM_S + (i & 1) * C::TMEM_SSTRIDE;
          const bool first_item = (plane == plo && part == 0);
          mbar_wait(bar_slot(slot, 2 + (i & 1)), (uint32_t)(i >> 1) & 1u);
          tc_fence_after();
          uint32_t pw[C::NMAX / 2];
          float csum = 0.f;
          for (int attempt = 0; attempt < 2; ++attempt) {
            float cmax = -INFINITY;
            csum = 0.f;
            uint32_t sva[16], svb[16];
            auto needed = [&](int r) {
              return plane_needed && r < nrows && r_base + r >= wy_lo && r_base + r < wy_hi;
            };
            if (needed(0)) tmem_ld16_issue(s_addr, sva);
#pragma unroll
            for (int r = 0; r < C::CY; ++r) {
              uint32_t (&cur)[16] = (r & 1) ? svb : sva;
              uint32_t (&nxt)[16] = (r & 1) ? sva : svb;
              const bool need_r = needed(r);
              if (need_r) tmem_ld16_wait(cur);
              if (r + 1 < C::CY && needed(r + 1)) tmem_ld16_issue(s_addr + (r + 1) * C::HX, nxt);
              if (need_r) {
                const int py = r_base + r;
                const bool rowok = plane_ok && py >= lo_y && py < lo_y + C::KY;
                float t[C::HX];
#pragma unroll
                for (int j = 0; j < C::HX; ++j) t[j] = fmaf(__uint_as_float(cur[j]), cs, xb[j]);
                float rmax = fmaxf(t[0], t[1]);
#pragma unroll
                for (int j = 2; j < C::HX; j += 2) rmax = fmax3(rmax, t[j], t[j + 1]);
                if (rowok) cmax = fmaxf(cmax, rmax);
                float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
                for (int j = 0; j < C::HX; j += 2) {
                  const float p0 = ex2(t[j]), p1 = ex2(t[j + 1]);
                  rs0 += p0; rs1 += p1;
                  const uint32_t w = pack_bf16(p0, p1);
                  pw[(r * C::HX + j) >> 1] = rowok ? w : 0u;
                }
                csum += rowok ? (rs0 + rs1) : 0.f;
              } else {
#pragma unroll
                for (int j = 0; j < C::HX; j += 2) pw[(r * C::HX + j) >> 1] = 0u;
              }
            }
            // the pass used the current reference maximum; move it and redo the chunk if it is off
            const float amax = fmaxf(run_max, cmax + m_ref);                 // absolute maximum so far
            const bool need = (cmax > kUp) || (amax > -INFINITY && amax < m_ref - kDown);
            if (attempt == 0 && __any_sync(0xffffffffu, need)) {
              const float alpha = need ? ex2(m_ref - amax) : 1.f;
              if (!first_item) {                     // O holds earlier chunks of this tile: rescale its rows
                mbar_wait(bar_slot(slot, 6 + ((i - 1) & 1)), (uint32_t)((i - 1) >> 1) & 1u);
                tc_fence_after();
#pragma unroll
                for (int j = 0; j < C::D; j += 16) {
                  float ov[16];
                  tmem_ld16(tm + C::TMEM_O + j, ov);
                  tmem_wait_ld();
                  uint32_t ow[16];
#pragma unroll
                  for (int u = 0; u < 16; ++u) ow[u] = __float_as_uint(ov[u] * alpha);
                  tmem_st16(tm + C::TMEM_O + j, ow);
                }
                tmem_wait_st();
              }
              lsum *= alpha;
              if (need) {
                m_ref = amax;
#pragma unroll
                for (int j = 0; j < C::HX; ++j) xb[j] = xbias[j] - m_ref;
              }
              continue;
            }
            run_max = amax;
            break;
          }
          lsum += csum;
#pragma unroll
          for (int j = C::CY * C::HX / 2; j < C::NMAX / 2; ++j) pw[j] = 0u;    // pad keys of a full part
          // P (bf16 pairs) over the front of the S buffer, then hand the item to the PV MMA
#pragma unroll
          for (int j = 0; j < C::NMAX / 2; j += 8)
            if (j < nwords) tmem_st8(s_addr + j, &pw[j]);
          tmem_wait_st();
          tc_fence_before();
          mbar_arrive(bar_slot(slot, 4 + (i & 1)));
        }
      }
      // ---- tile epilogue: O / l -> bf16 -> global, LSE
      mbar_wait(bar_slot(slot, 6 + ((i - 1) & 1)), (uint32_t)((i - 1) >> 1) & 1u);
      tc_fence_after();
      const float inv = 1.f / lsum;
      const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
      __nv_bfloat16* orow = o + (((long long)b * p.N + tok) * p.H + h) * C::D;
#pragma unroll
      for (int j = 0; j < C::D; j += 16) {
        float ov[16];
        tmem_ld16(tm + C::TMEM_O + j, ov);
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
      if (active) lse[((long long)b * p.H + h) * p.N + tok] = (m_ref + log2f(lsum)) * 0.69314718055994531f;
      // the O reads above must be complete before the next tile's first PV MMA overwrites O: that MMA
      // waits for this warpgroup's next p_full arrival, which follows these (waited-for) loads.
    }
  }

  // ---- teardown
  tc_fence_before();
  __syncthreads();
  if (warp == 3) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

template <class C>
cudaError_t launch_sweep(const Problem& p, const void* qr, const void* kr, const void* v, void* o, float* lse,
                         cudaStream_t stream, int* launches) {
  CUtensorMap tq, tk, tkt, tv, tvt;
  if (!make_map(&tq, qr, p, C::TX, C::TY, C::TL) || !make_map(&tk, kr, p, C::HX, C::CY, 1) ||
      !make_map(&tkt, kr, p, C::HX, C::TAIL, 1) || !make_map(&tv, v, p, C::HX, C::CY, 1) ||
      !make_map(&tvt, v, p, C::HX, C::TAIL, 1))
    return cudaErrorInvalidValue;
  SweepParams sp;
  sp.B = p.B; sp.H = p.H; sp.L = p.L; sp.Y = p.Y; sp.X = p.X; sp.N = p.N;
  sp.nty = (p.Y + C::TY - 1) / C::TY; sp.ntx = (p.X + C::TX - 1) / C::TX;
  sp.scale_log2e = p.scale * 1.4426950408889634f;
  const long long grid = (long long)p.B * p.H * sp.nty * sp.ntx;
  if (grid > 0x7fffffffLL) return cudaErrorInvalidValue;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(na3d_fwd_sweep_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  prof_begin("na3d_fwd_tcgen05_sweep", stream);
  na3d_fwd_sweep_kernel<C><<<(unsigned)grid, kSweepThreads, C::SMEM_BYTES, stream>>>(tq, tk, tkt, tv, tvt,
                                                                                 (__nv_bfloat16*)o, lse, sp);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace

// (kY, kX, CY) instantiations of the sweep kernel (head_dim 64, k_L = 3).
#define STRATA_SWEEP_CONFIGS(X) \
  X(7, 7, 5)                    \
  X(5, 5, 6)                    \
  X(3, 3, 5)

bool tc_sweep_supported(const Problem& p) {
  if (p.dtype != 1 || p.D != 64 || p.kL != 3) return false;
  bool inst = false;
#define X(KY_, KX_, CY_) \
  if (p.kY == KY_ && p.kX == KX_) inst = true;
  STRATA_SWEEP_CONFIGS(X)
#undef X
  if (!inst) return false;
  // the tiles of one slot must reach disjoint, increasing plane ranges (one pass over the levels)
  const int ntl = (p.L + 1) / 2;
  for (int t = 0; t + 2 < ntl; ++t)
    if (tile_plo(t + 2, p.L) < tile_phi(t, p.L)) return false;
  return true;
}

cudaError_t launch_fwd_sweep(const Problem& p, const void* qr, const void* kr, const void* v, void* o,
                             float* lse, cudaStream_t stream, int* launches) {
#define X(KY_, KX_, CY_)                 \
  if (p.kY == KY_ && p.kX == KX_)       \
    return launch_sweep<SweepCfg<KY_, KX_, CY_>>(p, qr, kr, v, o, lse, stream, launches);
  STRATA_SWEEP_CONFIGS(X)
#undef X
  return cudaErrorNotSupported;
}

}  // namespace strata
