// na3d_fwd_fused.cu -- fused StereoRoPE + 3D neighbourhood attention forward (tcgen05 / TMEM / TMA).
//
// Steps A2-A6 of DESIGN.md in ONE kernel (A1, the per-token cos/sin table, is rope.cu's small
// pre-kernel): Q and K arrive un-rotated, are rotated in registers by a dedicated warpgroup and go
// to the tensor cores from shared memory; the rotated copies never touch HBM.
//
// Work decomposition ("level sweep"): persistent CTAs, one per SM; CTA c takes the level COLUMNS c,
// c + gridDim.x, ... and every pipeline counter runs on across columns, so the loads, rotations and MMAs
// of the next column start while the previous one drains.  A level column of one (sample, head) is the
// TY x TX patch of every level, i.e. ceil(L / TL) query tiles of TL x TY x TX = 128 queries.  The
// key / value planes of the column's halo ((TY+kY-1) x (TX+kX-1) keys per level) stream through
// shared memory ONCE, level by level, in three parts of key rows ([0, G), [G, G+kY-1), [G+kY-1, HY)
// with G = 32 / TX query rows per softmax warp, so that away from the grid border a warp needs either
// every row of a part or none); every part is multiplied against the (at most two) query tiles
// whose clamped level windows (R1) reach its plane.
// Two independent tile pipelines ("slots") run inside the CTA: slot s owns tiles s, s+2, ...
// (their plane ranges are disjoint and increasing, checked on the host).  Each slot has its own MMA
// issuer thread, its own softmax warpgroup (one query row per thread = one TMEM lane) and 256 TMEM
// columns: O [0, D) fp32 | S0 | S1 (S is double buffered; P (bf16) is written over the front of the
// S buffer it came from and is the TMEM A-operand of the PV MMA).
//
// Warps (512 threads):
//   0-3    softmax + epilogue of slot 0        4-7   softmax + epilogue of slot 1
//   8-11   rotation warpgroup: rotates every K part IN PLACE in shared memory (the Q tile of a slot is
//          rotated the same way by that slot's softmax warpgroup, between two tiles)
//          (packed bf16x2 multiply-adds against the bf16 cos/sin table), then hands them to the MMA
//          issuers.  For the interleaved pairing the two halves of a pair are first gathered into
//          separate words and the rotated words are stored in that order: the same permutation of
//          the 8 channels of every 16-byte chunk is applied to Q and K, which leaves Q K^T unchanged.
//   12     TMA producer: K + rotary-table + V parts into a stage ring (the K loads run two parts ahead
//          of the V loads: a V stage is released by the PV MMA, long after the K stage of the same
//          part); Q tiles + their table rows; TMEM owner
//   13     QK^T issuer of both slots          14, 15   PV issuer of slot 0 / 1
//          (whole warp in uniform control flow, one elected lane issues; the QK^T issuer re-uses
//          an S buffer once the PV MMA that reads its P has been ISSUED: the tensor pipe executes in
//          issue order)
// Register budget via setmaxnreg: 184 / 184 / 88 / 56 per thread for the four warpgroups.
//
// Softmax: a thread (= query row) takes the whole S part (R key rows x HX columns) into registers with
// one batch of tcgen05.ld, and everything up to the P store is branch-free.  exp2 with a LAZY
// reference maximum -- the row maximum is computed only for the first part that holds a valid key
// of the row and when the part's sum overflows 2^40 (checked once per part, before P is stored).
// The x window of a query covers kX of the HX halo columns; with kX <= HX/2 at most one of the
// columns c and c + HX/2 is inside it, so the two halves of every key row are FOLDED with a
// per-thread bit select before the exponential (half the MUFU work); P is packed to bf16 folded and
// un-folded by one byte permute per output word (a masked slot replicates the zero sign bit).
#include <cstdlib>
#include <type_traits>

// 16 warps poll mbarriers here; a short sleep between polls leaves the issue slots to the working warps
// (measured on config 3: 8.05 ms without, 7.96 / 7.86 / 7.92 ms with 50 / 150 / 400 ns).
#define STRATA_WAIT_SLEEP_NS 150
#include "tc_common.cuh"

namespace strata {
namespace {

using namespace tc;

template <int D_, int KL_, int KY_, int KX_, int TL_, int TY_, int TX_, int NS_>
struct FusedCfg {
  static constexpr int D = D_, KL = KL_, KY = KY_, KX = KX_;
  static constexpr int TL = TL_, TY = TY_, TX = TX_, M = 128;
  static constexpr int HY = TY + KY - 1, HX = TX + KX - 1, HALF = HX / 2;
  static constexpr int G = 32 / TX;                                // query rows (y) per softmax warp
  static constexpr int NPARTS = 3;                                 // key-row parts of a halo plane
  static constexpr int RA = G, RB = KY - 1;                        // rows of parts 0 / 2 and of part 1
  static constexpr int RMAX = RA > RB ? RA : RB;
  __host__ __device__ static constexpr int part_begin(int p) { return p <= 0 ? 0 : p == 1 ? G : p == 2 ? G + KY - 1 : HY; }
  static constexpr int NA = (RA * HX + 15) / 16 * 16;              // UMMA N of parts 0 / 2 (whole TMA box)
  static constexpr int NB = (RB * HX + 15) / 16 * 16;              // UMMA N of part 1
  static constexpr int NMAX = ((NA > NB ? NA : NB) + 31) / 32 * 32;  // columns (= smem rows) of an S buffer / stage: whole 32-row rotation groups
  static constexpr int NF = (HALF + 1) / 2;                        // packed folded P words per key row
  static constexpr int DSUB = D / 64;                              // 128-byte sub-rows per head row
  static constexpr int SUB_KV = NMAX * 128, SUB_Q = M * 128;       // bytes of one sub-tile
  static constexpr int STAGE_BYTES = DSUB * SUB_KV, Q_BYTES = DSUB * SUB_Q;
  static constexpr int NSTAGE = NS_;
  static constexpr int NQBUF = (D == 64) ? 2 : 1;                  // Q buffers per slot
  static constexpr int TMEM_SLOT = 256, TMEM_O = 0, TMEM_S = D;
  static constexpr int NBARS = 5 * NSTAGE + 2 * 14 + 1;
  static constexpr int SMEM_BYTES = 1024 + (2 * NQBUF + 1) * Q_BYTES + 3 * NSTAGE * STAGE_BYTES + 8 * NBARS + 16 + 3 * 512;
  static constexpr bool FULLFOLD = (KX == HALF);                   // exactly one of the columns c, c + HALF is in the window
  static_assert(TL * TY * TX == 128 && (TY * TX) % 32 == 0 && TY == 2 * G, "128 queries per tile, one level per warp, two warps per level");
  static_assert(KL % 2 == 1 && KY % 2 == 1 && KX % 2 == 1 && TX % 2 == 0 && KY >= 3, "odd windows only (HX even)");
  static_assert(KX <= HALF, "the x fold needs kX <= HX / 2");
  static_assert(TL >= KL - 1, "tiles t and t+2 must reach disjoint planes");
  static_assert(D == 64 || D == 128, "head_dim 64 or 128");
  static_assert(HX <= 16, "halo row of at most 16 keys");
  static_assert(D + 2 * NMAX <= TMEM_SLOT, "TMEM columns of a slot");
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct FusedParams {
  int B, H, L, Y, X;
  int nty, ntx;
  long long N;
  float scale_log2e;
  int rope;       // 0: no rotation (rope_axes == 0)
  int ncols;      // level columns = B * H * nty * ntx; CTA c owns columns c, c + gridDim.x, ... (persistent)
#ifdef STRATA_TRACE
  unsigned long long* trace;   // debug: clock64 stamps of one CTA, [event][index]
  int trace_cta;
#endif
};

constexpr int kFusedThreads = 512;
// Warp roles.  The issue arbiter of an SM sub-partition prefers the highest warp id among the eligible
// warps (B300_MICROARCH.md), so the latency-critical single-thread roles get the highest ids.
constexpr int kWarpRot = 8, kWarpTma = 12, kWarpQk = 13, kWarpPv = 14;
#ifdef STRATA_TRACE
#define TRACE(ev, idx)                                                                     \
  do {                                                                                     \
    if (p.trace && (int)blockIdx.x == p.trace_cta && (idx) < 256) p.trace[(ev) * 256 + (idx)] = clock64(); \
  } while (0)
#else
#define TRACE(ev, idx) do {} while (0)
#endif
constexpr float kBig = 1099511627776.f;   // 2^40: partial row sums above this trigger a new reference maximum

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void ffma2(float& d0, float& d1, float a0, float a1, float b, float c0, float c1) {
  asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %4};\n\tmov.b64 rc, {%5, %6};\n\t"
      "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b), "f"(c0), "f"(c1));
}
__device__ __forceinline__ void fadd2(float& d0, float& d1, float a0, float a1, float b0, float b1) {
  asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
      "add.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d0), "=f"(d1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
__device__ __forceinline__ void ld16_issue(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr) : "memory");
}
// wait::ld with the loaded registers as in/out operands: no use of them can be scheduled above it.
__device__ __forceinline__ void ld16_wait(uint32_t (&r)[16]) {
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
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// One mbarrier arrival per WARP (barrier counts are in warps): every lane has made its own writes visible
// (fence.proxy.async / tcgen05.wait::st + tcgen05.fence::before_thread_sync) before the warp barrier; the
// arrival of lane 0 releases them cumulatively.  128 per-thread arrivals serialise in the barrier unit.
__device__ __forceinline__ void warp_arrive(uint32_t bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

// ---- A2 in packed bf16x2 arithmetic.  Table words (rope.cu): C = (cos m, cos m+1), S = (sin m, sin m+1).
__device__ __forceinline__ uint32_t bmul2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
__device__ __forceinline__ uint32_t bfma2(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t d;
  asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
  return d;
}
// (a, b) -> (a cos - b sin, a sin + b cos) on two pairs at once: A = (a_m, a_m+1), B = (b_m, b_m+1).
__device__ __forceinline__ void rot2(uint32_t& A, uint32_t& B, uint32_t C, uint32_t S) {
  const uint32_t nB = B ^ 0x80008000u;
  const uint32_t ra = bfma2(nB, S, bmul2(A, C));
  const uint32_t rb = bfma2(A, S, bmul2(B, C));
  A = ra; B = rb;
}
// Interleaved pairing: w0 = (a_m, b_m), w1 = (a_m+1, b_m+1).  The rotated pairs are left gathered,
// w0 = (a'_m, a'_m+1), w1 = (b'_m, b'_m+1): the same channel permutation for Q and K (see the header).
__device__ __forceinline__ void rot_interleaved(uint32_t& w0, uint32_t& w1, uint32_t C, uint32_t S) {
  uint32_t A = prmt(w0, w1, 0x5410u), B = prmt(w0, w1, 0x7632u);
  rot2(A, B, C, S);
  w0 = A; w1 = B;
}

// Rotate `rows` head rows in place.  x_smem / t_smem: operand tile and its table tile, both in the
// TMA 128-byte-swizzled layout [sub][row][128 B] with `sub_stride` bytes between sub-tiles.  The
// table tile has the operand's geometry (same box), so for the interleaved pairing the 16-byte
// chunk at a physical offset of one holds the (C, S, C, S) words of the four pairs at that offset of
// the other: the loop is linear over physical chunks.  128 threads, tid in [0, 128).
template <int DSUB, int PAIR>
__device__ __forceinline__ void rotate_inplace(uint32_t x_smem, uint32_t t_smem, uint32_t sub_stride, int rows, int tid) {
  if constexpr (PAIR == 0) {
    // `rows` is a multiple of 32 (the callers round the job up to whole 32-row groups; the extra rows are
    // pad rows of the stage that nothing reads): every thread owns exactly rows / 16 chunks per sub-tile,
    // two per step, no predicates and no divergent reconvergence points in the loop.
    const int nit = rows >> 5;
#pragma unroll
    for (int sub = 0; sub < DSUB; ++sub) {
      const uint32_t xb = x_smem + sub * sub_stride + tid * 16, tb = t_smem + sub * sub_stride + tid * 16;
      uint4 x0 = lds128(xb), t0 = lds128(tb), x1 = lds128(xb + 2048), t1 = lds128(tb + 2048);
#pragma unroll 1
      for (int it = 0; it < nit; ++it) {
        const uint32_t off = (uint32_t)it * 4096u;
        uint4 nx0 = x0, nt0 = t0, nx1 = x1, nt1 = t1;
        if (it + 1 < nit) {                                   // next step's chunks are in flight during the arithmetic
          nx0 = lds128(xb + off + 4096); nt0 = lds128(tb + off + 4096);
          nx1 = lds128(xb + off + 6144); nt1 = lds128(tb + off + 6144);
        }
        rot_interleaved(x0.x, x0.y, t0.x, t0.y); rot_interleaved(x0.z, x0.w, t0.z, t0.w);
        rot_interleaved(x1.x, x1.y, t1.x, t1.y); rot_interleaved(x1.z, x1.w, t1.z, t1.w);
        sts128(xb + off, x0); sts128(xb + off + 2048, x1);
        x0 = nx0; t0 = nt0; x1 = nx1; t1 = nt1;
      }
    }
  } else {
    // pair j = channels (j, j + D/2).  Work item = (row, c): the 8 pairs 8c .. 8c+7, c < D/16.
    constexpr int CPR = DSUB * 4;                       // work items per row
    const int n = rows * CPR;
    for (int idx = tid; idx < n; idx += 128) {
      const int row = idx / CPR, c = idx - row * CPR;
      const uint32_t sw = (uint32_t)(row & 7), rowoff = (uint32_t)row * 128u;
      uint32_t a_addr, b_addr;
      if (DSUB == 1) {                                  // a: logical chunk c, b: logical chunk c + 4
        a_addr = x_smem + rowoff + (((uint32_t)c ^ sw) << 4);
        b_addr = x_smem + rowoff + (((uint32_t)(c + 4) ^ sw) << 4);
      } else {                                          // a in sub-tile 0, b in sub-tile 1, same chunk
        a_addr = x_smem + rowoff + (((uint32_t)c ^ sw) << 4);
        b_addr = a_addr + sub_stride;
      }
      const int q0 = 2 * c, q1 = 2 * c + 1;             // table chunks (4 pairs each) of pairs 8c .. 8c+7
      const uint32_t t0_addr = t_smem + (uint32_t)(q0 >> 3) * sub_stride + rowoff + (((uint32_t)(q0 & 7) ^ sw) << 4);
      const uint32_t t1_addr = t_smem + (uint32_t)(q1 >> 3) * sub_stride + rowoff + (((uint32_t)(q1 & 7) ^ sw) << 4);
      uint4 xa = lds128(a_addr), xbv = lds128(b_addr), t0 = lds128(t0_addr), t1 = lds128(t1_addr);
      rot2(xa.x, xbv.x, t0.x, t0.y); rot2(xa.y, xbv.y, t0.z, t0.w);
      rot2(xa.z, xbv.z, t1.x, t1.y); rot2(xa.w, xbv.w, t1.z, t1.w);
      sts128(a_addr, xa); sts128(b_addr, xbv);
    }
  }
}

// Position of one slot in the global part stream (plane-major, part-minor).
template <class C>
struct SlotWalk {
  int t;   // current tile of the slot
  static __device__ __host__ __forceinline__ int plo(int t, int L) { return window_start(C::TL * t, C::KL, L); }
  static __device__ __host__ __forceinline__ int phi(int t, int L) {
    const int last = C::TL * t + C::TL - 1;
    return window_start(last < L - 1 ? last : L - 1, C::KL, L) + C::KL;
  }
  __device__ __forceinline__ void classify(int plane, int part, int nparts, int ntl, int L, bool& needed,
                                           bool& first, bool& last) {
    while (t < ntl && plane >= phi(t, L)) t += 2;
    needed = t < ntl && plane >= plo(t, L);
    first = needed && plane == plo(t, L) && part == 0;
    last = needed && plane == phi(t, L) - 1 && part == nparts - 1;
  }
};

// (a & m) | (b & ~m)
__device__ __forceinline__ uint32_t bitsel(uint32_t m, uint32_t a, uint32_t b) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, 0xCA;" : "=r"(d) : "r"(m), "r"(a), "r"(b));
  return d;
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
__device__ __forceinline__ void tmem_st2(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(r[0]), "r"(r[1]) : "memory");
}
__device__ __forceinline__ void tmem_st1(uint32_t taddr, uint32_t r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(r) : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t* r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld1(uint32_t taddr, uint32_t& r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(r) : "r"(taddr) : "memory");
}
// N (< 8) consecutive words as x4 + x2 + x1 stores
template <int N> __device__ __forceinline__ void tmem_st_words(uint32_t taddr, const uint32_t* r) {
  if (N & 4) tmem_st4(taddr, r);
  if (N & 2) tmem_st2(taddr + (N & 4), r + (N & 4));
  if (N & 1) tmem_st1(taddr + (N & 6), r[N & 6]);
}

// flags of one part for one slot, packed in a nibble of the per-CTA schedule table
constexpr uint32_t kNeeded = 1u, kFirst = 2u, kLast = 4u;
constexpr int kMaxChunks = 512;

// ------------------------------------------------------------------------------------------------
// Kernel
// ------------------------------------------------------------------------------------------------
template <class C, int PAIR>   // PAIR: strata_rope_pairing_t of the rotation
__global__ void __launch_bounds__(kFusedThreads, 1)
na3d_fwd_fused_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_ka,
                      const __grid_constant__ CUtensorMap tm_kb, const __grid_constant__ CUtensorMap tm_va,
                      const __grid_constant__ CUtensorMap tm_vb, const __grid_constant__ CUtensorMap tm_tq,
                      const __grid_constant__ CUtensorMap tm_ta, const __grid_constant__ CUtensorMap tm_tb,
                      __nv_bfloat16* __restrict__ o, float* __restrict__ lse, const FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t q_smem = base;                                        // [slot][buf] x Q_BYTES
  const uint32_t qt_smem = q_smem + 2 * C::NQBUF * C::Q_BYTES;         // table rows of the Q tile being rotated
  const uint32_t k_smem = qt_smem + C::Q_BYTES;
  const uint32_t t_smem = k_smem + C::NSTAGE * C::STAGE_BYTES;
  const uint32_t v_smem = t_smem + C::NSTAGE * C::STAGE_BYTES;
  const uint32_t bars = v_smem + C::NSTAGE * C::STAGE_BYTES;
  auto bar_kfull = [&](int s) { return bars + 8u * s; };                          // TMA -> rotation
  auto bar_krot = [&](int s) { return bars + 8u * (C::NSTAGE + s); };             // rotation -> MMA (128)
  auto bar_kempty = [&](int s) { return bars + 8u * (2 * C::NSTAGE + s); };       // QK issuer -> TMA
  auto bar_vfull = [&](int s) { return bars + 8u * (3 * C::NSTAGE + s); };
  auto bar_vempty = [&](int s) { return bars + 8u * (4 * C::NSTAGE + s); };
  // per slot: 0,1 qfull[buf]  2,3 qrot[buf]  4,5 qfree[buf]  6,7 sfull[buf]  8,9 pfull[buf]  10,11 pvdone[buf]
  // 12,13 pvissued[buf] (the PV MMA that reads P from S buffer `buf` has been ISSUED: MMAs execute in issue order,
  // so the next QK^T into that buffer may be issued without waiting for the PV MMA to complete)
  // Every barrier that is not waited on in every phase is split by parity of its use count: a waiter
  // may only test the parity of a phase when the barrier is known to be in that phase or the next.
  auto bar_slot = [&](int slot, int which) { return bars + 8u * (5 * C::NSTAGE + 14 * slot + which); };
  const uint32_t bar_qtempty = bars + 8u * (5 * C::NSTAGE + 28);
  const uint32_t tmem_word = bars + 8u * C::NBARS;
  uint32_t* tmem_word_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_word - raw));
  uint8_t* sched = smem_raw + (tmem_word + 16 - raw);                  // [L * nparts] nibble pairs

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- geometry of one level column: head fastest (the H heads of a token are one contiguous
  // H*D*2-byte run in HBM), then x, y, sample.  The CTA is persistent: it owns columns blockIdx.x,
  // blockIdx.x + gridDim.x, ...; every pipeline counter (stage ring position, items, tiles, Q jobs)
  // keeps running across columns, so the next column's loads, rotations and MMAs overlap the drain of
  // the previous one.
  struct Col {
    int h, b, x0, y0, hs_x, hs_y, hy, nparts, nchunks, bl;
  };
  auto column = [&](int col) {
    Col c;
    int bid = col;
    c.h = bid % p.H; bid /= p.H;
    const int tx = bid % p.ntx; bid /= p.ntx;
    const int ty = bid % p.nty;
    c.b = bid / p.nty;
    c.x0 = tx * C::TX; c.y0 = ty * C::TY;
    const int yl = min(c.y0 + C::TY, p.Y) - 1;
    c.hs_x = window_start(c.x0, C::KX, p.X); c.hs_y = window_start(c.y0, C::KY, p.Y);
    c.hy = window_start(yl, C::KY, p.Y) + C::KY - c.hs_y;     // key rows of the halo, <= HY
    c.nparts = c.hy > C::part_begin(2) ? 3 : c.hy > C::part_begin(1) ? 2 : 1;
    c.nchunks = p.L * c.nparts;
    c.bl = c.b * p.L;
    return c;
  };
  const int ntl = (p.L + C::TL - 1) / C::TL;
  const uint32_t op_tx = p.rope ? 2u : 1u;                        // operand + table bytes per barrier
  auto box_rows = [&](int part) { return part == 1 ? C::RB : C::RA; };
  // schedule tables, one per possible number of parts: sched_of(nparts)[plane * nparts + part]
  auto sched_of = [&](int nparts) { return sched + kMaxChunks * (nparts - 1); };

  // ---- one-time setup
  if (warp == kWarpTma && lane == 0) {
    tma_prefetch_desc(&tm_q); tma_prefetch_desc(&tm_ka); tma_prefetch_desc(&tm_kb);
    tma_prefetch_desc(&tm_va); tma_prefetch_desc(&tm_vb);
    if (p.rope) { tma_prefetch_desc(&tm_tq); tma_prefetch_desc(&tm_ta); tma_prefetch_desc(&tm_tb); }
    for (int s = 0; s < C::NSTAGE; ++s) {
      mbar_init(bar_kfull(s), 1); mbar_init(bar_krot(s), 4); mbar_init(bar_kempty(s), 1);
      mbar_init(bar_vfull(s), 1); mbar_init(bar_vempty(s), 2);
    }
    for (int slot = 0; slot < 2; ++slot) {
      mbar_init(bar_slot(slot, 0), 1); mbar_init(bar_slot(slot, 1), 1);
      mbar_init(bar_slot(slot, 2), 4); mbar_init(bar_slot(slot, 3), 4);
      mbar_init(bar_slot(slot, 4), 1); mbar_init(bar_slot(slot, 5), 1);
      mbar_init(bar_slot(slot, 6), 1); mbar_init(bar_slot(slot, 7), 1);
      mbar_init(bar_slot(slot, 8), 4); mbar_init(bar_slot(slot, 9), 4);
      mbar_init(bar_slot(slot, 10), 1); mbar_init(bar_slot(slot, 11), 1);
      mbar_init(bar_slot(slot, 12), 1); mbar_init(bar_slot(slot, 13), 1);
    }
    mbar_init(bar_qtempty, 4);
    fence_barrier_init();
  }
  if (warp == kWarpTma) tmem_alloc(tmem_word, 512);
  // schedule tables: which slot needs part g, and whether it is the first / last part of its tile
  for (int np = 1; np <= C::NPARTS; ++np)
    for (int g = threadIdx.x; g < p.L * np; g += kFusedThreads) {
      const int plane = g / np, part = g - plane * np;
      uint32_t e = 0;
      for (int t = 0; t < ntl; ++t) {
        const int lo = SlotWalk<C>::plo(t, p.L), hi = SlotWalk<C>::phi(t, p.L);
        if (plane < lo || plane >= hi) continue;
        uint32_t f = kNeeded;
        if (plane == lo && part == 0) f |= kFirst;
        if (plane == hi - 1 && part == np - 1) f |= kLast;
        e |= f << (4 * (t & 1));
      }
      sched_of(np)[g] = (uint8_t)e;
    }
  // V stages start as zeros: rows of a stage that a (shorter) part does not overwrite are multiplied
  // by P = 0 in the PV MMA and must therefore hold finite numbers.
  for (uint32_t off = threadIdx.x * 16u; off < (uint32_t)(C::NSTAGE * C::STAGE_BYTES); off += kFusedThreads * 16u)
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(v_smem + off), "r"(0u) : "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_word_ptr;

  if (warp >= kWarpTma) {
    reg_dec<56>();
    if (warp == kWarpTma) {
      // =========================== TMA producer ===========================
      int nrun[2] = {0, 0};                                           // tiles of each slot so far (all columns)
      int qjob = 0, gbase = 0;
      // a deferred V load: G < 0 = none; a = cy0 | hs_x << 16, b = plane (b * L + l), hm = h | mid << 16
      int v0G = -1, v0a = 0, v0b = 0, v0hm = 0, v1G = -1, v1a = 0, v1b = 0, v1hm = 0;
      auto issue_v = [&](int G, int a, int b, int hm) {
        const int s = G % C::NSTAGE;
        const uint32_t ph = (uint32_t)(G / C::NSTAGE) & 1u;
        const bool mid = (hm >> 16) != 0;
        mbar_wait(bar_vempty(s), ph ^ 1u);
        if (lane == 0) TRACE(1, G);
        if (elect_one()) {
          mbar_expect_tx(bar_vfull(s), (uint32_t)(box_rows(mid ? 1 : 0) * C::HX * 128 * C::DSUB));
#pragma unroll
          for (int jj = 0; jj < C::DSUB; ++jj)
            tma_load_5d(v_smem + s * C::STAGE_BYTES + jj * C::SUB_KV, mid ? &tm_vb : &tm_va, bar_vfull(s), 64 * jj, hm & 0xffff,
                        a >> 16, a & 0xffff, b);
        }
        __syncwarp();
      };
      for (int col = blockIdx.x; col < p.ncols; col += gridDim.x) {
        const Col c = column(col);
        const uint8_t* sc = sched_of(c.nparts);
        int nloc[2] = {0, 0};                                         // tiles of each slot in this column
        int part = 0, plane = 0;
        for (int g = 0; g < c.nchunks; ++g) {
          const uint32_t e = sc[g];
#pragma unroll
          for (int slot = 0; slot < 2; ++slot) {
            if (!((e >> (4 * slot)) & kFirst)) continue;
            const int n = nrun[slot]++;
            const int buf = n % C::NQBUF, use = n / C::NQBUF;         // use-th tile in this Q buffer
            if (use >= 1) mbar_wait(bar_slot(slot, 4 + buf), (uint32_t)(use - 1) & 1u);   // its last QK^T is done
            if (p.rope && qjob >= 1) mbar_wait(bar_qtempty, (uint32_t)(qjob - 1) & 1u);
            const uint32_t bar = bar_slot(slot, buf);
            const uint32_t qb = q_smem + (slot * C::NQBUF + buf) * C::Q_BYTES;
            const int l0 = c.bl + C::TL * (slot + 2 * nloc[slot]++);
            if (elect_one()) {
              mbar_expect_tx(bar, op_tx * C::Q_BYTES);
#pragma unroll
              for (int j = 0; j < C::DSUB; ++j) {
                tma_load_5d(qb + j * C::SUB_Q, &tm_q, bar, 64 * j, c.h, c.x0, c.y0, l0);
                if (p.rope) tma_load_5d(qt_smem + j * C::SUB_Q, &tm_tq, bar, 64 * j, 0, c.x0, c.y0, l0);
              }
            }
            __syncwarp();
            ++qjob;
          }
          const int G = gbase + g;
          const int s = G % C::NSTAGE;
          const uint32_t ph = (uint32_t)(G / C::NSTAGE) & 1u;
          const bool mid = part == 1;
          const uint32_t bytes = (uint32_t)(box_rows(part) * C::HX * 128 * C::DSUB);
          const int cy0 = c.hs_y + C::part_begin(part);
          mbar_wait(bar_kempty(s), ph ^ 1u);
          if (lane == 0) TRACE(0, G);
          if (elect_one()) {
            mbar_expect_tx(bar_kfull(s), op_tx * bytes);
#pragma unroll
            for (int j = 0; j < C::DSUB; ++j) {
              tma_load_5d(k_smem + s * C::STAGE_BYTES + j * C::SUB_KV, mid ? &tm_kb : &tm_ka, bar_kfull(s), 64 * j, c.h, c.hs_x, cy0, c.bl + plane);
              if (p.rope)
                tma_load_5d(t_smem + s * C::STAGE_BYTES + j * C::SUB_KV, mid ? &tm_tb : &tm_ta, bar_kfull(s), 64 * j, 0, c.hs_x, cy0, c.bl + plane);
            }
          }
          __syncwarp();
          // V of this part is loaded two steps later (see VJob): a V stage is released by the PV MMA, long
          // after the K stage of the same part (QK^T); waiting for it here would hold back the next K loads
          if (v0G >= 0) issue_v(v0G, v0a, v0b, v0hm);
          v0G = v1G; v0a = v1a; v0b = v1b; v0hm = v1hm;
          v1G = G; v1a = cy0 | (c.hs_x << 16); v1b = c.bl + plane; v1hm = c.h | ((mid ? 1 : 0) << 16);
          if (++part == c.nparts) { part = 0; ++plane; }
        }
        gbase += c.nchunks;
      }
      if (v0G >= 0) issue_v(v0G, v0a, v0b, v0hm);
      if (v1G >= 0) issue_v(v1G, v1a, v1b, v1hm);
    } else if (warp == kWarpQk) {
      // =========================== QK^T issuer (both slots) ===========================
      // The whole warp walks the schedule in uniform control flow (descriptors stay in uniform
      // registers); one elected lane issues the MMAs and commits.
      int it[2] = {0, 0}, nseq[2] = {-1, -1};
      int gbase = 0;
      for (int col = blockIdx.x; col < p.ncols; col += gridDim.x) {
      const Col c = column(col);
      const uint8_t* sc = sched_of(c.nparts);
      int part = 0;
      for (int g = 0; g < c.nchunks; ++g) {
        const uint32_t e = sc[g];
        const int G = gbase + g;
        const int s = G % C::NSTAGE;
        const uint32_t ph = (uint32_t)(G / C::NSTAGE) & 1u;
        const uint32_t idesc_qk = part == 1 ? instr_desc(C::M, C::NB, false) : instr_desc(C::M, C::NA, false);
        if (++part == c.nparts) part = 0;
        mbar_wait<false>(bar_krot(s), ph);
        if (lane == 0) TRACE(4, G);
        tc_fence_after();
#pragma unroll
        for (int slot = 0; slot < 2; ++slot) {
          const uint32_t es = (e >> (4 * slot)) & 15u;
          if (!(es & kNeeded)) continue;
          if (es & kFirst) ++nseq[slot];
          const int buf = nseq[slot] % C::NQBUF, use = nseq[slot] / C::NQBUF;
          if (es & kFirst) mbar_wait<false>(bar_slot(slot, 2 + buf), (uint32_t)use & 1u);       // Q tile rotated
          const int i = it[slot]++;
          if (i >= 2) {     // S buffer (i & 1) may be overwritten by MMAs issued after the PV MMA of item i - 2
            mbar_wait<false>(bar_slot(slot, 12 + (i & 1)), (uint32_t)((i - 2) >> 1) & 1u);
            tc_fence_after();
          }
          const uint32_t qb = q_smem + (slot * C::NQBUF + buf) * C::Q_BYTES;
          const uint32_t d_tmem = tmem + slot * C::TMEM_SLOT + C::TMEM_S + (i & 1) * C::NMAX;
          if (elect_one()) {
#pragma unroll
            for (int ks = 0; ks < C::D / 16; ++ks) {
              const uint32_t sub = (uint32_t)(ks >> 2), kin = (uint32_t)(ks & 3) * 32u;
              umma_ss(d_tmem, smem_desc(qb + sub * C::SUB_Q + kin),
                      smem_desc(k_smem + s * C::STAGE_BYTES + sub * C::SUB_KV + kin), idesc_qk, ks > 0 ? 1u : 0u);
            }
            umma_commit(bar_slot(slot, 6 + (i & 1)));
            if (es & kLast) umma_commit(bar_slot(slot, 4 + buf));    // every QK^T of the tile is done: Q buffer free
          }
          __syncwarp();
          if (lane == 0) TRACE(6 + slot, G);
        }
        if (elect_one()) umma_commit(bar_kempty(s));                 // both slots' QK^T of this part
        __syncwarp();
      }
      gbase += c.nchunks;
      }
    } else {
      // =========================== PV issuer of one slot ===========================
      const int slot = warp - kWarpPv;
      const uint32_t tm = tmem + slot * C::TMEM_SLOT;
      constexpr uint32_t idesc_pv = instr_desc(C::M, 64, true);
      int i = 0, gbase = 0;
      for (int col = blockIdx.x; col < p.ncols; col += gridDim.x) {
      const Col c = column(col);
      const uint8_t* sc = sched_of(c.nparts);
      int part = 0;
      for (int g = 0; g < c.nchunks; ++g) {
        const uint32_t es = (sc[g] >> (4 * slot)) & 15u;
        const int G = gbase + g;
        const int s = G % C::NSTAGE;
        const uint32_t ph = (uint32_t)(G / C::NSTAGE) & 1u;
        const int nk = (part == 1 ? C::NB : C::NA) / 16;
        if (++part == c.nparts) part = 0;
        if (!(es & kNeeded)) {        // this slot does not use the part: release it once it has landed
          mbar_wait<false>(bar_vfull(s), ph);        // (one arrival per slot and phase, never ahead of the producer)
          if (elect_one()) mbar_arrive(bar_vempty(s));
          __syncwarp();
          continue;
        }
        mbar_wait<false>(bar_slot(slot, 8 + (i & 1)), (uint32_t)(i >> 1) & 1u);       // P of item i is in TMEM
        if (lane == 0) TRACE(8 + slot, G);
        mbar_wait<false>(bar_vfull(s), ph);
        tc_fence_after();
        const uint32_t a_tmem = tm + C::TMEM_S + (i & 1) * C::NMAX;
        const uint32_t vb = v_smem + s * C::STAGE_BYTES;
        const uint32_t acc0 = (es & kFirst) ? 0u : 1u;
        if (elect_one()) {
          auto issue = [&](auto nkc) {               // fully unrolled: the descriptors are immediates off one base
#pragma unroll
            for (int ks = 0; ks < decltype(nkc)::value; ++ks) {
#pragma unroll
              for (int j = 0; j < C::DSUB; ++j)
                umma_ts(tm + C::TMEM_O + 64 * j, a_tmem + 8 * ks, smem_desc(vb + j * C::SUB_KV + ks * 16 * 128), idesc_pv,
                        ks > 0 ? 1u : acc0);
            }
          };
          if (nk == C::NB / 16) issue(std::integral_constant<int, C::NB / 16>{});
          else issue(std::integral_constant<int, C::NA / 16>{});
          umma_commit(bar_vempty(s));
          umma_commit(bar_slot(slot, 10 + (i & 1)));
          tc_fence_before();
          mbar_arrive(bar_slot(slot, 12 + (i & 1)));
        }
        __syncwarp();
        if (lane == 0) TRACE(10 + slot, G);
        ++i;
      }
      gbase += c.nchunks;
      }
    }
  } else if (warp >= kWarpRot) {
    // =========================== rotation warpgroup ===========================
    reg_dec<88>();
    const int tid = threadIdx.x - 32 * kWarpRot;
    // K parts only: the Q tile of a slot is rotated by that slot's softmax warpgroup while it waits for the
    // last PV MMA of its previous tile (see below).
    int gbase = 0;
    for (int col = blockIdx.x; col < p.ncols; col += gridDim.x) {
    const Col c = column(col);
    int part = 0;
    for (int g = 0; g < c.nchunks; ++g) {
      const int G = gbase + g;
      const int s = G % C::NSTAGE;
      int rows = box_rows(part) * C::HX;
      if (PAIR == 0) rows = (rows + 31) & ~31;            // whole 32-row groups (pad rows of the stage: never read)
      if (tid == 0) TRACE(5, G);
      mbar_wait(bar_kfull(s), (uint32_t)(G / C::NSTAGE) & 1u);     // operand (+ table) landed
      if (tid == 0) TRACE(2, G);
      if (p.rope) {
        rotate_inplace<C::DSUB, PAIR>(k_smem + s * C::STAGE_BYTES, t_smem + s * C::STAGE_BYTES, C::SUB_KV, rows, tid);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      }
      if (tid == 0) TRACE(3, G);
      warp_arrive(bar_krot(s));
      if (++part == c.nparts) part = 0;
    }
    gbase += c.nchunks;
    }
  } else {
    // =========================== softmax + epilogue of one slot ===========================
    reg_inc<184>();
    const int slot = warp >> 2;
    const int sp = warp & 3;                       // TMEM subpartition
    const int row = sp * 32 + lane;                // query row of the tile == TMEM lane
    const uint32_t tm = tmem + slot * C::TMEM_SLOT + ((uint32_t)(sp * 32) << 16);
    const int qx = row % C::TX, qy = (row / C::TX) % C::TY, ql = row / (C::TX * C::TY);
    const float cs = p.scale_log2e;
    // A2 for Q: this warpgroup rotates its slot's Q tiles in place (same code as the K parts), the next tile's
    // while the last PV MMA of the current tile is still running.
    const int ncols_cta = (p.ncols - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int qtotal = ncols_cta * (ntl > slot ? (ntl - slot + 1) / 2 : 0);      // Q tiles of this slot, all columns
    int nq = 0;
    auto rotate_next_q = [&]() {
      if (nq >= qtotal) return;
      const int buf = nq % C::NQBUF, use = nq / C::NQBUF;
      mbar_wait(bar_slot(slot, buf), (uint32_t)use & 1u);            // Q tile (+ its table rows) landed
      if (p.rope) {
        rotate_inplace<C::DSUB, PAIR>(q_smem + (slot * C::NQBUF + buf) * C::Q_BYTES, qt_smem, C::SUB_Q, C::M, row);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        warp_arrive(bar_qtempty);
      }
      warp_arrive(bar_slot(slot, 2 + buf));
      ++nq;
    };
    rotate_next_q();
    int i = 0;
    for (int col = blockIdx.x; col < p.ncols; col += gridDim.x) {
    const Col c = column(col);
    const int x0 = c.x0, y0 = c.y0, hs_x = c.hs_x, hs_y = c.hs_y, hy = c.hy, nparts = c.nparts, h = c.h, b = c.b;
    auto part_rows = [&](int part) { return min(C::part_begin(part + 1), hy) - C::part_begin(part); };
    const int ax = min(x0 + qx, p.X - 1), ay = min(y0 + qy, p.Y - 1);
    const bool active_xy = (x0 + qx < p.X) && (y0 + qy < p.Y);
    const int lo_x = window_start(ax, C::KX, p.X) - hs_x;
    const int lo_y = window_start(ay, C::KY, p.Y) - hs_y;
    const int wy_lo = __reduce_min_sync(0xffffffffu, lo_y), wy_hi = __reduce_max_sync(0xffffffffu, lo_y + C::KY);
    // x fold: of the halo columns c and c + HALF at most one lies in this query's window
    uint32_t m_lo[C::HALF];                        // all ones: column c is the one (else c + HALF, or neither)
    float xz[C::HALF];                             // 0 if one of the two is in the window, else -inf
#pragma unroll
    for (int c = 0; c < C::HALF; ++c) {
      const bool in_lo = c >= lo_x && c < lo_x + C::KX, in_hi = c + C::HALF >= lo_x && c + C::HALF < lo_x + C::KX;
      m_lo[c] = in_lo ? 0xffffffffu : 0u;
      xz[c] = (in_lo || in_hi) ? 0.f : -INFINITY;
    }
    // un-fold: P word j holds the halo columns (2j, 2j+1).  Column col comes from the folded value
    // fc = col mod HALF, which sits in half (fc & 1) of the packed word F[fc / 2]; psel[j] is the byte
    // selector of prmt(F[fc(2j) / 2], F[fc(2j+1) / 2]).  A column outside the window selects "sign of a
    // high byte", which is 0x00 because every P value is >= +0.
    uint32_t psel[C::HX / 2];
#pragma unroll
    for (int j = 0; j < C::HX / 2; ++j) {
      const int c0 = 2 * j, c1 = 2 * j + 1;
      const int f0 = c0 % C::HALF, f1 = c1 % C::HALF;
      const bool v0 = c0 >= lo_x && c0 < lo_x + C::KX, v1 = c1 >= lo_x && c1 < lo_x + C::KX;
      const uint32_t n0 = v0 ? (uint32_t)(2 * (f0 & 1)) | ((uint32_t)(2 * (f0 & 1) + 1) << 4) : 0x99u;
      const uint32_t n1 = v1 ? (uint32_t)(4 + 2 * (f1 & 1)) | ((uint32_t)(5 + 2 * (f1 & 1)) << 4) : 0xDDu;
      psel[j] = n0 | (n1 << 8);
    }

    for (int tile = slot; tile < ntl; tile += 2) {
      const int al = min(C::TL * tile + ql, p.L - 1);
      const bool active = active_xy && (C::TL * tile + ql < p.L);
      const int pw_lo = window_start(al, C::KL, p.L);              // planes of this query: [pw_lo, pw_lo + KL)
      const int wl_lo = __reduce_min_sync(0xffffffffu, pw_lo), wl_hi = __reduce_max_sync(0xffffffffu, pw_lo + C::KL);
      float m_ref = 0.f, lsum = 0.f;
      bool inited = false;
      const int plo = SlotWalk<C>::plo(tile, p.L), phi = SlotWalk<C>::phi(tile, p.L);
      for (int plane = plo; plane < phi; ++plane) {
        const bool plane_needed = plane >= wl_lo && plane < wl_hi;
        const bool plane_ok = plane >= pw_lo && plane < pw_lo + C::KL;
#pragma unroll 1
        for (int part = 0; part < nparts; ++part, ++i) {
          const int pb = C::part_begin(part);
          const int nrows = part_rows(part);
          const uint32_t s_addr = tm + C::TMEM_S + (i & 1) * C::NMAX;
          const bool first_item = (plane == plo && part == 0);
          // does some query of the warp attend a key row of this part? (warp-uniform)
          const bool warp_needs = plane_needed && max(0, wy_lo - pb) < min(nrows, wy_hi - pb);
          // rows of this part inside this query's window: [ya, yb)
          const int ya = plane_ok ? max(0, lo_y - pb) : 0;
          const int yb = plane_ok ? min(nrows, lo_y + C::KY - pb) : 0;
          mbar_wait(bar_slot(slot, 6 + (i & 1)), (uint32_t)(i >> 1) & 1u);
          if (sp == 0 && lane == 0) TRACE(12 + slot, i);
          tc_fence_after();

          // One part of R key rows (the whole TMA box: rows past the halo are zero keys, masked by [ya, yb)).
          auto do_part = [&](auto rc) {
            constexpr int R = decltype(rc)::value;
            constexpr int NCOL = R * C::HX, NW = ((NCOL + 15) / 16 * 16) / 2;
            float v[R][C::HALF];                     // folded logits
            {
              uint32_t sv[NCOL];
              tmem_ld_n<NCOL>(s_addr, sv);
#pragma unroll
              for (int r = 0; r < R; ++r)
#pragma unroll
                for (int c = 0; c < C::HALF; ++c)
                  v[r][c] = __uint_as_float(bitsel(m_lo[c], sv[r * C::HX + c], sv[r * C::HX + c + C::HALF]));
            }
            // maximum of this query's valid logits of the part (log2 units)
            // (csm: the scale as an opaque register, so that the compiler cannot hoist this rarely needed
            // computation out of its branch into the exponential pass)
            auto part_max = [&](float csm) {
              float cmax = -INFINITY;
#pragma unroll
              for (int r = 0; r < R; ++r) {
                float rmax = -INFINITY;
#pragma unroll
                for (int c = 0; c < C::HALF; ++c) rmax = fmaxf(rmax, C::FULLFOLD ? v[r][c] * csm : fmaf(v[r][c], csm, xz[c]));
                if (r >= ya && r < yb) cmax = fmaxf(cmax, rmax);
              }
              return cmax;
            };
            if (__any_sync(0xffffffffu, ya < yb && !inited)) {
              // ---- first valid keys of some query: its reference is the true maximum of this part
              float cso = cs;
              asm volatile("mov.f32 %0, %0;" : "+f"(cso));
              const float cmax = part_max(cso);
              if (!inited && cmax > -INFINITY) { m_ref = cmax; inited = true; }
            }
            float pr[R][C::HALF];                    // folded probabilities (times 2^-m_ref)
            float rs = 0.f;
            int attempt = 0;
#pragma unroll 1
            do {                                     // (rare block first: ONE copy of the exponential pass in the code)
              if (attempt > 0) {
                // ---- a logit far above the reference: move the reference to the true maximum and
                // rescale what was accumulated so far (P of this part is not stored yet)
                const bool mine = !(rs <= kBig);
                float cso = cs;
                asm volatile("mov.f32 %0, %0;" : "+f"(cso));
                const float new_ref = mine ? fmaxf(m_ref, part_max(cso)) : m_ref;
                const float alpha = new_ref != m_ref ? ex2(m_ref - new_ref) : 1.f;
                if (!first_item) {
                  // O holds earlier parts of this tile: all its PV MMAs are complete after pv_done(i - 1)
                  mbar_wait(bar_slot(slot, 10 + ((i - 1) & 1)), (uint32_t)((i - 1) >> 1) & 1u);
                  tc_fence_after();
#pragma unroll 1
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
                m_ref = new_ref;
              }
              // ---- p = 2^(s * cs - m_ref), branch-free over the whole part
              float e0 = 0.f, e1 = 0.f, e2 = 0.f, e3 = 0.f;
#pragma unroll
              for (int r = 0; r < R; ++r) {
                const float br = (r >= ya && r < yb) ? -m_ref : -INFINITY;
#pragma unroll
                for (int c = 0; c < C::HALF; c += 2) {
                  if (c + 1 < C::HALF) {
                    float t0, t1;
                    if (C::FULLFOLD) ffma2(t0, t1, v[r][c], v[r][c + 1], cs, br, br);
                    else ffma2(t0, t1, v[r][c], v[r][c + 1], cs, br + xz[c], br + xz[c + 1]);
                    pr[r][c] = ex2(t0); pr[r][c + 1] = ex2(t1);
                    if ((c >> 1) & 1) fadd2(e2, e3, e2, e3, pr[r][c], pr[r][c + 1]);
                    else fadd2(e0, e1, e0, e1, pr[r][c], pr[r][c + 1]);
                  } else {
                    pr[r][c] = ex2(fmaf(v[r][c], cs, C::FULLFOLD ? br : br + xz[c]));
                    e0 += pr[r][c];
                  }
                }
              }
              rs = (e0 + e1) + (e2 + e3);
              ++attempt;
            } while (attempt < 2 && __any_sync(0xffffffffu, !(rs <= kBig)));
            lsum += rs;
            // ---- pack folded pairs to bf16x2, un-fold with one byte permute per output word; P overlays
            // the front of S (every S column of the part is in registers by now)
            uint32_t pw[NW];
#pragma unroll
            for (int r = 0; r < R; ++r) {
              uint32_t f[C::NF];
#pragma unroll
              for (int m = 0; m < C::NF; ++m) f[m] = pack_bf16(pr[r][2 * m], 2 * m + 1 < C::HALF ? pr[r][2 * m + 1] : 0.f);
#pragma unroll
              for (int j = 0; j < C::HX / 2; ++j)
                pw[r * (C::HX / 2) + j] = prmt(f[((2 * j) % C::HALF) / 2], f[((2 * j + 1) % C::HALF) / 2], psel[j]);
            }
#pragma unroll
            for (int j = R * (C::HX / 2); j < NW; ++j) pw[j] = 0u;     // pad keys
            tmem_st_n<NW>(s_addr, pw);
          };

          if (warp_needs) {
            if (part == 1) do_part(std::integral_constant<int, C::RB>{});
            else do_part(std::integral_constant<int, C::RA>{});
          } else {
            // no query of this warp attends a key of this part: P = 0
            uint32_t z[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) z[u] = 0u;
            const int nwords = (part == 1 ? C::NB : C::NA) / 2;
            for (int j = 0; j < nwords; j += 8) tmem_st8(s_addr + j, z);
          }
          tmem_wait_st();
          tc_fence_before();
          if (sp == 0 && lane == 0) TRACE(14 + slot, i);
          warp_arrive(bar_slot(slot, 8 + (i & 1)));
        }
      }
      rotate_next_q();
      // ---- tile epilogue: O / l -> bf16 -> global, LSE
      mbar_wait(bar_slot(slot, 10 + ((i - 1) & 1)), (uint32_t)((i - 1) >> 1) & 1u);
      tc_fence_after();
      const float inv = 1.f / lsum;
      const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
      __nv_bfloat16* orow = o + (((long long)b * p.N + tok) * p.H + h) * C::D;
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
      // the O reads above are complete before the next tile's first PV MMA overwrites O: that MMA
      // waits for this warpgroup's next p_full arrival, which follows these (waited-for) loads.
    }
    }
  }

  // ---- teardown
  tc_fence_before();
  __syncthreads();
  if (warp == kWarpTma) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

// ------------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------------
template <class C>
bool fused_shape_ok(const Problem& p) {
  // the tiles of one slot must reach disjoint, increasing plane ranges (one pass over the levels)
  const int ntl = (p.L + C::TL - 1) / C::TL;
  if (p.L * C::NPARTS > kMaxChunks) return false;                    // per-CTA schedule table
  for (int t = 0; t + 2 < ntl; ++t)
    if (SlotWalk<C>::plo(t + 2, p.L) < SlotWalk<C>::phi(t, p.L)) return false;
  return true;
}

template <class C>
cudaError_t launch_fused(const Problem& p, const void* q, const void* k, const void* v, const void* table, void* o,
                         float* lse, cudaStream_t stream, int* launches) {
  CUtensorMap tq, tka, tkb, tva, tvb, ttq, tta, ttb;
  if (!make_map(&tq, q, p, C::TX, C::TY, C::TL) || !make_map(&tka, k, p, C::HX, C::RA, 1) ||
      !make_map(&tkb, k, p, C::HX, C::RB, 1) || !make_map(&tva, v, p, C::HX, C::RA, 1) ||
      !make_map(&tvb, v, p, C::HX, C::RB, 1))
    return cudaErrorInvalidValue;
  const bool rope = p.A > 0;
  if (rope) {
    Problem pt = p;
    pt.H = 1;                                  // the table is [B, L, Y, X, D] 16-bit words: one "head"
    if (!make_map(&ttq, table, pt, C::TX, C::TY, C::TL) || !make_map(&tta, table, pt, C::HX, C::RA, 1) ||
        !make_map(&ttb, table, pt, C::HX, C::RB, 1))
      return cudaErrorInvalidValue;
  } else {
    ttq = tq; tta = tka; ttb = tkb;            // never dereferenced
  }
  FusedParams fp;
  fp.B = p.B; fp.H = p.H; fp.L = p.L; fp.Y = p.Y; fp.X = p.X; fp.N = p.N;
  fp.nty = (p.Y + C::TY - 1) / C::TY; fp.ntx = (p.X + C::TX - 1) / C::TX;
  fp.scale_log2e = p.scale * 1.4426950408889634f;
  fp.rope = rope ? 1 : 0;
#ifdef STRATA_TRACE
  {
    const char* e = getenv("STRATA_TRACE_PTR");
    fp.trace = e ? (unsigned long long*)strtoull(e, nullptr, 0) : nullptr;
    const char* c = getenv("STRATA_TRACE_CTA");
    fp.trace_cta = c ? atoi(c) : 0;
  }
#endif
  const long long ncols = (long long)p.B * p.H * fp.nty * fp.ntx;
  if (ncols > 0x7fffffffLL) return cudaErrorInvalidValue;
  fp.ncols = (int)ncols;
  static int sm_count = 0;
  if (sm_count == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        sm_count <= 0) {
      (void)cudaGetLastError();
      sm_count = 148;
    }
  }
  const long long grid = ncols < sm_count ? ncols : sm_count;      // persistent: one CTA per SM
  auto kernel = p.pairing ? na3d_fwd_fused_kernel<C, 1> : na3d_fwd_fused_kernel<C, 0>;
  static bool attr_set[2] = {false, false};
  if (!attr_set[p.pairing ? 1 : 0]) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr_set[p.pairing ? 1 : 0] = true;
  }
  prof_begin("na3d_fwd_fused", stream);
  kernel<<<(unsigned)grid, kFusedThreads, C::SMEM_BYTES, stream>>>(
      tq, tka, tkb, tva, tvb, ttq, tta, ttb, (__nv_bfloat16*)o, lse, fp);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace

// (D, kL, kY, kX, TL, TY, TX, NSTAGE) instantiations.
#define STRATA_FUSED_CONFIGS(X) \
  X(64, 3, 7, 7, 2, 8, 8, 4)    \
  X(64, 3, 5, 5, 2, 8, 8, 4)    \
  X(64, 3, 3, 3, 2, 8, 8, 4)

bool fused_fwd_supported(const Problem& p) {
  if (p.dtype != 1) return false;
#define X(D_, KL_, KY_, KX_, TL_, TY_, TX_, NS_)                        \
  if (p.D == D_ && p.kL == KL_ && p.kY == KY_ && p.kX == KX_)          \
    return fused_shape_ok<FusedCfg<D_, KL_, KY_, KX_, TL_, TY_, TX_, NS_>>(p);
  STRATA_FUSED_CONFIGS(X)
#undef X
  return false;
}

cudaError_t launch_fwd_fused(const Problem& p, const void* q, const void* k, const void* v, const void* table,
                             void* o, float* lse, cudaStream_t stream, int* launches) {
#define X(D_, KL_, KY_, KX_, TL_, TY_, TX_, NS_)                        \
  if (p.D == D_ && p.kL == KL_ && p.kY == KY_ && p.kX == KX_)          \
    return launch_fused<FusedCfg<D_, KL_, KY_, KX_, TL_, TY_, TX_, NS_>>(p, q, k, v, table, o, lse, stream, launches);
  STRATA_FUSED_CONFIGS(X)
#undef X
  return cudaErrorNotSupported;
}

}  // namespace strata
