// na3d_fwd_plane.cu -- fused StereoRoPE + 3D neighbourhood attention forward (tcgen05 / TMEM / TMA), head_dim 64,
// k_L = 3.  Steps A1-A6 of DESIGN.md in ONE kernel: Q, K, V, the per-token stereographic coordinates and the
// frequency table are the only inputs; rotary angles (A1), the rotation of Q and K (A2), the clamped windows (A3),
// logits, softmax + LSE and the output (A4-A6) all happen here; nothing rotated ever touches HBM.
//
// WHAT BOUNDS THIS PATH ON B200 (measured): shared-memory bandwidth.  A tcgen05.mma reads its
// shared-memory operands at 128 B / clock and has priority over ld/st.shared, which get what is left; the dense
// 128-row tile against a 14 x 14 key halo already needs 53 KB of K / V operand reads per plane.  So every other
// byte is kept out of shared memory: Q never enters it (global -> registers -> rotated -> TMEM, the A operand of
// Q K^T), S and P live in TMEM, O goes from TMEM through registers to global memory, a K / V plane is staged
// once per level column and stays resident for every query tile that needs it.
//
// Work decomposition ("level sweep"): persistent CTAs, one per SM; CTA c takes the UNITS c, c + gridDim.x, ...
// A unit is hg consecutive heads of one (sample, y tile, x tile); one head of it is a level COLUMN: the 8 x 8 patch
// of every level, i.e. ceil(L / 2) query tiles of 2 x 8 x 8 = 128 queries.  The tiles of a column run one after the
// other; tile t needs the key / value planes [plo(t), phi(t)) (its rows' clamped level windows, PAPER.md:79,
// DESIGN.md R1), each a halo of HY x HX keys (14 x 14 for the 7 x 7 window).  A (tile, plane) pair is an ITEM:
//   issuer  : S[g & 1] = Q~ K~^T over the WHOLE plane (one commit)            N = 208 columns of TMEM
//   softmax : 16 warps.  Item g belongs to warp PAIR g & 1 (8 warps: two per TMEM subpartition).  A subpartition
//             holds the queries of 4 y rows of one level; they need at most NEED = 4 + kY - 1 of the HY key rows;
//             the two warps take half of those rows each: S rows -> registers (x folded, see below), both
//             meet at a 64-thread barrier (all reads done: P goes over the front of S), exp2 against the row's
//             reference, P (bf16) -> TMEM.
//   issuer  : O += P V (P is the TMEM A operand), then Q K^T of item g + 2 into the same buffer (the tensor pipe
//             executes in issue order).
// With two S buffers the two warp pairs work on consecutive planes at the same time: four softmax warps per
// scheduler hide each other's latencies, and a plane costs each warp one hand-off.
// TMEM (512 columns): O [0, 64) | S0 | S1 (2 x 208) | Q~ [480, 512) (bf16, the A operand of Q K^T).
//
// No running maximum, no rescaling, no reference at all: P = exp2(s * scale * log2 e).  With the inputs this path is
// built for (QK-RMSNorm: |logit| <= sqrt(d)) the exponentials sit in the middle of the fp32 / bf16
// exponent range; every plane uses the same (zero) reference, so O and the row sum need no correction, and a
// softmax warp needs nothing from the other warps that share its rows.  What can go wrong is a row whose
// exponentials leave the range: the epilogue checks the row sum (2^-80 < l < 2^100, i.e. the row maximum roughly
// within -55 .. +69), puts any other row on a list, and a small SIMT kernel recomputes the listed rows with a
// true two-pass softmax after the main kernel (na3d_fix_rows_kernel).  The result is exact either way.
//
// Warps (768 threads; registers via setmaxnreg: softmax 88, aux 104, control 24):
//   0-15   softmax (warp w: TMEM subpartition w & 3, pair w >> 3, half (w >> 2) & 1)
//   16-19  "aux", one per subpartition.  Per unit: coordinates of the halo -> (cos, sin) table in shared memory
//          (A1: fp32 fma chain, two-term Cody-Waite reduction, MUFU sin / cos, rounded to bf16; built once per unit
//          when the coordinates do not depend on the level -- the paper's case, PAPER.md:93-99 -- else per level).
//          Per tile: its query row global -> registers -> rotated (A2, packed bf16x2) -> TMEM; the epilogue of the
//          previous tile (O / l -> bf16 -> global, LSE).  Per plane: K rotated IN PLACE in shared memory.  For the
//          interleaved pairing the two halves of a pair are gathered into separate words and left in that order:
//          the same permutation of the 8 channels of every 16-byte chunk is applied to Q and K, which leaves
//          Q K^T unchanged.
//   20     TMA producer of K planes (ring of NSK stages); TMEM owner          21  MMA issuer, one elected lane
//   22     TMA producer of V planes (ring of NSV stages)                      23  idle (completes the warpgroup)
//
// x fold: the x window of a query covers kX of the HX halo columns; with kX <= HX / 2 at most one of the columns c
// and c + HX / 2 is inside it, so the two halves of every key row are FOLDED with a per-thread bit select before
// the exponential (half the MUFU work); P is packed to bf16 folded and un-folded by one byte permute per output
// word (a masked slot replicates the zero sign bit).
#include "tc_common.cuh"

namespace strata {
namespace {

using namespace tc;

template <int KY_, int KX_, int NSK_, int NSV_>
struct PlaneCfg {
  static constexpr int D = 64, KL = 3, KY = KY_, KX = KX_;
  static constexpr int TL = 2, TY = 8, TX = 8, M = 128;
  static constexpr int HY = TY + KY - 1, HX = TX + KX - 1, HALF = HX / 2;
  static constexpr int NTOK = HY * HX;                               // keys of a halo plane
  static constexpr int N = (NTOK + 15) / 16 * 16;                    // UMMA N (QK^T) / K extent (PV)
  static constexpr int G = 4;                                        // query rows (y) of a TMEM subpartition
  static constexpr int NEED = G + KY - 1;                            // key rows a subpartition can need
  static constexpr int NR = NEED / 2;                                // ... per softmax warp
  static constexpr int R0MAX = HY - NEED;                            // first needed key row is in [0, R0MAX]
  static constexpr int PW = HX / 2;                                  // packed P words per key row
  static constexpr int NF = (HALF + 1) / 2;                          // packed folded P words per key row
  static constexpr bool FULLFOLD = (KX == HALF);                     // exactly one of the columns c, c + HALF is in the window
  static constexpr int NSK = NSK_, NSV = NSV_;                       // K / V ring stages (a K plane is loaded and rotated well ahead)
  static constexpr int STAGE = N * 128;
  static constexpr int T_O = 0, T_S = D, T_Q = D + 2 * N, T_COLS = T_Q + D / 2;
  static constexpr int PADW = N / 2 - PW * HY;                       // P words behind the last key row
  static constexpr int NBARS = 3 * NSK + 2 * NSV + 8;
  static constexpr int CC_BYTES = NTOK * 16;
  static constexpr int XCH_BYTES = 2 * 4 * 128 * 4;                  // partial row sums
  static constexpr int SMEM_BYTES = 1024 + (NSK + NSV) * STAGE + STAGE + CC_BYTES + XCH_BYTES + 8 * NBARS + 16 + 512;
  static_assert(KY % 2 == 1 && KX % 2 == 1 && KY >= 3, "odd windows only (HX, HY even)");
  static_assert(KX <= HALF, "the x fold needs kX <= HX / 2");
  static_assert(HX <= 16 && NTOK <= 256, "halo of at most 256 keys per plane");
  static_assert(T_COLS <= 512, "TMEM columns");
  static_assert(NEED % 2 == 0 && N % 4 == 0, "key rows split between two warps");
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct PlaneParams {
  int B, H, L, Y, X;
  int nty, ntx;
  long long N;
  float scale_log2e;
  int A;          // rotary axes (0: no rotation)
  int ncols;      // level columns = B * H * nty * ntx
  int hg;         // heads per work unit
  unsigned long long* fix;   // [0] number of listed rows, [1] != 0: every row, [2 ...] the rows ((b * H + h) * N + token)
  unsigned int fix_cap;
};

constexpr int kPlaneThreads = 768;
constexpr int kWarpAux = 16, kWarpTma = 20, kWarpMma = 21, kWarpTmaV = 22;
constexpr int kBarPair = 1;               // named barriers 1-8: the two warps of a (pair, subpartition), 64 threads
constexpr int kBarAux = 13;               // the aux warpgroup, 128 threads
constexpr int kMaxLevels = 256;

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
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ float lds32(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
// One mbarrier arrival per WARP (barrier counts are in warps): every lane has made its own writes visible
// (fence.proxy.async / tcgen05.wait::st + tcgen05.fence::before_thread_sync) before the warp barrier; the
// arrival of lane 0 releases them cumulatively.
__device__ __forceinline__ void warp_arrive(uint32_t bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
// ---- A2 in packed bf16x2 arithmetic.  Table words: C = (cos m, cos m+1), S = (sin m, sin m+1).
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
  uint32_t nB;
  asm("neg.bf16x2 %0, %1;" : "=r"(nB) : "r"(B));
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
// One 16-byte chunk of an operand row against the table chunk at the same place (interleaved pairing).
__device__ __forceinline__ void rot_chunk(uint4& x, const uint4& t) {
  rot_interleaved(x.x, x.y, t.x, t.y);
  rot_interleaved(x.z, x.w, t.z, t.w);
}
// Half pairing: a = 8 channels j .. j+7, b = channels j + D/2 .. ; c, s = their cosines / sines.
__device__ __forceinline__ void rot_chunks_half(uint4& a, uint4& b, const uint4& c, const uint4& s) {
  rot2(a.x, b.x, c.x, s.x); rot2(a.y, b.y, c.y, s.y);
  rot2(a.z, b.z, c.z, s.z); rot2(a.w, b.w, c.w, s.w);
}
// A1: cos / sin of an fp32 angle.  The table is rounded to bf16 (2^-9): an fp32 angle (|phi| <~ 2e3 rad -> 1e-4 rad
// of rounding), a two-term Cody-Waite reduction to [-pi, pi] and the MUFU sin / cos (2^-21 abs on that range)
// are far inside that.
__device__ __forceinline__ void sincos_reduced(float phi, float& sn, float& cs) {
  const float n = rintf(phi * 0.15915494309189535f);
  const float r = fmaf(n, 1.7484555e-7f, fmaf(n, -6.2831854820251465f, phi));    // 2 pi = 6.2831854820251465 - 1.7484555e-7
  __sincosf(r, &sn, &cs);
}
// Pins a value in a register: the compiler can no longer re-derive it from its inputs at every use.
__device__ __forceinline__ uint32_t pinned(uint32_t x) {
  asm volatile("mov.u32 %0, %0;" : "+r"(x));
  return x;
}
// (a & m) | (b & ~m)
__device__ __forceinline__ uint32_t bitsel(uint32_t m, uint32_t a, uint32_t b) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, 0xCA;" : "=r"(d) : "r"(m), "r"(a), "r"(b));
  return d;
}

// Planes a query tile reaches: [plo, phi).
template <class C> __device__ __host__ __forceinline__ int tile_plo(int t, int L) { return window_start(C::TL * t, C::KL, L); }
template <class C> __device__ __host__ __forceinline__ int tile_phi(int t, int L) {
  const int last = C::TL * t + C::TL - 1;
  return window_start(last < L - 1 ? last : L - 1, C::KL, L) + C::KL;
}

// Shared-memory matrix descriptor from its low word (start address >> 4 | leading offset); the high word is the
// same for every operand here: 8-row groups 1024 bytes apart, version 1, 128-byte swizzle.
__device__ __forceinline__ uint32_t desc_lo(uint32_t addr) { return ((addr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ uint64_t desc_from_lo(uint32_t lo) { return ((uint64_t)0x40004040u << 32) | lo; }

// ------------------------------------------------------------------------------------------------
// Kernel
// ------------------------------------------------------------------------------------------------
template <class C, int PAIR>   // PAIR: strata_rope_pairing_t of the rotation
__global__ void __launch_bounds__(kPlaneThreads, 1)
na3d_fwd_plane_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
                      const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k, const float* __restrict__ coords,
                      const float* __restrict__ freqs, __nv_bfloat16* __restrict__ o, float* __restrict__ lse,
                      const PlaneParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  const uint32_t k_smem = base;                                        // [NSK] K planes
  const uint32_t v_smem = k_smem + C::NSK * C::STAGE;                  // [NSV] V planes
  const uint32_t t_smem = v_smem + C::NSV * C::STAGE;                   // (cos, sin) table of the halo, in K-plane geometry
  const uint32_t cc_smem = t_smem + C::STAGE;                          // coordinates of the halo tokens, float4 each
  const uint32_t lsum_sm = cc_smem + C::CC_BYTES;                      // [2 tile parities][4 warpgroups][128 rows] partial row sums
  const uint32_t bars = lsum_sm + 2 * 4 * 128 * 4;
  auto bar_kfull = [&](int s) { return bars + 8u * s; };                          // TMA -> aux
  auto bar_krot = [&](int s) { return bars + 8u * (C::NSK + s); };                // aux (4 warps) -> issuer
  auto bar_kempty = [&](int s) { return bars + 8u * (2 * C::NSK + s); };          // issuer commit (last Q K^T of the plane) -> TMA
  auto bar_vfull = [&](int s) { return bars + 8u * (3 * C::NSK + s); };           // TMA -> issuer
  auto bar_vempty = [&](int s) { return bars + 8u * (3 * C::NSK + C::NSV + s); }; // issuer commit (last P V of the plane) -> TMA
  const uint32_t bar_sfull = bars + 8u * (3 * C::NSK + 2 * C::NSV);               // [2] issuer commit -> softmax pair
  const uint32_t bar_pfull = bar_sfull + 16;                                      // [2] 8 softmax warps -> issuer
  const uint32_t bar_qready = bar_pfull + 16;                                     // aux (4 warps) -> issuer: Q~ of the tile is in TMEM
  const uint32_t bar_qfree = bar_qready + 8;                                      // issuer commit -> aux: every Q K^T of the tile is done
  const uint32_t bar_pvdone = bar_qfree + 8;                                      // issuer commit -> softmax pair of the tile's last plane: O is complete
  const uint32_t bar_ofree = bar_pvdone + 8;                                      // that pair (8 warps) -> issuer: O has been read out
  const uint32_t tmem_word = bars + 8u * C::NBARS;
  uint32_t* tmem_word_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_word - raw));
  uint8_t* lastuse = smem_raw + (tmem_word + 16 - raw);                // [L] last tile that needs the plane
  float4* cc = reinterpret_cast<float4*>(smem_raw + (cc_smem - raw));

  // (the shuffle makes the warp index provably warp-uniform for the compiler)
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  const int ntl = (p.L + C::TL - 1) / C::TL;

  // ---- geometry of one level column: head fastest, then x, y, sample.
  struct Col {
    int h, b, x0, y0, hs_x, hs_y;
  };
  auto column = [&](int col) {
    Col c;
    int bid = col;
    c.h = bid % p.H; bid /= p.H;
    const int tx = bid % p.ntx; bid /= p.ntx;
    const int ty = bid % p.nty;
    c.b = bid / p.nty;
    c.x0 = tx * C::TX; c.y0 = ty * C::TY;
    c.hs_x = window_start(c.x0, C::KX, p.X); c.hs_y = window_start(c.y0, C::KY, p.Y);
    return c;
  };
  // Walk over the columns of this CTA.  The columns of a unit differ in the head only.
  struct ColIter {
    Col c;
    int cl, hh;          // columns so far, head within the unit
    long long u;         // unit
  };
  auto col_begin = [&](ColIter& it) { it.cl = -1; it.hh = 0; it.u = 0; };
  auto col_advance = [&](ColIter& it) -> bool {
    ++it.cl;
    if (it.cl > 0 && ++it.hh < p.hg) { ++it.c.h; return true; }
    it.hh = 0;
    it.u = it.cl == 0 ? (long long)blockIdx.x : it.u + gridDim.x;
    if (it.u * p.hg >= p.ncols) return false;
    it.c = column((int)(it.u * p.hg));
    return true;
  };
  // columns this CTA works on
  const int nunits_cta = (int)(((long long)p.ncols / p.hg - (long long)blockIdx.x + gridDim.x - 1) / gridDim.x);
  const int ncols_cta = nunits_cta > 0 ? nunits_cta * p.hg : 0;

  // ---- one-time setup
  if (warp == kWarpTma && lane == 0) {
    tma_prefetch_desc(&tm_k); tma_prefetch_desc(&tm_v);
    for (int s = 0; s < C::NSK; ++s) { mbar_init(bar_kfull(s), 1); mbar_init(bar_krot(s), 4); mbar_init(bar_kempty(s), 1); }
    for (int s = 0; s < C::NSV; ++s) { mbar_init(bar_vfull(s), 1); mbar_init(bar_vempty(s), 1); }
    mbar_init(bar_sfull, 1); mbar_init(bar_sfull + 8, 1);
    mbar_init(bar_pfull, 8); mbar_init(bar_pfull + 8, 8);
    mbar_init(bar_qready, 4); mbar_init(bar_qfree, 1); mbar_init(bar_pvdone, 1); mbar_init(bar_ofree, 8);
    fence_barrier_init();
  }
  if (warp == kWarpTma) tmem_alloc(tmem_word, 512);
  for (int l = threadIdx.x; l < p.L; l += kPlaneThreads) {
    int lt = 0;
    for (int t = 0; t < ntl; ++t)
      if (l >= tile_plo<C>(t, p.L) && l < tile_phi<C>(t, p.L)) lt = t;
    lastuse[l] = (uint8_t)lt;
  }
  // K and V stages start as zeros: the rows behind the halo (N - NTOK) are keys outside every window (P = 0
  // there), which must hold finite numbers.
  for (uint32_t off = threadIdx.x * 16u; off < (uint32_t)(C::NSK + C::NSV) * C::STAGE; off += kPlaneThreads * 16u)
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(k_smem + off), "r"(0u) : "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_word_ptr;

  if (warp >= kWarpTma) reg_dec<24>();
  if (warp == kWarpTma || warp == kWarpTmaV) {
    // =========================== TMA producers: K planes (warp 20), V planes (warp 22) ===========================
    const bool isv = warp == kWarpTmaV;
    const int ns = isv ? C::NSV : C::NSK;
    const uint32_t stage0 = isv ? v_smem : k_smem;
    const CUtensorMap* map = isv ? &tm_v : &tm_k;
    ColIter it;
    col_begin(it);
    while (col_advance(it)) {
      const Col& c = it.c;
      for (int plane = 0; plane < p.L; ++plane) {
        const int li = it.cl * p.L + plane, s = li % ns;
        const uint32_t ph = (uint32_t)(li / ns) & 1u;
        const uint32_t full = isv ? bar_vfull(s) : bar_kfull(s);
        mbar_wait_bounded(isv ? bar_vempty(s) : bar_kempty(s), ph ^ 1u);
        if (elect_one()) {
          mbar_expect_tx(full, (uint32_t)(C::NTOK * 128));
          tma_load_5d(stage0 + s * C::STAGE, map, full, 0, c.h, c.hs_x, c.hs_y, c.b * p.L + plane);
        }
        __syncwarp();
      }
    }
  } else if (warp == kWarpMma) {
    // =========================== MMA issuer ===========================
    // The whole warp walks the item sequence in uniform control flow; one elected lane issues and commits.
    struct Cur {
      int cl, t, plane, plo, phi, tiles;   // tiles: tiles finished so far
      bool valid;
    };
    auto enter = [&](Cur& w) { w.plo = tile_plo<C>(w.t, p.L); w.phi = tile_phi<C>(w.t, p.L); w.plane = w.plo; };
    auto cur_init = [&](Cur& w) { w.cl = 0; w.t = 0; w.tiles = 0; w.valid = ncols_cta > 0; if (w.valid) enter(w); };
    auto cur_next = [&](Cur& w) {
      if (++w.plane < w.phi) return;
      ++w.tiles;
      if (++w.t >= ntl) { w.t = 0; if (++w.cl >= ncols_cta) { w.valid = false; return; } }
      enter(w);
    };
    Cur wq, wp;
    cur_init(wq); cur_init(wp);
    int iq = 0, ip = 0;
    constexpr uint32_t idesc_qk = instr_desc(C::M, C::N, false);
    constexpr uint32_t idesc_pv = instr_desc(C::M, C::D, true);

    auto issue_qk = [&]() {
      const int li = wq.cl * p.L + wq.plane, s = li % C::NSK;
      const uint32_t ph = (uint32_t)(li / C::NSK) & 1u;
      const bool first = wq.plane == wq.plo, last = wq.plane == wq.phi - 1;
      const bool release = (int)lastuse[wq.plane] == wq.t;
      if (first) mbar_wait<false>(bar_qready, (uint32_t)wq.tiles & 1u);          // Q~ of the tile is in TMEM
      mbar_wait<false>(bar_krot(s), ph);                                           // K plane rotated
      tc_fence_after();
      const uint32_t lo_k = desc_lo(k_smem + s * C::STAGE);
      const uint32_t d_tm = tmem + C::T_S + (iq & 1) * C::N;
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < C::D / 16; ++ks)
          umma_ts(d_tm, tmem + C::T_Q + 8u * ks, desc_from_lo(lo_k + 2u * ks), idesc_qk, ks > 0 ? 1u : 0u);
        umma_commit(bar_sfull + 8u * (iq & 1));
        if (release) umma_commit(bar_kempty(s));
        if (last) umma_commit(bar_qfree);
      }
      __syncwarp();
      ++iq;
      cur_next(wq);
    };
    auto issue_pv = [&]() {
      const int li = wp.cl * p.L + wp.plane, s = li % C::NSV;
      const uint32_t ph = (uint32_t)(li / C::NSV) & 1u;
      const bool first = wp.plane == wp.plo, last = wp.plane == wp.phi - 1;
      const bool release = (int)lastuse[wp.plane] == wp.t;
      mbar_wait<false>(bar_pfull + 8u * (ip & 1), (uint32_t)(ip >> 1) & 1u);      // P of the item is in TMEM
      mbar_wait<false>(bar_vfull(s), ph);
      if (first && wp.tiles > 0) mbar_wait<false>(bar_ofree, (uint32_t)(wp.tiles - 1) & 1u);   // O of the previous tile read out
      tc_fence_after();
      const uint32_t lo_v = desc_lo(v_smem + s * C::STAGE);
      const uint32_t a_tm = tmem + C::T_S + (ip & 1) * C::N;
      const uint32_t acc0 = first ? 0u : 1u;
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < C::N / 16; ++ks)
          umma_ts(tmem + C::T_O, a_tm + 8u * ks, desc_from_lo(lo_v + 128u * ks), idesc_pv, ks > 0 ? 1u : acc0);
        if (release) umma_commit(bar_vempty(s));
        if (last) umma_commit(bar_pvdone);
      }
      __syncwarp();
      ++ip;
      cur_next(wp);
    };
    if (wq.valid) issue_qk();
    if (wq.valid) issue_qk();
    while (wp.valid) {
      issue_pv();
      if (wq.valid) issue_qk();
    }
  } else if (warp > kWarpTmaV) {
    // (idle)
  } else if (warp >= kWarpAux) {
    // =========================== aux warpgroup ===========================
    reg_inc<104>();
    const int tid = threadIdx.x - 32 * kWarpAux;
    const int sp = warp & 3;
    const int row = sp * 32 + lane;                 // query row of the tile == TMEM lane
    const int qx = row % C::TX, qy = (row / C::TX) % C::TY, ql = row / (C::TX * C::TY);
    const uint32_t tm = tmem + ((uint32_t)(sp * 32) << 16);
    const bool rope = p.A > 0;
    constexpr int NPF = PAIR ? 8 : 4;                                  // rotary pairs per table work item
    // logical 16-byte chunk this thread owns in the plane-linear loops below
    const int cch = PAIR ? (tid & 3) : ((tid & 7) ^ ((tid >> 3) & 7));

    // A1, once per unit: coordinates of the halo of column c (this thread: halo tokens tid, tid + 128, row-major)
    // -> (cos, sin) of every halo token and rotary pair -> table, in the layout of a K plane.  The coordinates of
    // a column must not depend on the level (they are a function of the token's (lat, lon)); if
    // they do, every row of the problem is handed to the fix-up kernel, which takes each token's own coordinates.
    auto build_table = [&](const Col& c) {
      bar_sync(kBarAux, 128);                       // everyone is done with the current table and cache
      bool diff = false;
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int tok = tid + 128 * j;
        if (tok >= C::NTOK) continue;
        const int hyr = tok / C::HX, hx = tok - hyr * C::HX;
        const int y = min(c.hs_y + hyr, p.Y - 1), x = min(c.hs_x + hx, p.X - 1);
        const float* src = coords + ((((long long)c.b * p.L) * p.Y + y) * p.X + x) * p.A;
        const long long lstride = (long long)p.Y * p.X * p.A;
        float4 v = make_float4(src[0], p.A > 1 ? src[1] : 0.f, 0.f, 0.f);
#pragma unroll 1
        for (int l = 1; l < p.L; ++l) {
          const float* sl = src + l * lstride;
          diff |= __float_as_uint(sl[0]) != __float_as_uint(v.x);
          if (p.A > 1) diff |= __float_as_uint(sl[1]) != __float_as_uint(v.y);
        }
        cc[tok] = v;
      }
      if (diff) p.fix[1] = 1ull;                    // (any thread: the whole problem goes to the fix-up kernel)
      bar_sync(kBarAux, 128);
      float fr[2][NPF];
#pragma unroll
      for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int u = 0; u < NPF; ++u) fr[a][u] = (a < p.A) ? __ldg(freqs + a * (C::D / 2) + NPF * cch + u) : 0.f;
      if constexpr (PAIR == 0) {
#pragma unroll 1
        for (int qi = tid; qi < C::NTOK * 8; qi += 128) {
          const float4 xyz = cc[qi >> 3];
          float cs[4], sn[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) sincos_reduced(fmaf(xyz.y, fr[1][u], xyz.x * fr[0][u]), sn[u], cs[u]);
          uint4 w;
          w.x = pack_bf16(cs[0], cs[1]); w.y = pack_bf16(sn[0], sn[1]);
          w.z = pack_bf16(cs[2], cs[3]); w.w = pack_bf16(sn[2], sn[3]);
          sts128(t_smem + qi * 16, w);
        }
      } else {
#pragma unroll 1
        for (int qi = tid; qi < C::NTOK * 4; qi += 128) {
          const int r = qi >> 2;
          const float4 xyz = cc[r];
          float cs[8], sn[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) sincos_reduced(fmaf(xyz.y, fr[1][u], xyz.x * fr[0][u]), sn[u], cs[u]);
          uint4 wc, ws;
          wc.x = pack_bf16(cs[0], cs[1]); wc.y = pack_bf16(cs[2], cs[3]); wc.z = pack_bf16(cs[4], cs[5]); wc.w = pack_bf16(cs[6], cs[7]);
          ws.x = pack_bf16(sn[0], sn[1]); ws.y = pack_bf16(sn[2], sn[3]); ws.z = pack_bf16(sn[4], sn[5]); ws.w = pack_bf16(sn[6], sn[7]);
          const uint32_t rb = t_smem + r * 128, sw = (uint32_t)(r & 7);
          sts128(rb + (((uint32_t)cch ^ sw) << 4), wc);
          sts128(rb + (((uint32_t)(cch + 4) ^ sw) << 4), ws);
        }
      }
      bar_sync(kBarAux, 128);
    };

    auto q_row = [&](const Col& c, int t) {
      const int lv = min(C::TL * t + ql, p.L - 1), y = min(c.y0 + qy, p.Y - 1), x = min(c.x0 + qx, p.X - 1);
      const long long tok = ((long long)lv * p.Y + y) * p.X + x;
      return q + (((long long)c.b * p.N + tok) * p.H + c.h) * C::D;
    };
    // The query row of a tile: global -> registers (a tile ahead) -> rotated (A2) -> TMEM (bf16 pairs, K-major: the A
    // operand of Q K^T).  T: running number of the tile.
    uint4 qr[8];
    auto q_fetch = [&](const Col& c, int t) {
      const uint4* src = reinterpret_cast<const uint4*>(q_row(c, t));
#pragma unroll
      for (int j = 0; j < 8; ++j) qr[j] = __ldg(src + j);
    };
    auto q_task = [&](const Col& c, int t, int T) {
      if (rope) {
        const int tr = (qy + c.y0 - c.hs_y) * C::HX + qx + c.x0 - c.hs_x;       // table row of the query's token
        const uint32_t trb = t_smem + tr * 128, tsw = (uint32_t)(tr & 7);
        if constexpr (PAIR == 0) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const uint4 tb = lds128(trb + (((uint32_t)j ^ tsw) << 4));
            rot_chunk(qr[j], tb);
          }
        } else {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint4 tc_ = lds128(trb + (((uint32_t)j ^ tsw) << 4)), ts_ = lds128(trb + (((uint32_t)(j + 4) ^ tsw) << 4));
            rot_chunks_half(qr[j], qr[j + 4], tc_, ts_);
          }
        }
      }
      if (T > 0) { mbar_wait(bar_qfree, (uint32_t)(T - 1) & 1u); tc_fence_after(); }   // every Q K^T of the previous tile is done
      uint32_t w[32];
#pragma unroll
      for (int j = 0; j < 8; ++j) { w[4 * j] = qr[j].x; w[4 * j + 1] = qr[j].y; w[4 * j + 2] = qr[j].z; w[4 * j + 3] = qr[j].w; }
      tmem_st_n<32>(tm + C::T_Q, w);
      tmem_wait_st();
      tc_fence_before();
      warp_arrive(bar_qready);
    };
    // K plane `plane` of column number cl: rotate in place (A2), hand to the issuer.  The table has the K plane's
    // geometry, so the work is linear over physical 16-byte chunks: chunk tid + 128 j, all offsets immediates.
    auto rot_k = [&](int cl, int plane) {
      const int li = cl * p.L + plane, s = li % C::NSK;
      mbar_wait(bar_kfull(s), (uint32_t)(li / C::NSK) & 1u);
      if (rope) {
        if constexpr (PAIR == 0) {
          constexpr int nch = C::NTOK * 8, FULL = nch / 128, REM = nch % 128;
          const uint32_t kb = k_smem + s * C::STAGE + tid * 16, tb = t_smem + tid * 16;
#pragma unroll
          for (int j0 = 0; j0 < FULL; j0 += 4) {
            uint4 x[4], t[4];
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (j0 + j < FULL) { x[j] = lds128(kb + (j0 + j) * 2048); t[j] = lds128(tb + (j0 + j) * 2048); }
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (j0 + j < FULL) { rot_chunk(x[j], t[j]); sts128(kb + (j0 + j) * 2048, x[j]); }
          }
          if (REM > 0 && tid < REM) {
            uint4 x = lds128(kb + FULL * 2048);
            const uint4 t = lds128(tb + FULL * 2048);
            rot_chunk(x, t);
            sts128(kb + FULL * 2048, x);
          }
        } else {
          // item tid + 128 j: row (tid >> 2) + 32 j, logical chunks cch (channels a) and cch + 4 (channels b)
          constexpr int nit = C::NTOK * 4, FULL = nit / 128, REM = nit % 128;
          const uint32_t r0 = (uint32_t)(tid >> 2), sw = r0 & 7u;
          const uint32_t oa = r0 * 128 + (((uint32_t)cch ^ sw) << 4), ob = r0 * 128 + (((uint32_t)(cch + 4) ^ sw) << 4);
          const uint32_t kb = k_smem + s * C::STAGE;
#pragma unroll
          for (int j0 = 0; j0 < FULL; j0 += 2) {
            uint4 a[2], b[2], tc_[2], ts_[2];
#pragma unroll
            for (int j = 0; j < 2; ++j)
              if (j0 + j < FULL) {
                a[j] = lds128(kb + oa + (j0 + j) * 4096); b[j] = lds128(kb + ob + (j0 + j) * 4096);
                tc_[j] = lds128(t_smem + oa + (j0 + j) * 4096); ts_[j] = lds128(t_smem + ob + (j0 + j) * 4096);
              }
#pragma unroll
            for (int j = 0; j < 2; ++j)
              if (j0 + j < FULL) {
                rot_chunks_half(a[j], b[j], tc_[j], ts_[j]);
                sts128(kb + oa + (j0 + j) * 4096, a[j]); sts128(kb + ob + (j0 + j) * 4096, b[j]);
              }
          }
          if (REM > 0 && tid < REM) {
            uint4 a = lds128(kb + oa + FULL * 4096), b = lds128(kb + ob + FULL * 4096);
            const uint4 tc_ = lds128(t_smem + oa + FULL * 4096), ts_ = lds128(t_smem + ob + FULL * 4096);
            rot_chunks_half(a, b, tc_, ts_);
            sts128(kb + oa + FULL * 4096, a); sts128(kb + ob + FULL * 4096, b);
          }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      }
      warp_arrive(bar_krot(s));
    };

    // ---- static task order.  The K ring is one stage deeper than a tile needs, so the planes
    // new to a tile are rotated a tile ahead.  Per tile T: Q~(T) -> TMEM (the row was fetched a tile ago; fetch the
    // next, its reference) | the table of the next unit if one starts | the K planes new to tile T + 1.
    // Every wait of this sequence depends only on tasks that precede it: the ring slot of plane p is released by
    // the last Q K^T of plane p - NSK, which is one of the first two items of tile T (issued as soon as Q~(T) and
    // its planes are there) or earlier.
    ColIter it;
    col_begin(it);
    bool more = col_advance(it);
    int t = 0, T = 0;
    if (more) {
      q_fetch(it.c, 0);
      if (rope) build_table(it.c);
#pragma unroll 1
      for (int pl = 0; pl < tile_phi<C>(0, p.L); ++pl) rot_k(0, pl);
    }
    while (more) {
      const Col c = it.c;
      const int cl = it.cl;
      q_task(c, t, T);
      // the tile after this one
      const bool same_col = t + 1 < ntl;
      bool have_next = same_col;
      if (!same_col) { more = col_advance(it); have_next = more; }
      if (have_next) {
        q_fetch(same_col ? c : it.c, same_col ? t + 1 : 0);
        if (rope && !same_col && it.hh == 0) build_table(it.c);
        const int pa = same_col ? tile_phi<C>(t, p.L) : 0, pb = tile_phi<C>(same_col ? t + 1 : 0, p.L);
#pragma unroll 1
        for (int pl = pa; pl < pb; ++pl) rot_k(same_col ? cl : it.cl, pl);
      }
      ++T;
      t = same_col ? t + 1 : 0;
    }
  } else {
    // =========================== softmax ===========================
    reg_inc<88>();
    const int pair = warp >> 3, half = (warp >> 2) & 1, wg = warp >> 2;
    const int sp = warp & 3;                        // TMEM subpartition
    const int row = sp * 32 + lane;                 // query row of the tile == TMEM lane
    const int qx = row % C::TX, qy = (row / C::TX) % C::TY, ql = row / (C::TX * C::TY);
    const uint32_t s_tm = pinned(tmem + ((uint32_t)(sp * 32) << 16) + C::T_S + pair * C::N);   // S of this pair's items; P goes over its front
    const float cs = p.scale_log2e;
    const uint32_t bar_s = pinned(bar_sfull + 8u * pair), bar_p = pinned(bar_pfull + 8u * pair);
    const uint32_t bar_pr = pinned((uint32_t)(kBarPair + pair * 4 + sp));
    const uint32_t lane0 = pinned(lane == 0 ? 1u : 0u);
    const uint32_t ls_base = pinned(lsum_sm + (uint32_t)(wg * 128 + row) * 4u);
    const uint32_t ls_row = pinned(lsum_sm + (uint32_t)row * 4u);
    const uint32_t o_tm = pinned(tmem + ((uint32_t)(sp * 32) << 16) + C::T_O + half * (C::D / 2));   // this warp's half of the O row
    int ax = 0, ay = 0;                             // this query's token (clamped to the grid)
    bool active_xy = false;

    // per-unit constants of this query row (the columns of a unit share the tile, hence the windows)
    int rw = 0;                                     // first key row of this warp
    int r0 = 0;                                     // first key row the subpartition needs
    uint32_t rowbits = 0;                           // halo rows inside this query's window, from row rw
    uint32_t m_lo[C::HALF];                         // x fold: all ones: column c is in the window (else c + HALF, or neither)
    float xz[C::HALF];                              // 0 if one of the two is in the window, else -inf
    uint32_t psel[C::PW];                           // un-fold selectors, see below
    int g = 0, T = 0;                               // item / tile counters of the CTA
    ColIter it;
    col_begin(it);
    while (col_advance(it)) {
      const Col& c = it.c;
      if (it.hh == 0) {
        ax = min(c.x0 + qx, p.X - 1); ay = min(c.y0 + qy, p.Y - 1);
        active_xy = c.x0 + qx < p.X && c.y0 + qy < p.Y;
        const int lo_x = window_start(ax, C::KX, p.X) - c.hs_x;
        const int lo_y = window_start(ay, C::KY, p.Y) - c.hs_y;
        r0 = min(__reduce_min_sync(0xffffffffu, lo_y), C::R0MAX);
        rw = r0 + half * C::NR;
        rowbits = (((1u << C::KY) - 1u) << lo_y) >> rw;
#pragma unroll
        for (int cc_ = 0; cc_ < C::HALF; ++cc_) {
          const bool in_lo = cc_ >= lo_x && cc_ < lo_x + C::KX, in_hi = cc_ + C::HALF >= lo_x && cc_ + C::HALF < lo_x + C::KX;
          m_lo[cc_] = in_lo ? 0xffffffffu : 0u;
          xz[cc_] = (in_lo || in_hi) ? 0.f : -INFINITY;
        }
        // un-fold: P word j holds the halo columns (2j, 2j+1).  Column col comes from the folded value
        // fc = col mod HALF, which sits in half (fc & 1) of the packed word F[fc / 2]; psel[j] is the byte
        // selector of prmt(F[fc(2j) / 2], F[fc(2j+1) / 2]).  A column outside the window selects "sign of a
        // high byte", which is 0x00 because every P value is >= +0.
#pragma unroll
        for (int j = 0; j < C::PW; ++j) {
          const int c0 = 2 * j, c1 = 2 * j + 1;
          const int f0 = c0 % C::HALF, f1 = c1 % C::HALF;
          const bool v0 = c0 >= lo_x && c0 < lo_x + C::KX, v1 = c1 >= lo_x && c1 < lo_x + C::KX;
          const uint32_t n0 = v0 ? (uint32_t)(2 * (f0 & 1)) | ((uint32_t)(2 * (f0 & 1) + 1) << 4) : 0x99u;
          const uint32_t n1 = v1 ? (uint32_t)(4 + 2 * (f1 & 1)) | ((uint32_t)(5 + 2 * (f1 & 1)) << 4) : 0xDDu;
          psel[j] = n0 | (n1 << 8);
        }
      }

      for (int tile = 0; tile < ntl; ++tile, ++T) {
        const int al = min(C::TL * tile + ql, p.L - 1);
        const int pw_lo = window_start(al, C::KL, p.L);              // planes of this query (warp-uniform): [pw_lo, pw_lo + KL)
        const int plo = tile_plo<C>(tile, p.L), phi = tile_phi<C>(tile, p.L);
        float lsum = 0.f;
#pragma unroll 1
        for (int plane = plo; plane < phi; ++plane, ++g) {
          if ((g & 1) != pair) continue;
          const bool needed = plane >= pw_lo && plane < pw_lo + C::KL;
          mbar_wait(bar_s, (uint32_t)(g >> 1) & 1u);
          tc_fence_after();
          if (!needed) {
            // no query of this subpartition attends a key of this plane: P = 0 (this warp's half of the words)
            constexpr int NZ = C::N / 4;
            uint32_t z[NZ];
#pragma unroll
            for (int u = 0; u < NZ; ++u) z[u] = 0u;
            tmem_st_n<NZ>(s_tm + half * NZ, z);
          } else {
            // ---- this warp's key rows of S -> registers, folded; two rows per TMEM load
            float v[C::NR][C::HALF];
            {
              const uint32_t s_row = s_tm + rw * C::HX;
#pragma unroll
              for (int r = 0; r < C::NR; r += 2) {
                uint32_t sv[32];
                if (r + 1 < C::NR) { tmem_ld_x32(s_row + r * C::HX, sv); tmem_wait_ld(); reg_fence_16(sv); reg_fence_16(sv + 16); }
                else { tmem_ld_x16(s_row + r * C::HX, sv); tmem_wait_ld(); reg_fence_16(sv); }   // (columns behind the row: the next row or pad)
#pragma unroll
                for (int q2 = 0; q2 < 2; ++q2)
                  if (r + q2 < C::NR) {
#pragma unroll
                    for (int cc_ = 0; cc_ < C::HALF; ++cc_)
                      v[r + q2][cc_] = __uint_as_float(bitsel(m_lo[cc_], sv[q2 * C::HX + cc_], sv[q2 * C::HX + cc_ + C::HALF]));
                  }
              }
            }
            // P goes over the front of S.  The P rows of the first warp land on S rows it has read itself (P row r is
            // in S row r / 2); those of the second warp land on S rows of the first: it waits (below, before its
            // stores) until the first one has its rows in registers.
            if (half == 0) bar_arrive(bar_pr, 64);
            // ---- exponentials, row sums, P (bf16, un-folded) over the S rows
            uint32_t pw[C::NR * C::PW];
            float e0 = 0.f, e1 = 0.f;
#pragma unroll
            for (int r = 0; r < C::NR; ++r) {
              const float br = ((rowbits >> r) & 1u) ? 0.f : -INFINITY;
              float pr[C::HALF + 1];
              pr[C::HALF] = 0.f;
#pragma unroll
              for (int cc_ = 0; cc_ < C::HALF; cc_ += 2) {
                if (cc_ + 1 < C::HALF) {
                  float t0, t1;
                  if (C::FULLFOLD) ffma2(t0, t1, v[r][cc_], v[r][cc_ + 1], cs, br, br);
                  else ffma2(t0, t1, v[r][cc_], v[r][cc_ + 1], cs, br + xz[cc_], br + xz[cc_ + 1]);
                  pr[cc_] = ex2(t0); pr[cc_ + 1] = ex2(t1);
                  fadd2(e0, e1, e0, e1, pr[cc_], pr[cc_ + 1]);
                } else {
                  pr[cc_] = ex2(fmaf(v[r][cc_], cs, C::FULLFOLD ? br : br + xz[cc_]));
                  e0 += pr[cc_];
                }
              }
              uint32_t f[C::NF];
#pragma unroll
              for (int m = 0; m < C::NF; ++m) f[m] = pack_bf16(pr[2 * m], pr[2 * m + 1]);
#pragma unroll
              for (int jj = 0; jj < C::PW; ++jj)
                pw[r * C::PW + jj] = prmt(f[((2 * jj) % C::HALF) / 2], f[((2 * jj + 1) % C::HALF) / 2], psel[jj]);
            }
            lsum += e0 + e1;
            if (half == 1) bar_sync(bar_pr, 64);
            tmem_st_n<C::NR * C::PW>(s_tm + rw * C::PW, pw);
            // ---- key rows no query of the subpartition attends, pad keys: P = 0.  Away from the grid border the
            // needed rows are the first or the last NEED rows of the halo.
            constexpr int ZW = C::R0MAX * C::PW + C::PADW;
            uint32_t z[ZW];
#pragma unroll
            for (int u = 0; u < ZW; ++u) z[u] = 0u;
            if (half == 0) {
              if (r0 == C::R0MAX) tmem_st_n<C::R0MAX * C::PW>(s_tm, z);
              else {
#pragma unroll
                for (int kk = 0; kk < C::R0MAX; ++kk)
                  if (kk < r0) tmem_st_n<C::PW>(s_tm + kk * C::PW, z);
              }
            } else {
              if (r0 == 0) tmem_st_n<ZW>(s_tm + C::NEED * C::PW, z);
              else {
#pragma unroll
                for (int kk = 0; kk < C::R0MAX; ++kk)
                  if (r0 + C::NEED + kk < C::HY) tmem_st_n<C::PW>(s_tm + (r0 + C::NEED + kk) * C::PW, z);
                if constexpr (C::PADW > 0) tmem_st_n<C::PADW>(s_tm + C::HY * C::PW, z);
              }
            }
            sts32(ls_base + (uint32_t)(T & 1) * 2048u, lsum);
          }
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane0) mbar_arrive(bar_p);
          if (plane == phi - 1) {
            // ---- this pair handled the last plane of the tile: its epilogue (O / l -> bf16 -> global, LSE), in the
            // shadow of the P V and Q K^T the pair waits for anyway.  Each of the two warps of a subpartition takes
            // half of the O row.
            mbar_wait_bounded(bar_pvdone, (uint32_t)T & 1u);
            tc_fence_after();
            const uint32_t la = ls_row + (uint32_t)(T & 1) * 2048u;      // (read before O is released: tile T + 2 reuses the slots)
            const float ltot = (lds32(la) + lds32(la + 512)) + (lds32(la + 1024) + lds32(la + 1536));
            uint32_t ov[C::D / 2];
            tmem_ld_n<C::D / 2>(o_tm, ov);
            tc_fence_before();
            __syncwarp();
            if (lane0) mbar_arrive(bar_ofree);                       // O is in registers: the next tile may overwrite it
            if (active_xy && C::TL * tile + ql < p.L) {
              const float inv = 1.f / ltot;
              const long long tok = ((long long)al * p.Y + ay) * p.X + ax;
              __nv_bfloat16* orow = o + (((long long)c.b * p.N + tok) * p.H + c.h) * C::D + half * (C::D / 2);
#pragma unroll
              for (int u = 0; u < C::D / 2; u += 8) {
                uint4 w0;
                w0.x = pack_bf16(__uint_as_float(ov[u]) * inv, __uint_as_float(ov[u + 1]) * inv);
                w0.y = pack_bf16(__uint_as_float(ov[u + 2]) * inv, __uint_as_float(ov[u + 3]) * inv);
                w0.z = pack_bf16(__uint_as_float(ov[u + 4]) * inv, __uint_as_float(ov[u + 5]) * inv);
                w0.w = pack_bf16(__uint_as_float(ov[u + 6]) * inv, __uint_as_float(ov[u + 7]) * inv);
                reinterpret_cast<uint4*>(orow + u)[0] = w0;
              }
              if (half == 0) {
                const long long rid = ((long long)c.b * p.H + c.h) * p.N + tok;
                lse[rid] = log2f(ltot) * 0.69314718055994531f;
                if (!(ltot < kRowSumMax && ltot > kRowSumMin)) {   // out of the safe range (or NaN): the fix-up kernel recomputes the row
                  const unsigned long long idx = atomicAdd(p.fix, 1ull);
                  if (idx < p.fix_cap) p.fix[2 + idx] = (unsigned long long)rid;
                }
              }
            }
          }
        }
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
// Fix-up: the listed rows recomputed with a true two-pass softmax from the RAW Q, K (one warp per row, lane j owns the
// rotary pairs j, j + 32, ... of the D / 2; fp64 angle).  Rare by construction; correctness over speed.
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128)
na3d_fix_rows_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k,
                     const __nv_bfloat16* __restrict__ v, const float* __restrict__ coords,
                     const float* __restrict__ freqs, __nv_bfloat16* __restrict__ o, float* __restrict__ lse,
                     const unsigned long long* __restrict__ fix, unsigned int cap, Problem p) {
  constexpr int NP = D / 64;                                        // rotary pairs per lane
  const unsigned long long listed = fix[0];
  const bool all = listed > cap || fix[1] != 0;                     // the list overflowed / level-dependent coordinates: every row
  if (listed == 0 && !all) return;
  const unsigned long long total = all ? (unsigned long long)p.rows() : listed;
  const int lane = threadIdx.x & 31;
  const unsigned long long w0 = (unsigned long long)blockIdx.x * 4 + (threadIdx.x >> 5), nw = (unsigned long long)gridDim.x * 4;
  int c0[NP], c1[NP];
  float f[NP][3];
#pragma unroll
  for (int u = 0; u < NP; ++u) {
    const int j = lane + 32 * u;
    c0[u] = p.pairing ? j : 2 * j; c1[u] = p.pairing ? j + D / 2 : 2 * j + 1;
    for (int a = 0; a < 3; ++a) f[u][a] = (a < p.A) ? freqs[a * (D / 2) + j] : 0.f;
  }
  auto rotated = [&](const __nv_bfloat16* x, long long b, long long tok, int h, float (&ra)[NP], float (&rb)[NP]) {
    const __nv_bfloat16* src = x + ((b * p.N + tok) * p.H + h) * D;
#pragma unroll
    for (int u = 0; u < NP; ++u) {
      const float a_ = __bfloat162float(src[c0[u]]), b_ = __bfloat162float(src[c1[u]]);
      double phi = 0.0;
      for (int a = 0; a < p.A && a < 3; ++a) phi += (double)coords[(b * p.N + tok) * p.A + a] * (double)f[u][a];
      double sn, cs;
      sincos(phi, &sn, &cs);
      ra[u] = (float)(a_ * cs - b_ * sn); rb[u] = (float)(a_ * sn + b_ * cs);
    }
  };
  for (unsigned long long i = w0; i < total; i += nw) {
    const unsigned long long rid = all ? i : fix[2 + i];          // (b * H + h) * N + token
    const long long tok = (long long)(rid % (unsigned long long)p.N);
    const int h = (int)((rid / (unsigned long long)p.N) % (unsigned long long)p.H);
    const long long b = (long long)(rid / (unsigned long long)p.N / (unsigned long long)p.H);
    const int x = (int)(tok % p.X), y = (int)((tok / p.X) % p.Y), l = (int)(tok / ((long long)p.X * p.Y));
    const int sl = window_start(l, p.kL, p.L), sy = window_start(y, p.kY, p.Y), sx = window_start(x, p.kX, p.X);
    float qa[NP], qb[NP];
    rotated(q, b, tok, h, qa, qb);
    float mx = -INFINITY;
    for (int pass = 0; pass < 2; ++pass) {
      float sum = 0.f, oa[NP], ob[NP];
#pragma unroll
      for (int u = 0; u < NP; ++u) { oa[u] = 0.f; ob[u] = 0.f; }
      for (int dl = 0; dl < p.kL; ++dl)
        for (int dy = 0; dy < p.kY; ++dy)
          for (int dx = 0; dx < p.kX; ++dx) {
            const long long kt = ((long long)(sl + dl) * p.Y + sy + dy) * p.X + sx + dx;
            float ka[NP], kb[NP];
            rotated(k, b, kt, h, ka, kb);
            float s = 0.f;
#pragma unroll
            for (int u = 0; u < NP; ++u) s += qa[u] * ka[u] + qb[u] * kb[u];
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
            s *= p.scale;
            if (pass == 0) { mx = fmaxf(mx, s); continue; }
            const float pr = expf(s - mx);
            const __nv_bfloat16* vs = v + ((b * p.N + kt) * p.H + h) * D;
            sum += pr;
#pragma unroll
            for (int u = 0; u < NP; ++u) { oa[u] += pr * __bfloat162float(vs[c0[u]]); ob[u] += pr * __bfloat162float(vs[c1[u]]); }
          }
      if (pass == 1) {
        __nv_bfloat16* dst = o + ((b * p.N + tok) * p.H + h) * D;
#pragma unroll
        for (int u = 0; u < NP; ++u) { dst[c0[u]] = __float2bfloat16_rn(oa[u] / sum); dst[c1[u]] = __float2bfloat16_rn(ob[u] / sum); }
        if (lane == 0) lse[rid] = mx + logf(sum);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------------

template <class C>
bool plane_shape_ok(const Problem& p) {
  const int ntl = (p.L + C::TL - 1) / C::TL;
  if (p.L > kMaxLevels || p.L < C::KL || ntl > 255) return false;
  return true;
}

// K / V plane of the halo: [HX x HY] tokens of one head and level, 128-byte rows
template <class C>
bool make_plane_map(CUtensorMap* map, const void* ptr, const Problem& p) { return make_map(map, ptr, p, C::HX, C::HY, 1); }

DeviceState g_states[64];
std::mutex g_mu;

template <class C>
cudaError_t launch_plane(const Problem& p, int cfg_index, const void* q, const void* k, const void* v, const float* coords,
                         const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches) {
  CUtensorMap tk, tv;
  if (!make_plane_map<C>(&tk, k, p) || !make_plane_map<C>(&tv, v, p)) return cudaErrorInvalidValue;
  PlaneParams sp;
  sp.B = p.B; sp.H = p.H; sp.L = p.L; sp.Y = p.Y; sp.X = p.X; sp.N = p.N;
  sp.nty = (p.Y + C::TY - 1) / C::TY; sp.ntx = (p.X + C::TX - 1) / C::TX;
  sp.scale_log2e = p.scale * 1.4426950408889634f;
  sp.A = p.A;
  sp.fix = reinterpret_cast<unsigned long long*>(fix);
  sp.fix_cap = kFixCap;
  const long long ncols = (long long)p.B * p.H * sp.nty * sp.ntx;
  if (ncols > 0x7fffffffLL / 256) return cudaErrorInvalidValue;
  sp.ncols = (int)ncols;
  DeviceState* ds = device_state(g_states, g_mu);
  if (!ds) return cudaErrorInvalidDevice;
  // Heads per unit: as many as possible (the rotary table of a tile is built once per unit) while the units still
  // spread evenly over the SMs (at most ~3 % more units on the busiest CTA than on average).
  int hg = 1;
  for (int d = p.H; d >= 1; --d) {
    if (p.H % d) continue;
    const long long units = ncols / d, per = (units + ds->sm_count - 1) / ds->sm_count;
    if (units >= ds->sm_count && per * ds->sm_count * 100 <= units * 103) { hg = d; break; }
  }
  sp.hg = hg;
  const long long nunits = ncols / hg;
  const long long grid = nunits < ds->sm_count ? nunits : ds->sm_count;      // persistent: one CTA per SM
  auto kernel = p.pairing ? na3d_fwd_plane_kernel<C, 1> : na3d_fwd_plane_kernel<C, 0>;
  const int ai = 2 * cfg_index + (p.pairing ? 1 : 0);
  cudaError_t e = ensure_smem_attr(ds, g_mu, ai, kernel, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(fix, 0, 16, stream);
  if (e != cudaSuccess) return e;
  prof_begin("na3d_fwd_plane", stream);
  kernel<<<(unsigned)grid, kPlaneThreads, C::SMEM_BYTES, stream>>>(tk, tv, (const __nv_bfloat16*)q, (const __nv_bfloat16*)k, coords, freqs,
                                                                  (__nv_bfloat16*)o, lse, sp);
  prof_end(stream);
  if (launches) ++*launches;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_fix_rows(p, q, k, v, coords, freqs, o, lse, fix, stream, launches);
}

}  // namespace

// (index, kY, kX, K stages, V stages) instantiations (head_dim 64, k_L = 3).
#define STRATA_PLANE_CONFIGS(X) \
  X(0, 7, 7, 4, 3)              \
  X(1, 5, 5, 4, 3)              \
  X(2, 3, 3, 4, 3)

size_t plane_fwd_workspace_bytes() { return 16 + 8 * (size_t)kFixCap; }

// The rows listed in `fix` (plane_fwd_workspace_bytes() of device memory: [0] count, [1] != 0: every row, [2 ...] row
// ids), recomputed with the two-pass SIMT softmax.  head_dim 64 or 128, bf16.
cudaError_t launch_fix_rows(const Problem& p, const void* q, const void* k, const void* v, const float* coords,
                            const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches) {
  if (p.D != 64 && p.D != 128) return cudaErrorInvalidValue;
  prof_begin("na3d_fix_rows", stream);
  auto kernel = p.D == 64 ? na3d_fix_rows_kernel<64> : na3d_fix_rows_kernel<128>;
  // One warp per listed row, grid-stride.  8 blocks of 4 warps per SM: an empty list costs the same few microseconds
  // as a smaller grid (every block reads two words and returns), while the take-all case (list overflow, level-dependent
  // coordinates: every row of the problem) gets 32 warps per SM instead of 4 to hide its fp64 sincos and gather latency.
  kernel<<<148 * 8, 128, 0, stream>>>((const __nv_bfloat16*)q, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, coords, freqs,
                                  (__nv_bfloat16*)o, lse, reinterpret_cast<const unsigned long long*>(fix), kFixCap, p);
  prof_end(stream);
  if (launches) ++*launches;
  return cudaGetLastError();
}

bool plane_fwd_supported(const Problem& p) {
  if (p.dtype != 1 || p.D != 64 || p.kL != 3 || p.A > 2) return false;   // (A = 3: the level is a rotary axis, no shared table)
#define X(I_, KY_, KX_, NSK_, NSV_)                           \
  if (p.kY == KY_ && p.kX == KX_) return plane_shape_ok<PlaneCfg<KY_, KX_, NSK_, NSV_>>(p);
  STRATA_PLANE_CONFIGS(X)
#undef X
  return false;
}

cudaError_t launch_fwd_plane(const Problem& p, const void* q, const void* k, const void* v, const float* coords,
                             const float* freqs, void* o, float* lse, void* fix, cudaStream_t stream, int* launches) {
#define X(I_, KY_, KX_, NSK_, NSV_)                           \
  if (p.kY == KY_ && p.kX == KX_)                             \
    return launch_plane<PlaneCfg<KY_, KX_, NSK_, NSV_>>(p, I_, q, k, v, coords, freqs, o, lse, fix, stream, launches);
  STRATA_PLANE_CONFIGS(X)
#undef X
  return cudaErrorNotSupported;
}

}  // namespace strata
