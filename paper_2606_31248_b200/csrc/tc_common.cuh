// tc_common.cuh -- PTX wrappers (mbarrier, TMA, tcgen05 / TMEM), UMMA descriptors and the TMA tensor-map
// helper shared by the tensor-core kernels.  sm_100a only.
#pragma once
#include <cuda.h>

#include <mutex>

#include "common.cuh"

namespace strata {
namespace tc {

// ------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// try_wait blocks in hardware for a short, system-dependent time (about 40 cycles on B200) and returns false if
// the phase has not completed by then.  The wait loop is kept to two instructions (try_wait, branch): up to
// sixteen warps of a CTA sit in such loops, and every extra instruction per poll is taken from the issue slots
// of the working warps (a suspend-time hint, a nanosleep or a poll counter cost more than they save: the sleeps
// return after a few nanoseconds while other warps signal barriers).
template <bool SLEEP = true>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@!p bra WAIT_LOOP;\n\t}"
      :: "r"(bar), "r"(parity) : "memory");
}
// The same wait with a bound, for the waiters that are off the critical path (TMA producers, epilogues): every
// 65 536 failed polls (a millisecond or more) it looks at the global timer and traps once the wait has lasted more
// than kWaitBoundNs.  A protocol or parity bug normally stalls every role of a CTA, the producers and epilogues
// among them, so it ends as a failed launch (cudaErrorLaunchFailure) after a few seconds instead of a GPU that hangs
// until the process is killed.  No kernel of this library runs longer than tens of milliseconds.
constexpr unsigned long long kWaitBoundNs = 4000000000ull;
__device__ __forceinline__ void mbar_wait_bounded(uint32_t bar, uint32_t parity) {
  uint32_t polls = 0;
  unsigned long long t0 = 0;
  for (;;) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return;
    if ((++polls & 0xffffu) == 0) {
      unsigned long long now;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
      if (t0 == 0) t0 = now;
      else if (now - t0 > kWaitBoundNs) __trap();
    }
  }
}
// One lane of a converged warp (all 32 lanes must execute this).
__device__ __forceinline__ bool elect_one() {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok));
  return ok != 0;
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0,
                                            int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void umma_ss(uint32_t d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void umma_ts(uint32_t d, uint32_t a, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d), "r"(a), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr) : "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
        "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
               ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}
#include "tmem_regs.cuh"
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);   // .x (low 16 bits) = lo
  return *reinterpret_cast<uint32_t*>(&h);
}

// Shared-memory matrix descriptors (tcgen05, 128-byte swizzle, 8-row groups 1024 bytes apart).
//   K-major  (rows = M or N index, 64 contiguous bf16 of the contraction per row): Q tile, K chunk.
//   MN-major (rows = contraction index, 64 contiguous bf16 of N per row):          V chunk.
// bits [0,14) start >> 4 | [16,30) leading byte offset >> 4 | [32,46) stride byte offset >> 4 |
// [46,48) version = 1 | [61,64) layout = 2 (SWIZZLE_128B)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr) {
  return (uint64_t)((addr >> 4) & 0x3FFF) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}

// Instruction descriptor, kind::f16: D fp32 (bit 4), A = B = bf16 (bits 7, 10), N>>3 at 17, M>>4 at 24.
__host__ __device__ constexpr uint32_t instr_desc(int m, int n, bool b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)(m >> 4) << 24);
}


// ------------------------------------------------------------------------------------------------
// Host side: TMA tensor maps (driver entry point fetched through the runtime: no libcuda link)
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(sym);
    (void)cudaGetLastError();
  });
  return fn;
}

// Per-DEVICE launch state of one kernel family: the SM count and which kernels already have their dynamic
// shared-memory limit raised (cudaFuncSetAttribute is per device).  One instance per translation unit.
struct DeviceState {
  int sm_count = 0;
  bool attr[16] = {};
};
inline DeviceState* device_state(DeviceState (&states)[64], std::mutex& mu) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  DeviceState* s = &states[dev];
  if (s->sm_count == 0) {
    if (cudaDeviceGetAttribute(&s->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || s->sm_count <= 0) {
      (void)cudaGetLastError();
      s->sm_count = 148;
    }
  }
  return s;
}
// Raises the dynamic shared-memory limit of `kernel` once per device (slot: index of the kernel in the family).
template <class K>
inline cudaError_t ensure_smem_attr(DeviceState* ds, std::mutex& mu, int slot, K kernel, int bytes) {
  std::lock_guard<std::mutex> lock(mu);
  if (ds->attr[slot]) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) ds->attr[slot] = true;
  return e;
}

// Tensor [B*L, Y, X, H, D] bf16 as a rank-5 map (fastest first: d, h, x, y, b*l); box = 64 channels of
// one head x (bx, by, bl) tokens, 128-byte swizzle, out-of-bounds reads return zero.
// Encoding a map costs a driver call (~1 us); callers pass the same tensors step after step, so the last few maps
// are kept per host thread, keyed by everything the encoding depends on (base pointer, tensor shape, box).
inline bool make_map(CUtensorMap* map, const void* ptr, const Problem& p, int bx, int by, int bl) {
  struct Entry {
    const void* ptr = nullptr;
    long long bl_rows = 0;
    int D = 0, H = 0, X = 0, Y = 0, bx = 0, by = 0, bl = 0;
    CUtensorMap map;
  };
  constexpr int kEntries = 16;
  thread_local Entry cache[kEntries];
  thread_local int next = 0;
  const long long bl_rows = (long long)p.B * p.L;
  for (const Entry& c : cache)
    if (c.ptr == ptr && ptr && c.bl_rows == bl_rows && c.D == p.D && c.H == p.H && c.X == p.X && c.Y == p.Y && c.bx == bx &&
        c.by == by && c.bl == bl) {
      *map = c.map;
      return true;
    }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[5] = {(cuuint64_t)p.D, (cuuint64_t)p.H, (cuuint64_t)p.X, (cuuint64_t)p.Y,
                              (cuuint64_t)p.B * (cuuint64_t)p.L};
  const cuuint64_t e = 2;
  const cuuint64_t strides[4] = {(cuuint64_t)p.D * e, (cuuint64_t)p.H * p.D * e, (cuuint64_t)p.X * p.H * p.D * e,
                                 (cuuint64_t)p.Y * p.X * p.H * p.D * e};
  const cuuint32_t box[5] = {64, 1, (cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bl};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  if (fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(ptr), dims, strides, box, estr,
         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return false;
  Entry& slot = cache[next];
  next = (next + 1) % kEntries;
  slot.ptr = ptr; slot.bl_rows = bl_rows; slot.D = p.D; slot.H = p.H; slot.X = p.X; slot.Y = p.Y;
  slot.bx = bx; slot.by = by; slot.bl = bl; slot.map = *map;
  return true;
}


}  // namespace tc
}  // namespace strata
