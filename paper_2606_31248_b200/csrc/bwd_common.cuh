// bwd_common.cuh -- pieces of the tensor-core backward kernels (na3d_bwd_tc2.cu);
// include after tc_common.cuh.
#pragma once

namespace strata {
namespace {

using namespace tc;

struct BwdParams {
  int B, H, L, Y, X;
  int ntl, nty, ntx;
  long long N;
  float scale, scale_log2e;
  int pairing;   // strata_rope_pairing_t of the fused un-rotation
};


// packed fp32 pairs (one instruction for two columns)
struct F2 { float x, y; };
__device__ __forceinline__ F2 ffma2(F2 a, F2 b, F2 c) {
  F2 d;
  asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
      "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
  return d;
}
__device__ __forceinline__ F2 fadd2(F2 a, F2 b) {
  F2 d;
  asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
      "add.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}
__device__ __forceinline__ F2 fmul2(F2 a, F2 b) {
  F2 d;
  asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
      "mul.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}

// Streamed interval [lo, hi) of row index i on one axis: MODE 0 the window of query i (A3), MODE 1 the
// inverse neighbourhood of key i (B3).
template <int MODE>
__device__ __forceinline__ void row_interval(int i, int k, int n, int& lo, int& hi) {
  if (MODE == 0) {
    lo = window_start(i, k, n); hi = lo + k;
  } else {
    inverse_window(i, k, n, lo, hi); hi += 1;
  }
}


}  // namespace
}  // namespace strata
