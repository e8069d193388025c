// strata_na3d.cu -- the C ABI of libstrata_na3d.so (include/strata_na3d.h): validation, workspace
// carving, kernel-family dispatch, host-buffer variants.  No arithmetic lives here.
#include "../../include/strata_na3d.h"

#include "common.cuh"

namespace {

using strata::Problem;

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

thread_local int g_last_launches = 0;

// ---- optional per-kernel event timing -----------------------------------------------------------
constexpr int kMaxProf = 4096;
struct ProfState {
  bool on = false;
  int n = 0;
  cudaEvent_t beg[kMaxProf] = {}, end[kMaxProf] = {};
  const char* name[kMaxProf] = {};
};
thread_local ProfState g_prof;

bool make_problem(const strata_na3d_desc_t* d, Problem* p, strata_status_t* why) {
  *why = STRATA_ERR_INVALID_ARG;
  if (!d) return false;
  if (d->batch < 1 || d->heads < 1 || d->head_dim < 2 || (d->head_dim & 1)) return false;
  for (int a = 0; a < 3; ++a)
    if (d->grid[a] < 1 || d->window[a] < 1 || d->window[a] > d->grid[a]) return false;
  if (d->rope_axes < 0 || d->rope_pairing < 0 || d->rope_pairing > 1) return false;
  if (d->dtype != STRATA_DTYPE_F32 && d->dtype != STRATA_DTYPE_BF16) return false;
  if (d->impl < STRATA_IMPL_AUTO || d->impl > STRATA_IMPL_TCGEN05_TILE) return false;
  *why = STRATA_ERR_UNSUPPORTED;
  if (d->head_dim != 32 && d->head_dim != 64 && d->head_dim != 128) return false;
  if (d->rope_axes > 3) return false;
  p->B = d->batch; p->H = d->heads; p->D = d->head_dim;
  p->L = d->grid[0]; p->Y = d->grid[1]; p->X = d->grid[2];
  p->kL = d->window[0]; p->kY = d->window[1]; p->kX = d->window[2];
  p->A = d->rope_axes; p->pairing = d->rope_pairing; p->dtype = d->dtype;
  p->force_tile = d->impl == STRATA_IMPL_TCGEN05_TILE;
  p->scale = d->scale > 0.f ? d->scale : 1.0f / sqrtf((float)d->head_dim);
  p->N = (long long)p->L * p->Y * p->X;
  if ((double)p->rows() * p->D > 9.0e18) return false;
  *why = STRATA_OK;
  return true;
}

// Kernel path of a call.  The public strata_impl_t only distinguishes SIMT from TCGEN05.
enum Path { PATH_NONE = -1, PATH_SIMT = 1, PATH_TC_PREROT = 2, PATH_TC_PLANE = 3, PATH_COLUMN = 4 };

// AUTO -> the fused tcgen05 forward (na3d_fwd_plane.cu) when it covers the problem, else the tcgen05 tile kernels on
// pre-rotated operands, else SIMT.  PATH_NONE when `impl` asks for a family that does not cover the problem.
Path select_path(const strata_na3d_desc_t* d, const Problem& p, bool backward) {
  if (d->impl == STRATA_IMPL_SIMT) return PATH_SIMT;
  if (!backward && !p.force_tile && strata::plane_fwd_supported(p)) return PATH_TC_PLANE;
  if (!backward && !p.force_tile && strata::column_fwd_supported(p)) return PATH_COLUMN;
  const bool tc_ok = backward ? strata::tc_bwd_supported(p) : strata::tc_fwd_supported(p);
  if (tc_ok) return PATH_TC_PREROT;
  return d->impl == STRATA_IMPL_AUTO ? PATH_SIMT : PATH_NONE;
}

int select_impl(const strata_na3d_desc_t* d, const Problem& p, bool backward) {
  const Path path = select_path(d, p, backward);
  if (path == PATH_NONE) return -1;
  return path == PATH_SIMT ? STRATA_IMPL_SIMT : STRATA_IMPL_TCGEN05;   // (the column kernel counts as the tensor-core family)
}

struct Carve {
  char* base; size_t off;
  template <typename T> T* take(size_t bytes) {
    T* r = reinterpret_cast<T*>(base + off);
    off += align_up(bytes);
    return r;
  }
};

size_t ws_bytes(const Problem& p, Path path, bool backward) {
  const size_t e = (size_t)p.elems();
  const size_t stat = align_up((size_t)p.B * p.H * p.N * 4);
  if (backward && path == PATH_TC_PREROT)                               // qr, kr (bf16), stat (float2), fp32 rotary table
    return 2 * align_up(e * 2) + align_up(2 * stat) + align_up((size_t)p.B * p.N * (p.D / 2) * 8);
  if (backward) return 4 * align_up(e * 4) + stat;                       // qr, kr, dqr, dkr, delta
  if (path == PATH_TC_PLANE || path == PATH_COLUMN) return align_up(strata::plane_fwd_workspace_bytes());
  if (path == PATH_TC_PREROT) return 2 * align_up(e * 2);                // qr, kr (bf16)
  return 2 * align_up(e * 4);                                            // qr, kr (f32)
}

inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

strata_status_t cuda_status(cudaError_t e) {
  if (e == cudaSuccess) return STRATA_OK;
  (void)cudaGetLastError();
  return STRATA_ERR_CUDA;
}

size_t tensor_bytes(const Problem& p) { return (size_t)p.elems() * (p.dtype == 0 ? 4 : 2); }
size_t stat_bytes(const Problem& p) { return (size_t)p.B * p.H * p.N * 4; }
size_t coords_bytes(const Problem& p) { return (size_t)p.B * p.N * p.A * 4; }
size_t freqs_bytes(const Problem& p) { return (size_t)p.A * (p.D / 2) * 4; }

}  // namespace

namespace strata {
void prof_begin(const char* name, cudaStream_t stream) {
  ProfState& P = g_prof;
  if (!P.on || P.n >= kMaxProf) return;
  if (!P.beg[P.n]) { cudaEventCreate(&P.beg[P.n]); cudaEventCreate(&P.end[P.n]); }
  P.name[P.n] = name;
  cudaEventRecord(P.beg[P.n], stream);
}
void prof_end(cudaStream_t stream) {
  ProfState& P = g_prof;
  if (!P.on || P.n >= kMaxProf) return;
  cudaEventRecord(P.end[P.n], stream);
  ++P.n;
}
}  // namespace strata

extern "C" {

void strata_na3d_set_profiling(int enable) { g_prof.on = enable != 0; g_prof.n = 0; }

int strata_na3d_profile_read(float* ms, const char** names, int capacity) {
  ProfState& P = g_prof;
  for (int i = 0; i < P.n && i < capacity; ++i) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, P.beg[i], P.end[i]) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    if (ms) ms[i] = t;
    if (names) names[i] = P.name[i];
  }
  return P.n;
}

size_t strata_na3d_workspace_bytes(const strata_na3d_desc_t* desc, int backward) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return 0;
  const Path path = select_path(desc, p, backward != 0);
  if (path == PATH_NONE) return 0;
  return ws_bytes(p, path, backward != 0);
}

size_t strata_na3d_host_workspace_bytes(const strata_na3d_desc_t* desc, int backward) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return 0;
  const Path path = select_path(desc, p, backward != 0);
  if (path == PATH_NONE) return 0;
  const size_t t = align_up(tensor_bytes(p)), s = align_up(stat_bytes(p));
  const size_t geo = align_up(coords_bytes(p)) + align_up(freqs_bytes(p));
  const size_t staged = backward ? 8 * t + s + geo : 4 * t + s + geo;
  return staged + ws_bytes(p, path, backward != 0);
}

int strata_na3d_impl_selected(const strata_na3d_desc_t* desc, int backward) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return -1;
  return select_impl(desc, p, backward != 0);
}

strata_status_t strata_na3d_fwd(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                const void* v, const float* coords, const float* freqs, void* o,
                                float* lse, void* workspace, size_t workspace_bytes, void* stream) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (!q || !k || !v || !o || !lse) return STRATA_ERR_INVALID_ARG;
  if (p.A > 0 && (!coords || !freqs)) return STRATA_ERR_INVALID_ARG;
  if (misaligned(q) || misaligned(k) || misaligned(v) || misaligned(o) || misaligned(lse) ||
      misaligned(coords) || misaligned(freqs) || misaligned(workspace))
    return STRATA_ERR_INVALID_ARG;
  const Path path = select_path(desc, p, false);
  if (path == PATH_NONE) return STRATA_ERR_UNSUPPORTED;
  const size_t ws_need = ws_bytes(p, path, false);
  if (ws_need > 0 && (!workspace || workspace_bytes < ws_need)) return STRATA_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Carve ws{reinterpret_cast<char*>(workspace), 0};
  int launches = 0;
  cudaError_t e;
  if (path == PATH_TC_PLANE) {
    void* fix = ws.take<char>(strata::plane_fwd_workspace_bytes());
    e = strata::launch_fwd_plane(p, q, k, v, coords, freqs, o, lse, fix, st, &launches);
  } else if (path == PATH_COLUMN) {
    void* fix = ws.take<char>(strata::plane_fwd_workspace_bytes());
    e = strata::launch_fwd_column(p, q, k, v, coords, freqs, o, lse, fix, st, &launches);
  } else if (path == PATH_TC_PREROT) {
    void* qr = ws.take<char>((size_t)p.elems() * 2);
    void* kr = ws.take<char>((size_t)p.elems() * 2);
    e = strata::launch_rope_rotate(p, q, k, p.dtype, qr, kr, 1, coords, freqs, 1.f, st, &launches);
    if (e != cudaSuccess) return cuda_status(e);
    e = strata::launch_fwd_tc(p, qr, kr, v, o, lse, st, &launches);
  } else {
    float* qr = ws.take<float>((size_t)p.elems() * 4);
    float* kr = ws.take<float>((size_t)p.elems() * 4);
    e = strata::launch_rope_rotate(p, q, k, p.dtype, qr, kr, 0, coords, freqs, 1.f, st, &launches);
    if (e != cudaSuccess) return cuda_status(e);
    e = strata::launch_fwd_simt(p, qr, kr, v, o, lse, st, &launches);
  }
  if (e != cudaSuccess) return cuda_status(e);
  g_last_launches = launches;
  return STRATA_OK;
}

static strata_status_t bwd_impl(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                const void* v, const void* o, const void* d_o, const void* d_o_main, const float* lse,
                                const float* coords, const float* freqs, void* dq, void* dk,
                                void* dv, void* workspace, size_t workspace_bytes, void* stream) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (!q || !k || !v || !o || !d_o || !lse || !dq || !dk || !dv) return STRATA_ERR_INVALID_ARG;
  if (p.A > 0 && (!coords || !freqs)) return STRATA_ERR_INVALID_ARG;
  if (misaligned(q) || misaligned(k) || misaligned(v) || misaligned(o) || misaligned(d_o) ||
      misaligned(lse) || misaligned(coords) || misaligned(freqs) || misaligned(dq) ||
      misaligned(dk) || misaligned(dv) || misaligned(workspace))
    return STRATA_ERR_INVALID_ARG;
  const Path path = select_path(desc, p, true);
  if (path == PATH_NONE) return STRATA_ERR_UNSUPPORTED;
  if (!workspace || workspace_bytes < ws_bytes(p, path, true)) return STRATA_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Carve ws{reinterpret_cast<char*>(workspace), 0};
  const size_t eb = (size_t)p.elems() * 4;
  int launches = 0;
  cudaError_t e;
  if (path == PATH_TC_PREROT) {
    void* qr = ws.take<char>(eb / 2);
    void* kr = ws.take<char>(eb / 2);
    void* stat = ws.take<char>(2 * align_up(stat_bytes(p)));
    void* rtab = ws.take<char>((size_t)p.B * p.N * (p.D / 2) * 8);
    e = strata::launch_rope_rotate(p, q, k, p.dtype, qr, kr, 1, coords, freqs, 1.f, st, &launches);
    if (e != cudaSuccess) return cuda_status(e);
    if (p.A > 0) {
      e = strata::launch_rope_table_f32(p, rtab, coords, freqs, st, &launches);
      if (e != cudaSuccess) return cuda_status(e);
    }
    e = strata::launch_bwd_tc(p, qr, kr, v, o, d_o, d_o_main, lse, stat, p.A > 0 ? rtab : nullptr, dq, dk, dv, st, &launches);
    if (e != cudaSuccess) return cuda_status(e);
    g_last_launches = launches;
    return STRATA_OK;
  }
  float* qr = ws.take<float>(eb);
  float* kr = ws.take<float>(eb);
  float* dqr = ws.take<float>(eb);
  float* dkr = ws.take<float>(eb);
  float* delta = ws.take<float>(stat_bytes(p));
  e = strata::launch_rope_rotate(p, q, k, p.dtype, qr, kr, 0, coords, freqs, 1.f, st, &launches);
  if (e != cudaSuccess) return cuda_status(e);
  e = strata::launch_bwd_simt(p, qr, kr, v, o, d_o, d_o_main, lse, delta, dqr, dkr, dv, st, &launches);
  if (e != cudaSuccess) return cuda_status(e);
  // B4: dq = R(-phi) dqrot, dk = R(-phi) dkrot, rounded to the tensor dtype
  e = strata::launch_rope_rotate(p, dqr, dkr, 0, dq, dk, p.dtype, coords, freqs, -1.f, st, &launches);
  if (e != cudaSuccess) return cuda_status(e);
  g_last_launches = launches;
  return STRATA_OK;
}

strata_status_t strata_na3d_bwd(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                const void* v, const void* o, const void* d_o, const float* lse,
                                const float* coords, const float* freqs, void* dq, void* dk,
                                void* dv, void* workspace, size_t workspace_bytes, void* stream) {
  return bwd_impl(desc, q, k, v, o, d_o, d_o, lse, coords, freqs, dq, dk, dv, workspace, workspace_bytes, stream);
}

// ---- QK-RMSNorm + sigmoid head gate around the attention --------------------------------------------
size_t strata_na3d_normgate_workspace_bytes(const strata_na3d_desc_t* desc, int backward) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return 0;
  const Path path = select_path(desc, p, backward != 0);
  if (path == PATH_NONE) return 0;
  return (backward ? 3 : 2) * align_up(tensor_bytes(p)) + ws_bytes(p, path, backward != 0);
}

strata_status_t strata_na3d_normgate_fwd(const strata_na3d_desc_t* desc, const void* q, const void* k, const void* v,
                                         const float* coords, const float* freqs, const float* gate, float eps,
                                         void* o, float* lse, void* workspace, size_t workspace_bytes, void* stream) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (!q || !k || !o || !(eps >= 0.f)) return STRATA_ERR_INVALID_ARG;
  if (misaligned(q) || misaligned(k) || misaligned(gate) || misaligned(workspace)) return STRATA_ERR_INVALID_ARG;
  const size_t need = strata_na3d_normgate_workspace_bytes(desc, 0);
  if (need == 0) return STRATA_ERR_UNSUPPORTED;
  if (!workspace || workspace_bytes < need) return STRATA_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Carve ws{reinterpret_cast<char*>(workspace), 0};
  void* qn = ws.take<char>(tensor_bytes(p));
  void* kn = ws.take<char>(tensor_bytes(p));
  int launches = 0;
  cudaError_t e = strata::launch_rmsnorm_rows(p, q, qn, eps, st, &launches);
  if (e == cudaSuccess) e = strata::launch_rmsnorm_rows(p, k, kn, eps, st, &launches);
  if (e != cudaSuccess) return cuda_status(e);
  strata_status_t s = strata_na3d_fwd(desc, qn, kn, v, coords, freqs, o, lse, ws.base + ws.off, workspace_bytes - ws.off, stream);
  if (s != STRATA_OK) return s;
  launches += g_last_launches;
  if (gate) {
    e = strata::launch_gate_rows(p, o, o, gate, st, &launches);
    if (e != cudaSuccess) return cuda_status(e);
  }
  g_last_launches = launches;
  return STRATA_OK;
}

strata_status_t strata_na3d_normgate_bwd(const strata_na3d_desc_t* desc, const void* q, const void* k, const void* v,
                                         const void* o, const void* d_o, const float* lse, const float* coords,
                                         const float* freqs, const float* gate, float eps, void* dq, void* dk, void* dv,
                                         float* dgate, void* workspace, size_t workspace_bytes, void* stream) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (!q || !k || !o || !d_o || !dq || !dk || !(eps >= 0.f) || (gate && !dgate)) return STRATA_ERR_INVALID_ARG;
  if (misaligned(q) || misaligned(k) || misaligned(gate) || misaligned(dgate) || misaligned(workspace))
    return STRATA_ERR_INVALID_ARG;
  const size_t need = strata_na3d_normgate_workspace_bytes(desc, 1);
  if (need == 0) return STRATA_ERR_UNSUPPORTED;
  if (!workspace || workspace_bytes < need) return STRATA_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Carve ws{reinterpret_cast<char*>(workspace), 0};
  void* qn = ws.take<char>(tensor_bytes(p));
  void* kn = ws.take<char>(tensor_bytes(p));
  void* da = ws.take<char>(tensor_bytes(p));
  int launches = 0;
  cudaError_t e = strata::launch_rmsnorm_rows(p, q, qn, eps, st, &launches);
  if (e == cudaSuccess) e = strata::launch_rmsnorm_rows(p, k, kn, eps, st, &launches);
  // o = s a: the attention sees da = s dO, and B1's D_i = sum_c da_c a_c = sum_c dO_c o_c (raw gradient, gated output)
  if (e == cudaSuccess && gate) e = strata::launch_gate_rows(p, d_o, da, gate, st, &launches);
  if (e == cudaSuccess && gate) e = strata::launch_dgate_rows(p, d_o, o, gate, dgate, st, &launches);
  if (e != cudaSuccess) return cuda_status(e);
  strata_status_t s = bwd_impl(desc, qn, kn, v, o, d_o, gate ? da : d_o, lse, coords, freqs, dq, dk, dv, ws.base + ws.off,
                               workspace_bytes - ws.off, stream);
  if (s != STRATA_OK) return s;
  launches += g_last_launches;
  e = strata::launch_rmsnorm_bwd_rows(p, q, dq, eps, st, &launches);      // dq^, dk^ -> dq, dk (in place)
  if (e == cudaSuccess) e = strata::launch_rmsnorm_bwd_rows(p, k, dk, eps, st, &launches);
  if (e != cudaSuccess) return cuda_status(e);
  g_last_launches = launches;
  return STRATA_OK;
}

strata_status_t strata_na3d_fwd_host(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                     const void* v, const float* coords, const float* freqs,
                                     void* o, float* lse, void* workspace, size_t workspace_bytes,
                                     void* stream) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (!q || !k || !v || !o || !lse) return STRATA_ERR_INVALID_ARG;
  if (p.A > 0 && (!coords || !freqs)) return STRATA_ERR_INVALID_ARG;
  const size_t need = strata_na3d_host_workspace_bytes(desc, 0);
  if (need == 0) return STRATA_ERR_UNSUPPORTED;
  if (!workspace || workspace_bytes < need) return STRATA_ERR_WORKSPACE;
  if (misaligned(workspace)) return STRATA_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Carve ws{reinterpret_cast<char*>(workspace), 0};
  const size_t tb = tensor_bytes(p), sb = stat_bytes(p), cb = coords_bytes(p), fb = freqs_bytes(p);
  void* dq_ = ws.take<char>(tb); void* dk_ = ws.take<char>(tb); void* dv_ = ws.take<char>(tb);
  void* do_ = ws.take<char>(tb);
  float* dlse = ws.take<float>(sb);
  float* dco = ws.take<float>(cb); float* dfr = ws.take<float>(fb);
  cudaError_t e;
  if ((e = cudaMemcpyAsync(dq_, q, tb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  if ((e = cudaMemcpyAsync(dk_, k, tb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  if ((e = cudaMemcpyAsync(dv_, v, tb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  if (p.A > 0) {
    if ((e = cudaMemcpyAsync(dco, coords, cb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
    if ((e = cudaMemcpyAsync(dfr, freqs, fb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  }
  strata_status_t s = strata_na3d_fwd(desc, dq_, dk_, dv_, dco, dfr, do_, dlse, ws.base + ws.off,
                                      workspace_bytes - ws.off, stream);
  if (s != STRATA_OK) return s;
  if ((e = cudaMemcpyAsync(o, do_, tb, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_status(e);
  if ((e = cudaMemcpyAsync(lse, dlse, sb, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_status(e);
  return STRATA_OK;
}

strata_status_t strata_na3d_bwd_host(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                     const void* v, const void* o, const void* d_o,
                                     const float* lse, const float* coords, const float* freqs,
                                     void* dq, void* dk, void* dv, void* workspace,
                                     size_t workspace_bytes, void* stream) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (!q || !k || !v || !o || !d_o || !lse || !dq || !dk || !dv) return STRATA_ERR_INVALID_ARG;
  if (p.A > 0 && (!coords || !freqs)) return STRATA_ERR_INVALID_ARG;
  const size_t need = strata_na3d_host_workspace_bytes(desc, 1);
  if (need == 0) return STRATA_ERR_UNSUPPORTED;
  if (!workspace || workspace_bytes < need) return STRATA_ERR_WORKSPACE;
  if (misaligned(workspace)) return STRATA_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Carve ws{reinterpret_cast<char*>(workspace), 0};
  const size_t tb = tensor_bytes(p), sb = stat_bytes(p), cb = coords_bytes(p), fb = freqs_bytes(p);
  const void* hsrc[5] = {q, k, v, o, d_o};
  void* dsrc[5];
  for (int i = 0; i < 5; ++i) dsrc[i] = ws.take<char>(tb);
  void* dout[3];
  for (int i = 0; i < 3; ++i) dout[i] = ws.take<char>(tb);
  float* dlse = ws.take<float>(sb);
  float* dco = ws.take<float>(cb); float* dfr = ws.take<float>(fb);
  cudaError_t e;
  for (int i = 0; i < 5; ++i)
    if ((e = cudaMemcpyAsync(dsrc[i], hsrc[i], tb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  if ((e = cudaMemcpyAsync(dlse, lse, sb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  if (p.A > 0) {
    if ((e = cudaMemcpyAsync(dco, coords, cb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
    if ((e = cudaMemcpyAsync(dfr, freqs, fb, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_status(e);
  }
  strata_status_t s = strata_na3d_bwd(desc, dsrc[0], dsrc[1], dsrc[2], dsrc[3], dsrc[4], dlse, dco, dfr,
                                      dout[0], dout[1], dout[2], ws.base + ws.off,
                                      workspace_bytes - ws.off, stream);
  if (s != STRATA_OK) return s;
  void* hdst[3] = {dq, dk, dv};
  for (int i = 0; i < 3; ++i)
    if ((e = cudaMemcpyAsync(hdst[i], dout[i], tb, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_status(e);
  return STRATA_OK;
}

int strata_na3d_last_launch_count(void) { return g_last_launches; }

int strata_na3d_window_start(int i, int k, int n) {
  if (k < 1 || k > n || i < 0 || i >= n) return -1;
  return strata::window_start(i, k, n);
}

int strata_na3d_inverse_window(int j, int k, int n, int* lo, int* hi) {
  if (k < 1 || k > n || j < 0 || j >= n || !lo || !hi) return -1;
  strata::inverse_window(j, k, n, *lo, *hi);
  return 0;
}

const char* strata_status_string(strata_status_t s) {
  switch (s) {
    case STRATA_OK: return "ok";
    case STRATA_ERR_INVALID_ARG: return "invalid argument";
    case STRATA_ERR_UNSUPPORTED: return "unsupported configuration";
    case STRATA_ERR_WORKSPACE: return "workspace missing or too small";
    case STRATA_ERR_CUDA: return "CUDA error";
  }
  return "unknown status";
}

int strata_version(void) { return 100; }

}  // extern "C"
