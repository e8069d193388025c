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
  if (backward && path == PATH_TC_PREROT)               // qr, kr (bf16), stat (float2) + bias rows (16 B), fp32 rotary table
    return 2 * align_up(e * 2) + align_up(6 * stat) + align_up((size_t)p.B * p.N * (p.D / 2) * 8);
  if (backward) return 4 * align_up(e * 4) + stat;                       // qr, kr, dqr, dkr, delta
  if (path == PATH_TC_PLANE || path == PATH_COLUMN) return align_up(strata::plane_fwd_workspace_bytes());
  if (path == PATH_TC_PREROT) return align_up(strata::plane_fwd_workspace_bytes()) + 2 * align_up(e * 2);   // fix list, qr, kr (bf16)
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


// ---- host entry points: two staging slots of ONE sample each; copies in, kernels and copies out of consecutive
// samples overlap on three streams (the caller's stream runs the kernels; two internal streams carry the copies and
// are joined back into it before the call returns, so the call stays asynchronous and ordered on `stream`).
struct HostLayout {
  size_t tensor, stat, coords, freqs, slot, inner, total;          // bytes (aligned) of the per-sample pieces
};
HostLayout host_layout(const Problem& p1, Path path, bool backward) {
  HostLayout h;
  h.tensor = align_up(tensor_bytes(p1)); h.stat = align_up(stat_bytes(p1));
  h.coords = align_up(coords_bytes(p1)); h.freqs = align_up(freqs_bytes(p1));
  h.slot = (backward ? 8 : 4) * h.tensor + h.stat + h.coords;
  h.inner = align_up(ws_bytes(p1, path, backward));
  h.total = 2 * h.slot + h.freqs + h.inner;
  return h;
}
struct HostPipe {
  int dev = -1;
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t entry = nullptr, in_ready[2] = {}, compute_done[2] = {}, out_done[2] = {};
};
HostPipe* host_pipe() {
  thread_local HostPipe pipes[8];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
  HostPipe* hp = nullptr;
  for (HostPipe& c : pipes) if (c.dev == dev) { hp = &c; break; }
  if (!hp) {
    for (HostPipe& c : pipes) if (c.dev < 0) { hp = &c; break; }
    if (!hp) return nullptr;
    bool ok = cudaStreamCreateWithFlags(&hp->s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&hp->s_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&hp->entry, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i)
      ok = cudaEventCreateWithFlags(&hp->in_ready[i], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&hp->compute_done[i], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&hp->out_done[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { (void)cudaGetLastError(); return nullptr; }
    hp->dev = dev;
  }
  return hp;
}
#define STRATA_CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_status(e_); } while (0)

// One pass of the per-sample pipeline.  n_in / n_out: tensors of the sample copied in / out (q, k, v[, o, d_o] /
// o | dq, dk, dv); lse goes in (backward) or out (forward).
strata_status_t host_pipeline(const strata_na3d_desc_t* desc, bool backward, const void* const* h_in, int n_in,
                              void* const* h_out, int n_out, const float* h_lse_in, float* h_lse_out,
                              const float* h_coords, const float* h_freqs, void* workspace, size_t workspace_bytes,
                              cudaStream_t st);

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
  strata_na3d_desc_t d1 = *desc;
  d1.batch = 1;                                                     // the host entry points work one sample at a time
  Problem p1;
  if (!make_problem(&d1, &p1, &why)) return 0;
  const Path path = select_path(&d1, p1, backward != 0);
  if (path == PATH_NONE) return 0;
  return host_layout(p1, path, backward != 0).total;
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
    void* fix = ws.take<char>(strata::plane_fwd_workspace_bytes());
    void* qr = ws.take<char>((size_t)p.elems() * 2);
    void* kr = ws.take<char>((size_t)p.elems() * 2);
    const void *qin = q, *kin = k;
    if (p.A > 0) {                                          // (no rotary axes: the kernel reads Q, K as they are)
      e = strata::launch_rope_rotate(p, q, k, p.dtype, qr, kr, 1, coords, freqs, 1.f, st, &launches);
      if (e != cudaSuccess) return cuda_status(e);
      qin = qr; kin = kr;
    }
    e = strata::launch_fwd_tc(p, qin, kin, v, o, lse, fix, st, &launches);
    if (e != cudaSuccess) return cuda_status(e);
    e = strata::launch_fix_rows(p, q, k, v, coords, freqs, o, lse, fix, st, &launches);   // rows the kernel listed (usually none)
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
    void* stat = ws.take<char>(6 * align_up(stat_bytes(p)));
    void* rtab = ws.take<char>((size_t)p.B * p.N * (p.D / 2) * 8);
    if (p.A > 0) {                                          // the table serves A2 here and B4 in the epilogues
      e = strata::launch_rope_table_f32(p, rtab, coords, freqs, st, &launches);
      if (e == cudaSuccess) e = strata::launch_rope_rotate_table(p, q, k, qr, kr, rtab, 1.f, st, &launches);
    } else {
      e = strata::launch_rope_rotate(p, q, k, p.dtype, qr, kr, 1, coords, freqs, 1.f, st, &launches);
    }
    if (e != cudaSuccess) return cuda_status(e);
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
  // every argument is checked before the first kernel is enqueued (the inner strata_na3d_fwd would only see v, lse,
  // coords, freqs after the two normalisation kernels are already on the stream)
  if (!q || !k || !v || !o || !lse || !(eps >= 0.f)) return STRATA_ERR_INVALID_ARG;
  if (p.A > 0 && (!coords || !freqs)) return STRATA_ERR_INVALID_ARG;
  if (misaligned(q) || misaligned(k) || misaligned(v) || misaligned(o) || misaligned(lse) || misaligned(coords) ||
      misaligned(freqs) || misaligned(gate) || misaligned(workspace))
    return STRATA_ERR_INVALID_ARG;
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
  if (!q || !k || !v || !o || !d_o || !lse || !dq || !dk || !dv || !(eps >= 0.f) || (gate && !dgate))
    return STRATA_ERR_INVALID_ARG;                                  // (all of it before the first enqueue, as in the forward)
  if (p.A > 0 && (!coords || !freqs)) return STRATA_ERR_INVALID_ARG;
  if (misaligned(q) || misaligned(k) || misaligned(v) || misaligned(o) || misaligned(d_o) || misaligned(lse) ||
      misaligned(coords) || misaligned(freqs) || misaligned(dq) || misaligned(dk) || misaligned(dv) || misaligned(gate) ||
      misaligned(dgate) || misaligned(workspace))
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
  if (!q || !k || !v || !o || !lse) return STRATA_ERR_INVALID_ARG;
  const void* in[3] = {q, k, v};
  void* out[1] = {o};
  return host_pipeline(desc, false, in, 3, out, 1, nullptr, lse, coords, freqs, workspace, workspace_bytes,
                       reinterpret_cast<cudaStream_t>(stream));
}

strata_status_t strata_na3d_bwd_host(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                     const void* v, const void* o, const void* d_o,
                                     const float* lse, const float* coords, const float* freqs,
                                     void* dq, void* dk, void* dv, void* workspace,
                                     size_t workspace_bytes, void* stream) {
  if (!q || !k || !v || !o || !d_o || !lse || !dq || !dk || !dv) return STRATA_ERR_INVALID_ARG;
  const void* in[5] = {q, k, v, o, d_o};
  void* out[3] = {dq, dk, dv};
  return host_pipeline(desc, true, in, 5, out, 3, lse, nullptr, coords, freqs, workspace, workspace_bytes,
                       reinterpret_cast<cudaStream_t>(stream));
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
    case STRATA_ERR_STATIC_SCRATCH: return "problem needs more scratch than the library's static array holds (STRATA_STATIC_SCRATCH_BYTES)";
  }
  return "unknown status";
}

int strata_version(void) { return 200; }

}  // extern "C"

namespace {

strata_status_t host_pipeline(const strata_na3d_desc_t* desc, bool backward, const void* const* h_in, int n_in,
                              void* const* h_out, int n_out, const float* h_lse_in, float* h_lse_out,
                              const float* h_coords, const float* h_freqs, void* workspace, size_t workspace_bytes,
                              cudaStream_t st) {
  Problem p; strata_status_t why;
  if (!make_problem(desc, &p, &why)) return why;
  if (p.A > 0 && (!h_coords || !h_freqs)) return STRATA_ERR_INVALID_ARG;
  strata_na3d_desc_t d1 = *desc;
  d1.batch = 1;
  Problem p1;
  if (!make_problem(&d1, &p1, &why)) return why;
  const Path path = select_path(&d1, p1, backward);
  if (path == PATH_NONE) return STRATA_ERR_UNSUPPORTED;
  const HostLayout L = host_layout(p1, path, backward);
  if (!workspace || workspace_bytes < L.total) return STRATA_ERR_WORKSPACE;
  if (misaligned(workspace)) return STRATA_ERR_INVALID_ARG;
  HostPipe* hp = host_pipe();
  if (!hp) return STRATA_ERR_CUDA;
  char* base = reinterpret_cast<char*>(workspace);
  float* d_freqs = reinterpret_cast<float*>(base + 2 * L.slot);
  char* inner = base + 2 * L.slot + L.freqs;
  const size_t tb = tensor_bytes(p1), sb = stat_bytes(p1), cb = coords_bytes(p1), fb = freqs_bytes(p1);
  // slot layout: inputs | outputs | lse | coords
  auto slot_tensor = [&](int slot, int i) { return base + slot * L.slot + (size_t)i * L.tensor; };
  auto slot_lse = [&](int slot) { return reinterpret_cast<float*>(base + slot * L.slot + (size_t)(n_in + n_out) * L.tensor); };
  auto slot_coords = [&](int slot) { return reinterpret_cast<float*>(base + slot * L.slot + (size_t)(n_in + n_out) * L.tensor + L.stat); };

  STRATA_CK(cudaEventRecord(hp->entry, st));                       // the copies start after what is already on `stream`
  STRATA_CK(cudaStreamWaitEvent(hp->s_in, hp->entry, 0));
  STRATA_CK(cudaStreamWaitEvent(hp->s_out, hp->entry, 0));
  if (p.A > 0) STRATA_CK(cudaMemcpyAsync(d_freqs, h_freqs, fb, cudaMemcpyHostToDevice, hp->s_in));
  int launches = 0;
  // From here on work may sit on the two internal streams: whatever happens, they are joined back into `stream`
  // before the call returns, so that an error half-way leaves no copy running behind the caller's back.
  auto enqueue = [&]() -> strata_status_t {
    for (int b = 0; b < p.B; ++b) {
      const int s = b & 1;
      // ---- copies in (slot s was last read by the kernels of sample b - 2)
      if (b >= 2) STRATA_CK(cudaStreamWaitEvent(hp->s_in, hp->compute_done[s], 0));
      for (int i = 0; i < n_in; ++i)
        STRATA_CK(cudaMemcpyAsync(slot_tensor(s, i), static_cast<const char*>(h_in[i]) + (size_t)b * tb, tb,
                                  cudaMemcpyHostToDevice, hp->s_in));
      if (h_lse_in) STRATA_CK(cudaMemcpyAsync(slot_lse(s), h_lse_in + (size_t)b * (sb / 4), sb, cudaMemcpyHostToDevice, hp->s_in));
      if (p.A > 0) STRATA_CK(cudaMemcpyAsync(slot_coords(s), h_coords + (size_t)b * (cb / 4), cb, cudaMemcpyHostToDevice, hp->s_in));
      STRATA_CK(cudaEventRecord(hp->in_ready[s], hp->s_in));
      // ---- kernels of the sample on the caller's stream (its outputs of sample b - 2 must have left the slot)
      STRATA_CK(cudaStreamWaitEvent(st, hp->in_ready[s], 0));
      if (b >= 2) STRATA_CK(cudaStreamWaitEvent(st, hp->out_done[s], 0));
      strata_status_t rc;
      if (!backward)
        rc = strata_na3d_fwd(&d1, slot_tensor(s, 0), slot_tensor(s, 1), slot_tensor(s, 2), slot_coords(s), d_freqs,
                             slot_tensor(s, n_in), slot_lse(s), inner, L.inner, st);
      else
        rc = strata_na3d_bwd(&d1, slot_tensor(s, 0), slot_tensor(s, 1), slot_tensor(s, 2), slot_tensor(s, 3), slot_tensor(s, 4),
                             slot_lse(s), slot_coords(s), d_freqs, slot_tensor(s, n_in), slot_tensor(s, n_in + 1),
                             slot_tensor(s, n_in + 2), inner, L.inner, st);
      if (rc != STRATA_OK) return rc;
      launches += g_last_launches;
      STRATA_CK(cudaEventRecord(hp->compute_done[s], st));
      // ---- copies out
      STRATA_CK(cudaStreamWaitEvent(hp->s_out, hp->compute_done[s], 0));
      for (int i = 0; i < n_out; ++i)
        STRATA_CK(cudaMemcpyAsync(static_cast<char*>(h_out[i]) + (size_t)b * tb, slot_tensor(s, n_in + i), tb,
                                  cudaMemcpyDeviceToHost, hp->s_out));
      if (h_lse_out) STRATA_CK(cudaMemcpyAsync(h_lse_out + (size_t)b * (sb / 4), slot_lse(s), sb, cudaMemcpyDeviceToHost, hp->s_out));
      STRATA_CK(cudaEventRecord(hp->out_done[s], hp->s_out));
    }
    return STRATA_OK;
  };
  auto join = [&]() -> strata_status_t {                             // `stream` waits for everything on s_out and s_in
    STRATA_CK(cudaEventRecord(hp->entry, hp->s_out));
    STRATA_CK(cudaStreamWaitEvent(st, hp->entry, 0));
    STRATA_CK(cudaEventRecord(hp->entry, hp->s_in));
    STRATA_CK(cudaStreamWaitEvent(st, hp->entry, 0));
    return STRATA_OK;
  };
  const strata_status_t rc_enqueue = enqueue();
  const strata_status_t rc_join = join();
  if (rc_enqueue != STRATA_OK) return rc_enqueue;
  if (rc_join != STRATA_OK) return rc_join;
  g_last_launches = launches;
  return STRATA_OK;
}

}  // namespace
