// plk_api.cu -- the C ABI of include/plk.h: instance, arena sub-allocation, validation, level scheduling and kernel
// launches.  No device memory is allocated here (the arena is the caller's); no arithmetic of the method runs on
// the host.  Citations as in plk.h (P: PAPER.md line, S8x: SURVEY.md section 8(x)).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/plk.h"
#include "plk_common.cuh"
#include "plk_gen.cuh"
#include "plk_misc.cuh"
#include "plk_nuc.cuh"
#include "plk_nuc_tma.cuh"
#include "plk_nuc_lean.cuh"
#include "plk_cross.cuh"
#include "plk_cross_tc.cuh"
#include "plk_cache.cuh"
#include "plk_schedule.h"
#ifdef PLK_WITH_TENSOR
#include "plk_tc.cuh"
#include "plk_tc5.cuh"
#include "plk_tc5_pre.cuh"
#include "plk_tc5_pre2.cuh"
#endif

using namespace plk;

namespace {

constexpr size_t ALIGN = 1024;
constexpr size_t RING_BYTES = 8u << 20;  // parameter staging ring (pinned host + device mirror)
constexpr size_t PLAN_BYTES = 4u << 20;  // descriptor blocks of the cached evaluation graphs (plk_evaluate*)
constexpr int PLAN_MAX = 8;              // cached evaluation graphs per instance
inline size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
constexpr int NUC_MAX_WALK_WARPS = 16384;  // walk-shape grid cap (256 SMs x 64 warps); sizes the partial-sum rows
inline int nuc_lanes_per_pattern(int C) { return C % 4 == 0 ? 4 : (C % 2 == 0 ? 2 : 1); }  // NucMap<C>::LP

struct Layout {
  int S, SP, C, P;
  size_t w;                 // bytes per real
  size_t W;                 // one partials slot
  size_t mx_bytes;          // per-slot maxima (SP = 64, deferred rescaling), else 0
  int post_slots, compact_slots, pre_slots;
  size_t compact_bytes, matrix_bytes, eigen_bytes, scale_bytes;
  int n_tiles, max_grad;
  size_t off_post, off_compact, off_pre, off_pre_mx, off_matrix, off_eigen, off_scale, off_weights, off_pi,
      off_rates, off_catw, off_site, off_block_partial, off_grad_partial, off_grad_out, off_logl, off_site_deriv,
      off_stage, off_ring, off_plan, off_eval_t, off_eval_out, off_qp, off_otf_ready, off_otf_sync, off_matrix_t, off_matrix_d, off_matrix_dt, off_cat_scratch, off_cross_partial, off_cross_out, total;
  size_t stage_bytes;
};

bool compute_layout(const plk_config& c, Layout& L) {
  if (c.tip_count < 2 || c.pattern_count < 1 || c.category_count < 1 || c.category_count > 16) return false;
  if (c.state_count < 2 || c.state_count > 64) return false;
  if (c.state_count == 4 && c.category_count > 8) return false;
  if (c.partials_buffer_count < c.tip_count || c.compact_buffer_count < 0 ||
      c.compact_buffer_count > c.tip_count || c.partials_slot_count < 0 || c.preorder_buffer_count < 0 ||
      c.preorder_slot_count < 0 || c.matrix_buffer_count < 1 || c.eigen_buffer_count < 1 ||
      c.scale_buffer_count < 0)
    return false;
  if (c.precision != PLK_FP64 && c.precision != PLK_FP32) return false;
  L.S = c.state_count;
  L.SP = c.state_count == 4 ? 4 : (c.state_count <= 32 ? 32 : 64);  // 5..32 states (amino acids: 20) pad to 32
  L.C = c.category_count;
  L.P = c.pattern_count;
  L.w = c.precision == PLK_FP64 ? 8 : 4;
  L.W = round_up((size_t)L.C * L.P * L.SP * L.w, ALIGN);
  L.mx_bytes = L.SP == 4 ? 0 : round_up((size_t)L.C * L.P * L.w, ALIGN);
  L.post_slots = c.partials_slot_count > 0 ? c.partials_slot_count : c.partials_buffer_count - c.compact_buffer_count;
  L.compact_slots = c.compact_buffer_count;
  L.pre_slots = c.preorder_slot_count > 0 ? c.preorder_slot_count : c.preorder_buffer_count;
  L.compact_bytes = round_up((size_t)L.P, ALIGN);
  L.matrix_bytes = round_up((size_t)L.C * L.SP * L.SP * L.w, ALIGN);
  // eigen buffer: U, Uinv (S*S fp64), lambda (S fp64), Q64 (S*S fp64), QT (SP*SP reals)
  L.eigen_bytes = round_up((size_t)(3 * L.S * L.S + L.S) * 8, ALIGN) + round_up((size_t)L.SP * L.SP * L.w, ALIGN);
  L.scale_bytes = L.SP == 4 ? round_up((size_t)L.P * 2, ALIGN) : L.mx_bytes;
  if (L.SP == 4) {
    // rows of gradient partial sums: one per block (level shape, k_deriv4) or one per warp (walk shape, capped)
    const int ppw = 32 / nuc_lanes_per_pattern(L.C);
    const int n_chunks = (L.P + ppw - 1) / ppw;
    const int level_blocks = (n_chunks + NUC_WARPS - 1) / NUC_WARPS;
    const int walk_warps = n_chunks < NUC_MAX_WALK_WARPS ? n_chunks : NUC_MAX_WALK_WARPS;
    L.n_tiles = level_blocks > walk_warps ? level_blocks : walk_warps;
    if (L.n_tiles < n_chunks + NT_CW) L.n_tiles = n_chunks + NT_CW;  // TMA level shape: one per (pattern tile, warp)
  } else {
    L.n_tiles = (L.P + GEN_TP - 1) / GEN_TP;
  }
  L.max_grad = c.partials_buffer_count;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += round_up(bytes, ALIGN); return at; };
  L.off_post = take((size_t)L.post_slots * L.W);
  L.off_compact = take((size_t)L.compact_slots * L.compact_bytes);
  L.off_pre = take((size_t)L.pre_slots * L.W);
  L.off_pre_mx = take((size_t)L.pre_slots * L.mx_bytes);
  L.off_matrix = take((size_t)c.matrix_buffer_count * L.matrix_bytes);
  L.off_eigen = take((size_t)c.eigen_buffer_count * L.eigen_bytes);
  L.off_scale = take((size_t)c.scale_buffer_count * L.scale_bytes);
  L.off_weights = take((size_t)L.P * 8);
  L.off_pi = take((size_t)L.SP * 8);
  L.off_rates = take((size_t)L.C * 8);
  L.off_catw = take((size_t)L.C * 8);
  L.off_site = take((size_t)L.P * 8);
  // one partial per block of k_root (128 threads, G threads per pattern: G = 1 for SP = 4, SP / 4 otherwise)
  L.off_block_partial = take(((size_t)L.P * (L.SP == 4 ? 1 : L.SP / 4) + 127) / 128 * 8 + 8);
  L.off_grad_partial = take((size_t)L.max_grad * L.n_tiles * 8);
  L.off_grad_out = take((size_t)L.max_grad * 8);
  L.off_logl = take(64);
  L.off_site_deriv = take((c.flags & PLK_FLAG_SITE_DERIVATIVES) ? (size_t)L.max_grad * L.P * 8 : 0);
  L.stage_bytes = round_up((size_t)L.C * L.P * L.S * 8, ALIGN);
  L.off_stage = take(L.stage_bytes);
  L.off_ring = take(RING_BYTES);
  L.off_plan = take(PLAN_BYTES);
  L.off_eval_t = take((size_t)c.matrix_buffer_count * 8);        // plk_evaluate: branch lengths, [logL, gradient]
  L.off_eval_out = take((size_t)(1 + c.partials_buffer_count) * 8);
  // caching variants of P:101 (plk_cache.cuh): Q p_k next to every full partials slot; ready flags of the one-launch
  // on-the-fly post-order pass (one per operation and pattern) and its ticket counters
  L.off_qp = take((c.flags & PLK_FLAG_CACHE_RATE_PRODUCTS) ? (size_t)L.post_slots * L.W : 0);
  L.off_otf_ready = take((c.flags & PLK_FLAG_ON_THE_FLY_MATRICES) ? (size_t)c.partials_buffer_count * L.P * 4 : 0);
  L.off_otf_sync = take(64);
  // fp32 tensor-core instances (tcgen05 pre-order kernels, plk_tc5_pre*.cuh): per matrix buffer M^T, D = M Q and D^T,
  // and the per-category num / den scratch of the class-specialised kernels ([slot][num, den][C][P] floats)
  const bool tc5 = L.SP == 64 && c.precision == PLK_FP32 && (c.flags & PLK_FLAG_TENSOR_CORES) && !(c.flags & PLK_FLAG_NO_TCGEN05);
  L.off_matrix_t = take(tc5 ? (size_t)c.matrix_buffer_count * L.matrix_bytes : 0);
  // derivative matrices D = M Q: 4-state specialised gradient kernels (plk_nuc_lean.cuh, compact-tip children) and tc5
  L.off_matrix_d = take((L.SP == 4 || tc5) ? (size_t)c.matrix_buffer_count * L.matrix_bytes : 0);
  L.off_matrix_dt = take(tc5 ? (size_t)c.matrix_buffer_count * L.matrix_bytes : 0);
  L.off_cat_scratch = take((tc5 && c.preorder_buffer_count > 0) ? (size_t)L.max_grad * 2 * L.C * L.P * 4 : 0);
  // rate-matrix gradient (plk_cross.cuh): per-block partial sums and the S x S result
  L.off_cross_partial = take(c.preorder_buffer_count > 0
                                 ? (L.SP == 4 ? (size_t)16 * CROSS4_SPLITS * ((L.P + CROSS4_THREADS - 1) / CROSS4_THREADS)
                                              : (size_t)std::max((L.P + CROSS64_TP - 1) / CROSS64_TP, L.SP == 64 ? CROSS_TC_MAX_GRID : 0) * L.SP * L.SP) * 8
                                 : 0);
  L.off_cross_out = take((size_t)L.SP * L.SP * 8);
  L.total = o;
  return true;
}

}  // namespace

struct plk_instance {
  plk_config cfg;
  Layout L;
  cudaStream_t stream;
  char* arena;
  bool f32;
  bool deferred;  // SP = 64: rescaling deferred to the consumer
  // buffer tables (host bookkeeping only)
  std::vector<int> post_slot, post_kind, post_pending_scale;
  std::vector<char> post_written;
  std::vector<char> qp_valid;   // PLK_FLAG_CACHE_RATE_PRODUCTS: Q p_k of this post-order buffer is current
  unsigned int otf_epoch = 0;   // value of the ready flags of the current on-the-fly launch
  std::vector<int> pre_slot;
  std::vector<char> pre_written, pre_has_mx;
  std::vector<char> matrix_written, scale_written, eigen_written, q_written;
  std::vector<double> h_q4;  // 4-state instances: host copy of every Q [eigen][16] (working precision, widened)
  int next_post_slot = 0, next_compact_slot = 0, next_pre_slot = 0;
  bool have_weights = false, have_pi = false, have_rates = false, have_catw = false;
  int root_pre_filled = -1;
  // parameter ring
  char* h_ring = nullptr;
  size_t ring_pos = 0;
  int64_t launches = 0;
  int sm_count = 148;
  int nt_bps[2][2] = {{0, 0}, {0, 0}};  // resident CTAs per SM of the TMA kernels [post|pre][level|walk]
  int lean_bps[3] = {0, 0, 0};          // the same for k_pre4_lean<T, CLS> (T is fixed per instance)
  int grad_parts = 0;  // partial sums per gradient slot written by the LAST gradient launch (row stride L.n_tiles)
  // cached evaluation graphs (plk_evaluate*): one per distinct call signature
  struct EvalPlan {
    uint64_t key = 0;
    int uses = 0;              // the first use runs eagerly (it also binds slots and sets kernel attributes)
    bool failed = false;       // capture was refused once (e.g. legacy default stream): stay eager
    cudaGraphExec_t exec = nullptr;
    int64_t launches = 0;      // kernels in the graph
  };
  std::vector<EvalPlan> plans;
  std::vector<char> plan_host;  // host image of the plan region (descriptors of the captured launches)
  size_t plan_pos = 0;          // bump pointer inside the plan region
  bool planning = false;        // ring_alloc serves from the plan region, copy_ring is deferred
  uint64_t model_epoch = 0;     // bumped by every setter whose value is baked into launch parameters
  uint64_t binding_epoch = 0;   // bumped when a buffer index is bound to a slot or changes kind

  template <typename X> X* at(size_t off) const { return reinterpret_cast<X*>(arena + off); }
  void* post_ptr(int idx) const {
    if (post_kind[idx] == KIND_STATES) return arena + L.off_compact + (size_t)post_slot[idx] * L.compact_bytes;
    return arena + L.off_post + (size_t)post_slot[idx] * L.W;
  }
  void* qp_ptr(int idx) const { return arena + L.off_qp + (size_t)post_slot[idx] * L.W; }
  void* pre_ptr(int idx) const { return arena + L.off_pre + (size_t)pre_slot[idx] * L.W; }
  void* pre_mx_ptr(int idx) const { return arena + L.off_pre_mx + (size_t)pre_slot[idx] * L.mx_bytes; }
  void* matrix_ptr(int idx) const { return arena + L.off_matrix + (size_t)idx * L.matrix_bytes; }
  void* scale_ptr(int idx) const { return arena + L.off_scale + (size_t)idx * L.scale_bytes; }
  char* eigen_base(int idx) const { return arena + L.off_eigen + (size_t)idx * L.eigen_bytes; }
  double* eig_U(int idx) const { return reinterpret_cast<double*>(eigen_base(idx)); }
  double* eig_Uinv(int idx) const { return eig_U(idx) + L.S * L.S; }
  double* eig_Q64(int idx) const { return eig_U(idx) + 2 * L.S * L.S; }
  double* eig_lam(int idx) const { return eig_U(idx) + 3 * L.S * L.S; }
  void* eig_QT(int idx) const { return eigen_base(idx) + round_up((size_t)(3 * L.S * L.S + L.S) * 8, ALIGN); }
};

namespace {

#define CU(call)                                  \
  do {                                            \
    cudaError_t e_ = (call);                      \
    if (e_ != cudaSuccess) return PLK_ERR_CUDA;   \
  } while (0)
#define CHECK_LAUNCH(inst)                        \
  do {                                            \
    ++(inst)->launches;                           \
    if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA; \
  } while (0)

// Reserve `bytes` in the parameter ring; returns the host pointer and the matching device pointer.  The host
// region is copied to the device with copy_ring() after it was filled.  Wrapping synchronises the stream so that
// earlier asynchronous copies have left the pinned buffer.
int ring_alloc(plk_instance* in, size_t bytes, char** h, char** d) {
  bytes = round_up(bytes, 256);
  if (in->planning) {  // graph capture: descriptors live in the plan region for as long as the graph does
    if (in->plan_pos + bytes > PLAN_BYTES) return PLK_ERR_OUT_OF_MEMORY;
    *h = in->plan_host.data() + in->plan_pos;
    *d = in->arena + in->L.off_plan + in->plan_pos;
    in->plan_pos += bytes;
    return PLK_SUCCESS;
  }
  if (bytes > RING_BYTES) return PLK_ERR_OUT_OF_MEMORY;
  if (in->ring_pos + bytes > RING_BYTES) {
    CU(cudaStreamSynchronize(in->stream));
    in->ring_pos = 0;
  }
  *h = in->h_ring + in->ring_pos;
  *d = in->arena + in->L.off_ring + in->ring_pos;
  in->ring_pos += bytes;
  return PLK_SUCCESS;
}
int copy_ring(plk_instance* in, const char* h, char* d, size_t bytes) {
  if (in->planning) return PLK_SUCCESS;  // uploaded in one piece after the capture (plk_evaluate_device)
  CU(cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, in->stream));
  return PLK_SUCCESS;
}

int bind_post_full(plk_instance* in, int idx, int kind) {
  if (in->post_slot[idx] >= 0 && in->post_kind[idx] != KIND_STATES) {
    if (in->post_kind[idx] != kind) ++in->binding_epoch;
    in->post_kind[idx] = kind;
    return PLK_SUCCESS;
  }
  if (in->next_post_slot >= in->L.post_slots) return PLK_ERR_OUT_OF_MEMORY;
  in->post_slot[idx] = in->next_post_slot++;
  in->post_kind[idx] = kind;
  ++in->binding_epoch;
  return PLK_SUCCESS;
}
int bind_pre(plk_instance* in, int idx) {
  if (in->pre_slot[idx] >= 0) return PLK_SUCCESS;
  if (in->next_pre_slot >= in->L.pre_slots) return PLK_ERR_OUT_OF_MEMORY;
  in->pre_slot[idx] = in->next_pre_slot++;
  ++in->binding_epoch;
  return PLK_SUCCESS;
}

template <typename F>
int by_precision(const plk_instance* in, F&& f) {
  return in->f32 ? f(float()) : f(double());
}

inline unsigned blocks_for(size_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

// host fp64 -> device staging -> padded T rows at dst
int upload_rows(plk_instance* in, const double* src, void* dst, size_t rows) {
  const Layout& L = in->L;
  const size_t bytes = rows * L.S * 8;
  if (bytes > L.stage_bytes) return PLK_ERR_OUT_OF_MEMORY;
  double* stage = in->at<double>(L.off_stage);
  CU(cudaMemcpyAsync(stage, src, bytes, cudaMemcpyHostToDevice, in->stream));
  int rc = by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    k_pad_rows<T><<<blocks_for(rows * L.SP, 256), 256, 0, in->stream>>>(stage, static_cast<T*>(dst), rows, L.S, L.SP);
    return PLK_SUCCESS;
  });
  CHECK_LAUNCH(in);
  CU(cudaStreamSynchronize(in->stream));  // the staging area is reused by the next setter
  return rc;
}

int upload_small(plk_instance* in, const double* src, size_t n, size_t off, size_t n_padded) {
  std::vector<double> tmp(n_padded, 0.0);
  for (size_t i = 0; i < n; ++i) {
    if (!std::isfinite(src[i])) return PLK_ERR_OUT_OF_RANGE;
    tmp[i] = src[i];
  }
  CU(cudaMemcpyAsync(in->arena + off, tmp.data(), n_padded * 8, cudaMemcpyHostToDevice, in->stream));
  CU(cudaStreamSynchronize(in->stream));
  return PLK_SUCCESS;
}

int download(plk_instance* in, double* host, const double* dev, size_t n) {
  CU(cudaMemcpyAsync(host, dev, n * 8, cudaMemcpyDeviceToHost, in->stream));
  CU(cudaStreamSynchronize(in->stream));
  return PLK_SUCCESS;
}

// ---- kernel dispatch helpers ---------------------------------------------------------------------------------
// geometry of the 4-state kernels (plk_nuc.cuh): chunks of 32 / LP patterns, one warp each
struct NucGeom {
  int ppw, n_chunks, level_blocks;
};
inline NucGeom nuc_geom(const Layout& L) {
  NucGeom g;
  g.ppw = 32 / nuc_lanes_per_pattern(L.C);
  g.n_chunks = (L.P + g.ppw - 1) / g.ppw;
  g.level_blocks = (g.n_chunks + NUC_WARPS - 1) / NUC_WARPS;
  return g;
}
// walk shape: one resident wave in which every warp owns the same number of chunks (no tail wave)
template <typename K>
int nuc_walk_warps(const plk_instance* in, K kernel, int n_chunks, int* total_warps) {
  int blocks_per_sm = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, kernel, NUC_THREADS, 0));
  if (blocks_per_sm < 1) return PLK_ERR_CUDA;
  long resident = (long)in->sm_count * blocks_per_sm * NUC_WARPS;
  if (resident > NUC_MAX_WALK_WARPS) resident = NUC_MAX_WALK_WARPS;
  const int per_warp = (int)((n_chunks + resident - 1) / resident);
  *total_warps = (n_chunks + per_warp - 1) / per_warp;
  return PLK_SUCCESS;
}

// Which shape serves a call with `n_ops` operations in `n_levels` dependency levels:
// the walk costs one dependent global round trip per operation (~1 us) but a single launch and re-reads fresh
// children from L2; the level shape costs one launch (~4 us) per level.  Once the patterns alone fill the GPU the
// walk is bandwidth-bound like the level shape and moves fewer bytes, so it wins regardless of the list length.
// The specialised pre-order kernels (plk_nuc_lean.cuh) exist for C = 4 in the level order only.
inline bool nuc_lean_ok(const plk_instance* in) {
  return in->L.SP == 4 && in->L.C == 4 && !(in->cfg.flags & (PLK_FLAG_NO_TMA | PLK_FLAG_NO_LEVEL_BATCH | PLK_FLAG_PATTERN_WALK_ONLY));
}
// fp32 codon instances on tcgen05: the class-specialised, pipelined gradient kernels of plk_tc5_pre2.cuh
inline bool tc5_classes_ok(const plk_instance* in) {
#ifdef PLK_WITH_TENSOR
  return in->L.SP == 64 && in->f32 && (in->cfg.flags & PLK_FLAG_TENSOR_CORES) &&
         !(in->cfg.flags & (PLK_FLAG_NO_TCGEN05 | PLK_FLAG_NO_LEVEL_BATCH));
#else
  return false;
#endif
}
bool nuc_use_walk(const plk_instance* in, int n_ops, int n_levels, bool pre_gradient = false) {
  const int flags = in->cfg.flags;
  if (flags & (PLK_FLAG_NO_LEVEL_BATCH | PLK_FLAG_LEVEL_BATCH_ONLY)) return false;
  if (flags & PLK_FLAG_PATTERN_WALK_ONLY) return true;
  if (pre_gradient && nuc_lean_ok(in)) return false;
  const NucGeom g = nuc_geom(in->L);
  if (g.n_chunks >= in->sm_count * 8) return true;
  return (double)n_ops * 1.0 <= (double)n_levels * 4.0;
}

template <typename T>
int launch_post4(plk_instance* in, const DevOp* d_ops, int n_ops) {
  const Layout& L = in->L;
  dim3 grid(nuc_geom(L).level_blocks, n_ops);
  switch (L.C) {
#define CASE(CC) case CC: k_post4<T, CC><<<grid, NUC_THREADS, 0, in->stream>>>(d_ops, L.P); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return PLK_ERR_UNSUPPORTED;
  }
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}

template <typename T>
int launch_post4_walk(plk_instance* in, const DevOp* d_ops, int n_ops) {
  const Layout& L = in->L;
  const NucGeom g = nuc_geom(L);
  int tw = 0, rc = PLK_SUCCESS;
  switch (L.C) {
#define CASE(CC)                                                                                             \
  case CC:                                                                                                   \
    rc = nuc_walk_warps(in, k_post4_walk<T, CC>, g.n_chunks, &tw);                                           \
    if (rc) return rc;                                                                                       \
    k_post4_walk<T, CC><<<(tw + NUC_WARPS - 1) / NUC_WARPS, NUC_THREADS, 0, in->stream>>>(d_ops, n_ops, L.P, \
                                                                                           g.n_chunks, tw);  \
    break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return PLK_ERR_UNSUPPORTED;
  }
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}

inline NucModel nuc_model(const plk_instance* in, double* site) {
  const Layout& L = in->L;
  return NucModel{in->at<double>(L.off_catw), in->at<double>(L.off_rates), in->at<double>(L.off_weights), site};
}

template <typename T>
int launch_pre4(plk_instance* in, const DevPreItem* d_items, int n, const T* Q, double* site) {
  const Layout& L = in->L;
  const NucGeom g = nuc_geom(L);
  dim3 grid(g.level_blocks, n);
  const NucModel md = nuc_model(in, site);
  double* gp = in->at<double>(L.off_grad_partial);
  switch (L.C) {
#define CASE(CC) case CC: k_pre4<T, CC><<<grid, NUC_THREADS, 0, in->stream>>>(d_items, L.P, Q, md, gp, L.n_tiles); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return PLK_ERR_UNSUPPORTED;
  }
  CHECK_LAUNCH(in);
  in->grad_parts = g.level_blocks;
  return PLK_SUCCESS;
}

template <typename T>
int launch_pre4_walk(plk_instance* in, const DevPreItem* d_items, int n, const T* Q, double* site) {
  const Layout& L = in->L;
  const NucGeom g = nuc_geom(L);
  const NucModel md = nuc_model(in, site);
  double* gp = in->at<double>(L.off_grad_partial);
  int tw = 0, rc = PLK_SUCCESS;
  switch (L.C) {
#define CASE(CC)                                                                                           \
  case CC:                                                                                                 \
    rc = nuc_walk_warps(in, k_pre4_walk<T, CC>, g.n_chunks, &tw);                                          \
    if (rc) return rc;                                                                                     \
    k_pre4_walk<T, CC><<<(tw + NUC_WARPS - 1) / NUC_WARPS, NUC_THREADS, 0, in->stream>>>(d_items, n, L.P,  \
                                                                                          g.n_chunks, tw, \
                                                                                          Q, md, gp,       \
                                                                                          L.n_tiles);      \
    break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return PLK_ERR_UNSUPPORTED;
  }
  CHECK_LAUNCH(in);
  in->grad_parts = tw;
  return PLK_SUCCESS;
}

// ---- TMA-staged 4-state kernels (plk_nuc_tma.cuh) ------------------------------------------------------------
// walk = true: the one-launch order, where the register-staged kernels are the faster ones (they re-read fresh
// children from L2 with plain loads); the TMA walk runs only when the walk order is forced by flag.
inline bool nuc_use_tma(const plk_instance* in, bool walk = false) {
  const int C = in->L.C;
  if (walk && !(in->cfg.flags & PLK_FLAG_PATTERN_WALK_ONLY)) return false;
  return !(in->cfg.flags & (PLK_FLAG_NO_TMA | PLK_FLAG_NO_LEVEL_BATCH)) && (C == 1 || C == 2 || C == 4 || C == 8);
}
// grid of a TMA kernel: walk -> every CTA owns at least one full tile of rows; level -> at most one CTA per tile
template <typename K>
int nt_grid(plk_instance* in, K kernel, size_t smem, int which, bool walk, long long n_units, int* grid) {
  int& bps = in->nt_bps[which][walk ? 1 : 0];
  if (bps == 0) {
    CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, NT_THREADS, smem));
    if (bps < 1) return PLK_ERR_CUDA;
  }
  long long g = (long long)in->sm_count * bps;
  if (g > n_units) g = n_units;
  *grid = g < 1 ? 1 : (int)g;
  return PLK_SUCCESS;
}

template <typename T, int C>
int launch_post4_tma_c(plk_instance* in, const DevOp* d_ops, int n_ops, bool walk) {
  const Layout& L = in->L;
  using St = NtStage<T, C, 2, false>;
  const size_t smem = (size_t)NT_NS * St::BYTES;
  const int n_rows = (L.P + NucMap<C>::PPW - 1) / NucMap<C>::PPW;
  const long long n_tp = (L.P + St::TP - 1) / St::TP;
  NtSched sc{walk ? 1 : 0, n_ops, L.P, n_rows};
  int grid = 0, rc;
  if (walk) {
    rc = nt_grid(in, k_post4_tma<T, C, true>, smem, 0, true, n_rows / NT_CW > 0 ? n_rows / NT_CW : 1, &grid);
    if (rc) return rc;
    k_post4_tma<T, C, true><<<grid, NT_THREADS, smem, in->stream>>>(d_ops, sc);
  } else {
    rc = nt_grid(in, k_post4_tma<T, C, false>, smem, 0, false, n_tp * n_ops, &grid);
    if (rc) return rc;
    k_post4_tma<T, C, false><<<grid, NT_THREADS, smem, in->stream>>>(d_ops, sc);
  }
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}
template <typename T>
int launch_post4_tma(plk_instance* in, const DevOp* d_ops, int n_ops, bool walk) {
  switch (in->L.C) {
    case 1: return launch_post4_tma_c<T, 1>(in, d_ops, n_ops, walk);
    case 2: return launch_post4_tma_c<T, 2>(in, d_ops, n_ops, walk);
    case 4: return launch_post4_tma_c<T, 4>(in, d_ops, n_ops, walk);
    case 8: return launch_post4_tma_c<T, 8>(in, d_ops, n_ops, walk);
    default: return PLK_ERR_UNSUPPORTED;
  }
}

template <typename T, int C>
int launch_pre4_tma_c(plk_instance* in, const DevPreItem* d_items, int n, const T* Q, double* site, bool walk) {
  const Layout& L = in->L;
  using St = NtStage<T, C, 3, true>;
  const size_t smem = (size_t)NT_NS * St::BYTES;
  const int n_rows = (L.P + NucMap<C>::PPW - 1) / NucMap<C>::PPW;
  const long long n_tp = (L.P + St::TP - 1) / St::TP;
  NtSched sc{walk ? 1 : 0, n, L.P, n_rows};
  const NucModel md = nuc_model(in, site);
  double* gp = in->at<double>(L.off_grad_partial);
  int grid = 0, rc;
  if (walk) {
    rc = nt_grid(in, k_pre4_tma<T, C, true>, smem, 1, true, n_rows / NT_CW > 0 ? n_rows / NT_CW : 1, &grid);
    if (rc) return rc;
    k_pre4_tma<T, C, true><<<grid, NT_THREADS, smem, in->stream>>>(d_items, sc, Q, md, gp, L.n_tiles);
    in->grad_parts = grid * NT_CW;
  } else {
    rc = nt_grid(in, k_pre4_tma<T, C, false>, smem, 1, false, n_tp * n, &grid);
    if (rc) return rc;
    k_pre4_tma<T, C, false><<<grid, NT_THREADS, smem, in->stream>>>(d_items, sc, Q, md, gp, L.n_tiles);
    in->grad_parts = (int)n_tp * NT_CW;
  }
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}
template <typename T>
int launch_pre4_tma(plk_instance* in, const DevPreItem* d_items, int n, const T* Q, double* site, bool walk) {
  switch (in->L.C) {
    case 1: return launch_pre4_tma_c<T, 1>(in, d_items, n, Q, site, walk);
    case 2: return launch_pre4_tma_c<T, 2>(in, d_items, n, Q, site, walk);
    case 4: return launch_pre4_tma_c<T, 4>(in, d_items, n, Q, site, walk);
    case 8: return launch_pre4_tma_c<T, 8>(in, d_items, n, Q, site, walk);
    default: return PLK_ERR_UNSUPPORTED;
  }
}

// Launch with the programmatic-stream-serialisation attribute (programmatic dependent launch): the grid may become
// resident while the previous launch of the stream drains; the kernels order themselves with griddepcontrol
// (plk_nuc_lean.cuh).  pdl = false is a plain stream-ordered launch.
template <typename... KArgs, typename... Args>
cudaError_t launch_chain(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, bool pdl,
                         Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// specialised fused pre-order + gradient kernels (plk_nuc_lean.cuh): items of one class, level order.  `first`: the
// first launch of its dependency level (it waits for the previous level before it reads; the other classes of the
// level are independent of it and overlap its tail).
template <typename T, int CLS>
int launch_pre4_lean_c(plk_instance* in, const DevPreItem* d_items, int n, const double* h_q, double* site,
                       bool first) {
  const Layout& L = in->L;
  using St = NtStage<T, NL_C, 3, true, NlRows<T>::R>;
  const size_t smem = (size_t)NT_NS * St::BYTES;
  int& bps = in->lean_bps[CLS];
  if (bps == 0) {
    CU(cudaFuncSetAttribute(k_pre4_lean<T, CLS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_pre4_lean<T, CLS>, NT_THREADS, smem));
    if (bps < 1) return PLK_ERR_CUDA;
  }
  const long long n_tp = (L.P + St::TP - 1) / St::TP;
  long long g = (long long)in->sm_count * bps;
  if (g > n_tp * n) g = n_tp * n;
  const bool pdl = !(in->cfg.flags & PLK_FLAG_NO_PDL);
  NlQ<T> Q;
  for (int i = 0; i < 16; ++i) Q.v[i] = (T)h_q[i];
  CU(launch_chain(k_pre4_lean<T, CLS>, dim3((unsigned)g), dim3(NT_THREADS), smem, in->stream, pdl, d_items, n, L.P, Q,
                  (long long)L.off_matrix_d - (long long)L.off_matrix, nuc_model(in, site),
                  in->at<double>(L.off_grad_partial), L.n_tiles, (first || !pdl) ? 1 : 0));
  in->grad_parts = (int)n_tp * NT_CW;
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}
template <typename T>
int launch_pre4_lean(plk_instance* in, int cls, const DevPreItem* d_items, int n, const double* Q, double* site,
                     bool first_launch) {
  switch (cls) {
    case 0: return launch_pre4_lean_c<T, 0>(in, d_items, n, Q, site, first_launch);
    case 1: return launch_pre4_lean_c<T, 1>(in, d_items, n, Q, site, first_launch);
    case 2: {  // both children compact tips: lane-per-pattern kernel, no staging ring
      if (in->cfg.flags & PLK_FLAG_NO_TMA) return launch_pre4_lean_c<T, 2>(in, d_items, n, Q, site, first_launch);
      const Layout& L = in->L;
      const bool pdl = !(in->cfg.flags & PLK_FLAG_NO_PDL);
      constexpr int TPW = NlTipsTpw<T>::V;
      const int n_tp = (L.P + 32 * NlTipsRows<T>::R - 1) / (32 * NlTipsRows<T>::R);
      for (int first = 0; first < n; first += 32768) {
        const int m = n - first < 32768 ? n - first : 32768;
        dim3 grid((n_tp + NT_CW * TPW - 1) / (NT_CW * TPW), m);
        CU(launch_chain(k_grad4_tips<T>, grid, dim3(NT_CW * 32), 0, in->stream, pdl, d_items + first, L.P,
                        (long long)L.off_matrix_d - (long long)L.off_matrix, nuc_model(in, site),
                        in->at<double>(L.off_grad_partial), L.n_tiles, ((first_launch && first == 0) || !pdl) ? 1 : 0));
        CHECK_LAUNCH(in);
      }
      in->grad_parts = n_tp * NT_CW;
      return PLK_SUCCESS;
    }
    default: return PLK_ERR_GENERAL;
  }
}

template <typename T>
int launch_deriv4(plk_instance* in, const DevBranch* d_br, int n, const T* Q, double* site) {
  const Layout& L = in->L;
  dim3 grid(blocks_for(L.P, NUC_THREADS), n);
  const double* cw = in->at<double>(L.off_catw);
  const double* cr = in->at<double>(L.off_rates);
  const double* wt = in->at<double>(L.off_weights);
  double* gp = in->at<double>(L.off_grad_partial);
  switch (L.C) {
#define CASE(CC) case CC: k_deriv4<T, CC><<<grid, NUC_THREADS, 0, in->stream>>>(d_br, L.P, Q, cw, cr, wt, gp, L.n_tiles, site); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return PLK_ERR_UNSUPPORTED;
  }
  CHECK_LAUNCH(in);
  in->grad_parts = (int)grid.x;
  return PLK_SUCCESS;
}

template <typename K>
int opt_in_smem(K kernel, size_t bytes) {
  if (bytes > 48 * 1024) CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return PLK_SUCCESS;
}

template <typename T>
int launch_post64(plk_instance* in, const DevOp* d_ops, int n_ops) {
  const Layout& L = in->L;
  if (L.SP == 32) {  // 5..32 states: the CUDA-core kernels instantiated for 32 padded states (plk_gen.cuh)
    int rc = opt_in_smem(k_post64t<T, 32>, GenT<T, 32>::SMEM);
    if (rc) return rc;
    dim3 grid((L.P + GenT<T, 32>::PT - 1) / GenT<T, 32>::PT, L.C, n_ops);
    k_post64t<T, 32><<<grid, 128, GenT<T, 32>::SMEM, in->stream>>>(d_ops, L.P, L.S, L.C);
    CHECK_LAUNCH(in);
    return PLK_SUCCESS;
  }
#ifdef PLK_WITH_TENSOR
  if (in->cfg.flags & PLK_FLAG_TENSOR_CORES) {
    if (sizeof(T) == 4 && !(in->cfg.flags & PLK_FLAG_NO_TCGEN05))
      return tc5::launch_post(in->stream, d_ops, n_ops, L.P, L.S, L.C, in->sm_count, &in->launches);
    return tc_launch_post<T>(in->stream, d_ops, n_ops, L.P, L.S, L.C, in->sm_count, &in->launches);
  }
#endif
  int rc = opt_in_smem(k_post64t<T, 64>, GenT<T, 64>::SMEM);
  if (rc) return rc;
  dim3 grid((L.P + GenT<T, 64>::PT - 1) / GenT<T, 64>::PT, L.C, n_ops);
  k_post64t<T, 64><<<grid, 128, GenT<T, 64>::SMEM, in->stream>>>(d_ops, L.P, L.S, L.C);
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}

template <typename T>
int launch_pre64(plk_instance* in, const DevPreItem* d_items, int n, const T* Q, double* site) {
  const Layout& L = in->L;
  const double* cw = in->at<double>(L.off_catw);
  const double* cr = in->at<double>(L.off_rates);
  const double* wt = in->at<double>(L.off_weights);
  double* gp = in->at<double>(L.off_grad_partial);
  if (L.SP == 32) {
    int rc = opt_in_smem(k_pre64<T, 32>, pre64_smem<T, 32>());
    if (rc) return rc;
    dim3 grid(L.n_tiles, n);
    k_pre64<T, 32><<<grid, GEN_THREADS, pre64_smem<T, 32>(), in->stream>>>(d_items, L.P, L.S, L.C, Q, cw, cr, wt, gp, L.n_tiles, site);
    CHECK_LAUNCH(in);
    in->grad_parts = L.n_tiles;
    return PLK_SUCCESS;
  }
#ifdef PLK_WITH_TENSOR
  if (in->cfg.flags & PLK_FLAG_TENSOR_CORES)
  {
    if constexpr (sizeof(T) == 4) {
      if (!(in->cfg.flags & PLK_FLAG_NO_TCGEN05))
        return tc5::pre::launch_pre(in->stream, d_items, n, L.P, L.S, L.C, Q, (long long)L.off_matrix_t - (long long)L.off_matrix,
                                    cw, cr, wt, gp, L.n_tiles, site, in->sm_count, &in->grad_parts, &in->launches);
    }
    return tc_launch_pre<T>(in->stream, d_items, n, L.P, L.S, L.C, Q, cw, cr, wt, gp, L.n_tiles, site, &in->grad_parts,
                            &in->launches);
  }
#endif
  int rc = opt_in_smem(k_pre64<T>, pre64_smem<T>());
  if (rc) return rc;
  dim3 grid(L.n_tiles, n);
  k_pre64<T><<<grid, GEN_THREADS, pre64_smem<T>(), in->stream>>>(d_items, L.P, L.S, L.C, Q, cw, cr, wt, gp, L.n_tiles, site);
  CHECK_LAUNCH(in);
  in->grad_parts = L.n_tiles;
  return PLK_SUCCESS;
}

template <typename T>
int launch_deriv64(plk_instance* in, const DevBranch* d_br, int n, const T* Q, double* site) {
  const Layout& L = in->L;
  if (L.SP == 32) {
    int r2 = opt_in_smem(k_deriv64<T, 32>, deriv64_smem<T, 32>());
    if (r2) return r2;
    dim3 grid32(L.n_tiles, n);
    k_deriv64<T, 32><<<grid32, GEN_THREADS, deriv64_smem<T, 32>(), in->stream>>>(
        d_br, L.P, L.S, L.C, Q, in->at<double>(L.off_catw), in->at<double>(L.off_rates), in->at<double>(L.off_weights),
        in->at<double>(L.off_grad_partial), L.n_tiles, site);
    CHECK_LAUNCH(in);
    in->grad_parts = L.n_tiles;
    return PLK_SUCCESS;
  }
  int rc = opt_in_smem(k_deriv64<T>, deriv64_smem<T>());
  if (rc) return rc;
  dim3 grid(L.n_tiles, n);
  k_deriv64<T><<<grid, GEN_THREADS, deriv64_smem<T>(), in->stream>>>(
      d_br, L.P, L.S, L.C, Q, in->at<double>(L.off_catw), in->at<double>(L.off_rates), in->at<double>(L.off_weights),
      in->at<double>(L.off_grad_partial), L.n_tiles, site);
  CHECK_LAUNCH(in);
  in->grad_parts = L.n_tiles;
  return PLK_SUCCESS;
}

int check_model_ready(const plk_instance* in, bool need_rates) {
  if (!in->have_catw || !in->have_pi || !in->have_weights) return PLK_ERR_UNINITIALIZED;
  if (need_rates && !in->have_rates) return PLK_ERR_UNINITIALIZED;
  return PLK_SUCCESS;
}

// operand description of a post-order buffer used as input
int operand_of(const plk_instance* in, int idx, const void** ptr, int* kind, const void** pending) {
  if (idx < 0 || idx >= in->cfg.partials_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (in->post_slot[idx] < 0 || !in->post_written[idx]) return PLK_ERR_UNINITIALIZED;
  *ptr = in->post_ptr(idx);
  *kind = in->post_kind[idx];
  *pending = (in->deferred && in->post_pending_scale[idx] >= 0) ? in->scale_ptr(in->post_pending_scale[idx]) : nullptr;
  return PLK_SUCCESS;
}


// P:101 variant (a): Qp_k = Q p_k for the listed post-order buffers (full or single-category partials; compact tips
// need none), stored in the slot that shadows the buffer's partials slot.
int cache_rate_products_impl(plk_instance* in, int eigen, const int32_t* post_idx, int count) {
  const Layout& L = in->L;
  if (!(in->cfg.flags & PLK_FLAG_CACHE_RATE_PRODUCTS)) return PLK_ERR_UNSUPPORTED;
  if (count < 0 || (count > 0 && post_idx == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  if (eigen < 0 || eigen >= in->cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->q_written[eigen]) return PLK_ERR_UNINITIALIZED;
  std::vector<DevQpItem> items;
  for (int i = 0; i < count; ++i) {
    const void* ptr;
    const void* pending;
    int kind;
    int rc = operand_of(in, post_idx[i], &ptr, &kind, &pending);
    if (rc) return rc;
    in->qp_valid[post_idx[i]] = 1;
    if (kind == KIND_STATES) continue;  // Q e_z is a column of Q: nothing to cache
    items.push_back(DevQpItem{ptr, in->qp_ptr(post_idx[i]), kind, 0});
  }
  const int n = (int)items.size();
  if (n == 0) return PLK_SUCCESS;
  char *h, *d;
  int rc = ring_alloc(in, (size_t)n * sizeof(DevQpItem), &h, &d);
  if (rc) return rc;
  std::memcpy(h, items.data(), (size_t)n * sizeof(DevQpItem));
  rc = copy_ring(in, h, d, (size_t)n * sizeof(DevQpItem));
  if (rc) return rc;
  const DevQpItem* di = reinterpret_cast<const DevQpItem*>(d);
  for (int first = 0; first < n; first += 32768) {
    const int m = n - first < 32768 ? n - first : 32768;
    rc = by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      const T* Q = static_cast<const T*>(in->eig_QT(eigen));
      if (L.SP == 4) {
        dim3 grid(blocks_for((size_t)L.C * L.P, 256), m);
        k_rate_products4<T><<<grid, 256, 0, in->stream>>>(di + first, L.P, L.C, Q);
      } else if (L.SP == 32) {
        int r2 = opt_in_smem(k_rate_products64<T, 32>, rate_products64_smem<T, 32>());
        if (r2) return r2;
        dim3 grid(L.n_tiles, L.C, m);
        k_rate_products64<T, 32><<<grid, GEN_THREADS, rate_products64_smem<T, 32>(), in->stream>>>(di + first, L.P, L.S, L.C, Q);
      } else {
        int r2 = opt_in_smem(k_rate_products64<T>, rate_products64_smem<T>());
        if (r2) return r2;
        dim3 grid(L.n_tiles, L.C, m);
        k_rate_products64<T><<<grid, GEN_THREADS, rate_products64_smem<T>(), in->stream>>>(di + first, L.P, L.S, L.C, Q);
      }
      return PLK_SUCCESS;
    });
    if (rc) return rc;
    CHECK_LAUNCH(in);
  }
  return PLK_SUCCESS;
}

}  // namespace

// =================================================================================================================
extern "C" {

size_t plk_arena_bytes(const plk_config* cfg) {
  Layout L;
  if (cfg == nullptr || !compute_layout(*cfg, L)) return 0;
  return L.total;
}

int plk_create(const plk_config* cfg, void* d_arena, size_t arena_bytes, void* cuda_stream, plk_instance** out) {
  if (out == nullptr) return PLK_ERR_OUT_OF_RANGE;
  *out = nullptr;
  if (cfg == nullptr || d_arena == nullptr) return PLK_ERR_OUT_OF_RANGE;
  Layout L;
  if (!compute_layout(*cfg, L)) {
    if (cfg->state_count < 2 || cfg->state_count > 64) return PLK_ERR_UNSUPPORTED;
    if (cfg->state_count == 4 && cfg->category_count > 8) return PLK_ERR_UNSUPPORTED;
    return PLK_ERR_OUT_OF_RANGE;
  }
  if (cfg->flags & ~(PLK_FLAG_TENSOR_CORES | PLK_FLAG_NO_LEVEL_BATCH | PLK_FLAG_SITE_DERIVATIVES | PLK_FLAG_LEVEL_BATCH_ONLY |
                     PLK_FLAG_PATTERN_WALK_ONLY | PLK_FLAG_NO_TMA | PLK_FLAG_NO_TCGEN05 | PLK_FLAG_NO_PDL |
                     PLK_FLAG_CACHE_RATE_PRODUCTS | PLK_FLAG_ON_THE_FLY_MATRICES))
    return PLK_ERR_UNSUPPORTED;
  if ((cfg->flags & PLK_FLAG_ON_THE_FLY_MATRICES) && L.SP == 4) return PLK_ERR_UNSUPPORTED;  // large state spaces only
  if ((cfg->flags & PLK_FLAG_LEVEL_BATCH_ONLY) && (cfg->flags & PLK_FLAG_PATTERN_WALK_ONLY)) return PLK_ERR_UNSUPPORTED;
#ifndef PLK_WITH_TENSOR
  if ((cfg->flags & PLK_FLAG_TENSOR_CORES) && L.SP == 64) return PLK_ERR_UNSUPPORTED;
#endif
  if (arena_bytes < L.total) return PLK_ERR_OUT_OF_MEMORY;
  if (reinterpret_cast<uintptr_t>(d_arena) % ALIGN != 0) return PLK_ERR_OUT_OF_RANGE;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) return PLK_ERR_CUDA;
  int dev = 0, sms = 0;
  cudaPointerAttributes pa;
  if (cudaPointerGetAttributes(&pa, d_arena) != cudaSuccess || pa.type != cudaMemoryTypeDevice) return PLK_ERR_CUDA;
  dev = pa.device;  // the arena's device (the caller keeps it current while it uses the instance)
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return PLK_ERR_CUDA;
  plk_instance* in = new (std::nothrow) plk_instance();
  if (in == nullptr) return PLK_ERR_OUT_OF_MEMORY;
  in->cfg = *cfg;
  in->L = L;
  in->stream = static_cast<cudaStream_t>(cuda_stream);
  in->arena = static_cast<char*>(d_arena);
  in->f32 = cfg->precision == PLK_FP32;
  in->sm_count = sms;
  in->deferred = L.SP != 4;
  in->post_slot.assign(cfg->partials_buffer_count, -1);
  in->post_kind.assign(cfg->partials_buffer_count, KIND_PARTIALS);
  in->post_pending_scale.assign(cfg->partials_buffer_count, -1);
  in->post_written.assign(cfg->partials_buffer_count, 0);
  in->qp_valid.assign(cfg->partials_buffer_count, 0);
  in->pre_slot.assign(cfg->preorder_buffer_count, -1);
  in->pre_written.assign(cfg->preorder_buffer_count, 0);
  in->pre_has_mx.assign(cfg->preorder_buffer_count, 0);
  in->matrix_written.assign(cfg->matrix_buffer_count, 0);
  in->scale_written.assign(cfg->scale_buffer_count, 0);
  in->eigen_written.assign(cfg->eigen_buffer_count, 0);
  in->q_written.assign(cfg->eigen_buffer_count, 0);
  in->h_q4.assign((size_t)cfg->eigen_buffer_count * 16, 0.0);
  if (cudaHostAlloc(reinterpret_cast<void**>(&in->h_ring), RING_BYTES, cudaHostAllocDefault) != cudaSuccess) {
    delete in;
    return PLK_ERR_CUDA;
  }
  // zero everything outside the big partials regions once: padding of matrices / frequencies must be zero
  const size_t small_from = L.off_matrix;
  if (cudaMemsetAsync(in->arena + small_from, 0, L.total - small_from, in->stream) != cudaSuccess ||
      cudaStreamSynchronize(in->stream) != cudaSuccess) {
    cudaFreeHost(in->h_ring);
    delete in;
    return PLK_ERR_CUDA;
  }
  *out = in;
  return PLK_SUCCESS;
}

int plk_destroy(plk_instance* in) {
  if (in == nullptr) return PLK_SUCCESS;
  cudaStreamSynchronize(in->stream);
  for (auto& pl : in->plans)
    if (pl.exec != nullptr) cudaGraphExecDestroy(pl.exec);
  if (in->h_ring) cudaFreeHost(in->h_ring);
  delete in;
  return PLK_SUCCESS;
}

const char* plk_error_string(int status) {
  switch (status) {
    case PLK_SUCCESS: return "success";
    case PLK_ERR_GENERAL: return "general error";
    case PLK_ERR_OUT_OF_MEMORY: return "arena too small or no free buffer slot";
    case PLK_ERR_OUT_OF_RANGE: return "index, count, shape or value out of range";
    case PLK_ERR_UNINITIALIZED: return "buffer or model component read before it was written";
    case PLK_ERR_UNSUPPORTED: return "unsupported configuration";
    case PLK_ERR_FLOATING_POINT: return "log-likelihood or derivative is not finite";
    case PLK_ERR_CUDA: return "CUDA error (no device or a runtime call failed)";
    case PLK_ERR_STOP_CODON: return "stop codon in a codon alignment";
    case PLK_ERR_STATIC_SCRATCH_LIMIT:
      return "problem exceeds the static scratch of the no-allocation entry point (PLK_STATIC_SCRATCH_DOUBLES / PLK_STATIC_SCALE_MAX)";
    default: return "unknown status";
  }
}

// ---- setters ----------------------------------------------------------------------------------------------------

int plk_set_tip_states(plk_instance* in, int tip, const int32_t* states) {
  if (in == nullptr || states == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (tip < 0 || tip >= in->cfg.tip_count) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  if (!(in->post_slot[tip] >= 0 && in->post_kind[tip] == KIND_STATES)) {
    if (in->post_slot[tip] >= 0) return PLK_ERR_OUT_OF_RANGE;  // already bound as partials
    if (in->next_compact_slot >= L.compact_slots) return PLK_ERR_OUT_OF_MEMORY;
    in->post_slot[tip] = in->next_compact_slot++;
    in->post_kind[tip] = KIND_STATES;
    ++in->binding_epoch;
  }
  if ((size_t)L.P * 4 > L.stage_bytes) return PLK_ERR_OUT_OF_MEMORY;
  int32_t* stage = in->at<int32_t>(L.off_stage);
  CU(cudaMemcpyAsync(stage, states, (size_t)L.P * 4, cudaMemcpyHostToDevice, in->stream));
  k_pack_states<<<blocks_for(L.P, 256), 256, 0, in->stream>>>(stage, static_cast<uint8_t*>(in->post_ptr(tip)), L.P, L.S);
  CHECK_LAUNCH(in);
  CU(cudaStreamSynchronize(in->stream));
  in->post_written[tip] = 1;
  in->post_pending_scale[tip] = -1;
  return PLK_SUCCESS;
}

int plk_set_tip_states_u8(plk_instance* in, int tip, const uint8_t* states) {
  if (in == nullptr || states == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (tip < 0 || tip >= in->cfg.tip_count) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  if (!(in->post_slot[tip] >= 0 && in->post_kind[tip] == KIND_STATES)) {
    if (in->post_slot[tip] >= 0) return PLK_ERR_OUT_OF_RANGE;  // already bound as partials
    if (in->next_compact_slot >= L.compact_slots) return PLK_ERR_OUT_OF_MEMORY;
    in->post_slot[tip] = in->next_compact_slot++;
    in->post_kind[tip] = KIND_STATES;
    ++in->binding_epoch;
  }
  CU(cudaMemcpyAsync(in->post_ptr(tip), states, (size_t)L.P, cudaMemcpyHostToDevice, in->stream));
  in->post_written[tip] = 1;
  in->post_pending_scale[tip] = -1;
  return PLK_SUCCESS;
}

int plk_set_all_tip_states_u8(plk_instance* in, const uint8_t* states, int count) {
  if (in == nullptr || states == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (count < 0 || count > in->cfg.tip_count) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  int fresh = 0;
  for (int tip = 0; tip < count; ++tip) {
    if (in->post_slot[tip] >= 0 && in->post_kind[tip] != KIND_STATES) return PLK_ERR_OUT_OF_RANGE;  // bound as partials
    if (in->post_slot[tip] < 0) ++fresh;
  }
  if (in->next_compact_slot + fresh > L.compact_slots) return PLK_ERR_OUT_OF_MEMORY;
  for (int tip = 0; tip < count; ++tip)
    if (in->post_slot[tip] < 0) {
      in->post_slot[tip] = in->next_compact_slot++;
      in->post_kind[tip] = KIND_STATES;
      ++in->binding_epoch;
    }
  // runs of tips that sit in consecutive compact slots travel as ONE pitched copy (usually a single run: all tips)
  for (int first = 0; first < count;) {
    int last = first;
    while (last + 1 < count && in->post_slot[last + 1] == in->post_slot[last] + 1) ++last;
    // a pitched host -> device copy runs at a third of the PCIe rate (one DMA descriptor per row: 0.75 ms for 12.8 MB);
    // so: one LINEAR copy of as many rows as the staging area holds, then a kernel scatters the rows into the slots
    const size_t rows_per_chunk = L.compact_bytes == (size_t)L.P ? (size_t)(last - first + 1) : L.stage_bytes / (size_t)L.P;
    if (rows_per_chunk == 0) return PLK_ERR_OUT_OF_MEMORY;
    for (int r0 = first; r0 <= last; r0 += (int)rows_per_chunk) {
      const size_t rows = (size_t)(last - r0 + 1) < rows_per_chunk ? (size_t)(last - r0 + 1) : rows_per_chunk;
      const uint8_t* src = states + (size_t)r0 * L.P;
      if (L.compact_bytes == (size_t)L.P) {
        CU(cudaMemcpyAsync(in->post_ptr(r0), src, rows * L.P, cudaMemcpyHostToDevice, in->stream));
      } else {
        char* stage = in->arena + L.off_stage;
        CU(cudaMemcpyAsync(stage, src, rows * L.P, cudaMemcpyHostToDevice, in->stream));
        k_scatter_rows<<<dim3(blocks_for(((size_t)L.P + 15) / 16, 256), (unsigned)rows), 256, 0, in->stream>>>(
            reinterpret_cast<const uint8_t*>(stage), static_cast<uint8_t*>(in->post_ptr(r0)), (size_t)L.P, L.compact_bytes);
        CHECK_LAUNCH(in);
      }
    }
    first = last + 1;
  }
  for (int tip = 0; tip < count; ++tip) {
    in->post_written[tip] = 1;
    in->post_pending_scale[tip] = -1;
  }
  return PLK_SUCCESS;
}

int plk_set_tip_partials(plk_instance* in, int tip, const double* partials) {
  if (in == nullptr || partials == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (tip < 0 || tip >= in->cfg.tip_count) return PLK_ERR_OUT_OF_RANGE;
  if (in->post_slot[tip] >= 0 && in->post_kind[tip] == KIND_STATES) return PLK_ERR_OUT_OF_RANGE;
  int rc = bind_post_full(in, tip, KIND_BCAST);
  if (rc) return rc;
  rc = upload_rows(in, partials, in->post_ptr(tip), (size_t)in->L.P);
  if (rc) return rc;
  in->qp_valid[tip] = 0;
  in->post_written[tip] = 1;
  in->post_pending_scale[tip] = -1;
  return PLK_SUCCESS;
}

int plk_set_partials(plk_instance* in, int buffer, const double* partials) {
  if (in == nullptr || partials == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (buffer < 0 || buffer >= in->cfg.partials_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (in->post_slot[buffer] >= 0 && in->post_kind[buffer] == KIND_STATES) return PLK_ERR_OUT_OF_RANGE;
  int rc = bind_post_full(in, buffer, KIND_PARTIALS);
  if (rc) return rc;
  rc = upload_rows(in, partials, in->post_ptr(buffer), (size_t)in->L.C * in->L.P);
  if (rc) return rc;
  in->qp_valid[buffer] = 0;
  in->post_written[buffer] = 1;
  in->post_pending_scale[buffer] = -1;
  return PLK_SUCCESS;
}

int plk_set_pattern_weights(plk_instance* in, const double* w) {
  if (in == nullptr || w == nullptr) return PLK_ERR_OUT_OF_RANGE;
  int rc = upload_small(in, w, in->L.P, in->L.off_weights, in->L.P);
  if (rc == PLK_SUCCESS) in->have_weights = true;
  return rc;
}
int plk_set_state_frequencies(plk_instance* in, const double* pi) {
  if (in == nullptr || pi == nullptr) return PLK_ERR_OUT_OF_RANGE;
  int rc = upload_small(in, pi, in->L.S, in->L.off_pi, in->L.SP);
  if (rc == PLK_SUCCESS) {
    in->have_pi = true;
    in->root_pre_filled = -1;
  }
  return rc;
}
int plk_set_category_rates(plk_instance* in, const double* r) {
  if (in == nullptr || r == nullptr) return PLK_ERR_OUT_OF_RANGE;
  int rc = upload_small(in, r, in->L.C, in->L.off_rates, in->L.C);
  if (rc == PLK_SUCCESS) in->have_rates = true;
  return rc;
}
int plk_set_category_weights(plk_instance* in, const double* w) {
  if (in == nullptr || w == nullptr) return PLK_ERR_OUT_OF_RANGE;
  int rc = upload_small(in, w, in->L.C, in->L.off_catw, in->L.C);
  if (rc == PLK_SUCCESS) in->have_catw = true;
  return rc;
}

static int rebuild_rate_matrix(plk_instance* in, int eigen) {
  const Layout& L = in->L;
  char *h, *d;
  int rc = ring_alloc(in, sizeof(void*), &h, &d);
  if (rc) return rc;
  void* qt = in->eig_QT(eigen);
  std::memcpy(h, &qt, sizeof(void*));
  rc = copy_ring(in, h, d, sizeof(void*));
  if (rc) return rc;
  const size_t smem = transition_smem(L.S);
  rc = by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    int r2 = opt_in_smem(k_transition<T>, smem);
    if (r2) return r2;
    k_transition<T><<<dim3(1, 1), 256, smem, in->stream>>>(in->eig_U(eigen), in->eig_Uinv(eigen), in->eig_lam(eigen), nullptr,
                                                 nullptr, reinterpret_cast<void* const*>(d), in->eig_Q64(eigen), L.S,
                                                 L.SP, 1, 1);
    return PLK_SUCCESS;
  });
  if (rc) return rc;
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}

// 4-state instances keep a host copy of Q in working precision: the class-specialised gradient kernels take it by
// value (plk_nuc_lean.cuh NlQ).  Called by the two setters of Q, which synchronise anyway.
static int fetch_q4(plk_instance* in, int eigen) {
  if (in->L.SP != 4) return PLK_SUCCESS;
  double* dst = in->h_q4.data() + (size_t)eigen * 16;
  if (in->f32) {
    float q[16];
    CU(cudaMemcpyAsync(q, in->eig_QT(eigen), sizeof(q), cudaMemcpyDeviceToHost, in->stream));
    CU(cudaStreamSynchronize(in->stream));
    for (int i = 0; i < 16; ++i) dst[i] = q[i];
  } else {
    CU(cudaMemcpyAsync(dst, in->eig_QT(eigen), 16 * sizeof(double), cudaMemcpyDeviceToHost, in->stream));
    CU(cudaStreamSynchronize(in->stream));
  }
  return PLK_SUCCESS;
}

int plk_set_eigen_decomposition(plk_instance* in, int eigen, const double* U, const double* Uinv, const double* lam) {
  if (in == nullptr || U == nullptr || Uinv == nullptr || lam == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (eigen < 0 || eigen >= in->cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  const int S = in->L.S;
  for (int i = 0; i < S * S; ++i)
    if (!std::isfinite(U[i]) || !std::isfinite(Uinv[i])) return PLK_ERR_OUT_OF_RANGE;
  for (int i = 0; i < S; ++i)
    if (!std::isfinite(lam[i])) return PLK_ERR_OUT_OF_RANGE;
  CU(cudaMemcpyAsync(in->eig_U(eigen), U, (size_t)S * S * 8, cudaMemcpyHostToDevice, in->stream));
  CU(cudaMemcpyAsync(in->eig_Uinv(eigen), Uinv, (size_t)S * S * 8, cudaMemcpyHostToDevice, in->stream));
  CU(cudaMemcpyAsync(in->eig_lam(eigen), lam, (size_t)S * 8, cudaMemcpyHostToDevice, in->stream));
  int rc = rebuild_rate_matrix(in, eigen);
  if (rc) return rc;
  CU(cudaStreamSynchronize(in->stream));
  rc = fetch_q4(in, eigen);
  if (rc) return rc;
  in->eigen_written[eigen] = 1;
  in->q_written[eigen] = 1;
  ++in->model_epoch;
  return PLK_SUCCESS;
}

int plk_set_rate_matrix(plk_instance* in, int eigen, const double* Q) {
  if (in == nullptr || Q == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (eigen < 0 || eigen >= in->cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  for (int i = 0; i < L.S * L.S; ++i)
    if (!std::isfinite(Q[i])) return PLK_ERR_OUT_OF_RANGE;
  CU(cudaMemcpyAsync(in->eig_Q64(eigen), Q, (size_t)L.S * L.S * 8, cudaMemcpyHostToDevice, in->stream));
  by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    k_pad_matrices<T><<<blocks_for((size_t)L.SP * L.SP, 256), 256, 0, in->stream>>>(
        in->eig_Q64(eigen), static_cast<T*>(in->eig_QT(eigen)), 1, L.S, L.SP);
    return PLK_SUCCESS;
  });
  CHECK_LAUNCH(in);
  CU(cudaStreamSynchronize(in->stream));
  int rc = fetch_q4(in, eigen);
  if (rc) return rc;
  in->q_written[eigen] = 1;
  ++in->model_epoch;
  return PLK_SUCCESS;
}

int plk_set_transition_matrix(plk_instance* in, int matrix, const double* m) {
  if (in == nullptr || m == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (matrix < 0 || matrix >= in->cfg.matrix_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  const size_t bytes = (size_t)L.C * L.S * L.S * 8;
  if (bytes > L.stage_bytes) return PLK_ERR_OUT_OF_MEMORY;
  double* stage = in->at<double>(L.off_stage);
  CU(cudaMemcpyAsync(stage, m, bytes, cudaMemcpyHostToDevice, in->stream));
  by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    k_pad_matrices<T><<<blocks_for((size_t)L.C * L.SP * L.SP, 256), 256, 0, in->stream>>>(
        stage, static_cast<T*>(in->matrix_ptr(matrix)), L.C, L.S, L.SP);
    return PLK_SUCCESS;
  });
  CHECK_LAUNCH(in);
  CU(cudaStreamSynchronize(in->stream));
  in->matrix_written[matrix] = 1;
  return PLK_SUCCESS;
}

// ---- step 1: transition matrices ------------------------------------------------------------------------------

static int update_matrices_impl(plk_instance* in, int eigen, const int32_t* matrix_idx, const double* h_t,
                                const double* d_t, int count) {
  if (in == nullptr || count < 0) return PLK_ERR_OUT_OF_RANGE;
  if (count == 0) return PLK_SUCCESS;
  if (matrix_idx == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (eigen < 0 || eigen >= in->cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->eigen_written[eigen] || !in->have_rates) return PLK_ERR_UNINITIALIZED;
  const Layout& L = in->L;
  for (int i = 0; i < count; ++i) {
    if (matrix_idx[i] < 0 || matrix_idx[i] >= in->cfg.matrix_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (h_t != nullptr && !(h_t[i] >= 0.0 && std::isfinite(h_t[i]))) return PLK_ERR_OUT_OF_RANGE;
  }
  char *h, *d;
  const size_t ptr_bytes = round_up((size_t)count * sizeof(void*), 256);
  int rc = ring_alloc(in, ptr_bytes + (size_t)count * 8, &h, &d);
  if (rc) return rc;
  void** hp = reinterpret_cast<void**>(h);
  for (int i = 0; i < count; ++i) hp[i] = in->matrix_ptr(matrix_idx[i]);
  size_t bytes = ptr_bytes;
  if (h_t != nullptr) {
    std::memcpy(h + ptr_bytes, h_t, (size_t)count * 8);
    bytes += (size_t)count * 8;
    d_t = reinterpret_cast<const double*>(d + ptr_bytes);
  }
  rc = copy_ring(in, h, d, bytes);
  if (rc) return rc;
  const size_t smem = transition_smem(L.S);
  rc = by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    int r2 = opt_in_smem(k_transition<T>, smem);
    if (r2) return r2;
    k_transition<T><<<dim3(count, L.C), L.S <= 8 ? 32 : 256, smem, in->stream>>>(in->eig_U(eigen), in->eig_Uinv(eigen), in->eig_lam(eigen),
                                                     in->at<double>(L.off_rates), d_t,
                                                     reinterpret_cast<void* const*>(d), nullptr, L.S, L.SP, L.C, 0);
    return PLK_SUCCESS;
  });
  if (rc) return rc;
  CHECK_LAUNCH(in);
  for (int i = 0; i < count; ++i) in->matrix_written[matrix_idx[i]] = 1;
  return PLK_SUCCESS;
}

int plk_update_transition_matrices(plk_instance* in, int eigen, const int32_t* matrix_idx, const double* t, int count) {
  if (count > 0 && t == nullptr) return PLK_ERR_OUT_OF_RANGE;
  return update_matrices_impl(in, eigen, matrix_idx, t, nullptr, count);
}
int plk_update_transition_matrices_device(plk_instance* in, int eigen, const int32_t* matrix_idx, const double* d_t,
                                          int count) {
  if (count > 0 && d_t == nullptr) return PLK_ERR_OUT_OF_RANGE;
  return update_matrices_impl(in, eigen, matrix_idx, nullptr, d_t, count);
}

// ---- steps 2-3: post-order ---------------------------------------------------------------------------------------

int plk_update_partials(plk_instance* in, const plk_op* ops, int count) {
  if (in == nullptr || count < 0) return PLK_ERR_OUT_OF_RANGE;
  if (count == 0) return PLK_SUCCESS;
  std::vector<int> level;
  const int n_levels = schedule_post(ops, count, level);
  if (n_levels < 0) return n_levels;
  const plk_config& cfg = in->cfg;
  // validate everything before touching any state
  for (int i = 0; i < count; ++i) {
    const plk_op& o = ops[i];
    if (o.dest >= cfg.partials_buffer_count || o.child1 >= cfg.partials_buffer_count ||
        o.child2 >= cfg.partials_buffer_count || o.child1_matrix >= cfg.matrix_buffer_count ||
        o.child2_matrix >= cfg.matrix_buffer_count || o.dest_scale >= cfg.scale_buffer_count || o.dest_scale < -1)
      return PLK_ERR_OUT_OF_RANGE;
    if (!in->matrix_written[o.child1_matrix] || !in->matrix_written[o.child2_matrix]) return PLK_ERR_UNINITIALIZED;
    if (in->post_slot[o.dest] >= 0 && in->post_kind[o.dest] == KIND_STATES) return PLK_ERR_OUT_OF_RANGE;
  }
  {  // children must be written already or produced earlier in this list
    std::vector<char> will(cfg.partials_buffer_count, 0);
    int fresh = 0;
    for (int i = 0; i < count; ++i) {
      const plk_op& o = ops[i];
      if (!(in->post_written[o.child1] || will[o.child1]) || !(in->post_written[o.child2] || will[o.child2]))
        return PLK_ERR_UNINITIALIZED;
      if (in->post_slot[o.dest] < 0 && !will[o.dest]) ++fresh;
      will[o.dest] = 1;
    }
    if (in->next_post_slot + fresh > in->L.post_slots) return PLK_ERR_OUT_OF_MEMORY;
  }
  // host bookkeeping in list order, launch items sorted by level
  std::vector<DevOp> items(count);
  for (int i = 0; i < count; ++i) {
    const plk_op& o = ops[i];
    int rc = bind_post_full(in, o.dest, KIND_PARTIALS);
    if (rc) return rc;
    DevOp& d = items[i];
    d.dest = in->post_ptr(o.dest);
    const int ch[2] = {o.child1, o.child2};
    const int mt[2] = {o.child1_matrix, o.child2_matrix};
    for (int k = 0; k < 2; ++k) {
      rc = operand_of(in, ch[k], &d.child[k], &d.kind[k], &d.cscale[k]);
      if (rc) return rc;
      d.mat[k] = in->matrix_ptr(mt[k]);
    }
    d.scale = o.dest_scale >= 0 ? in->scale_ptr(o.dest_scale) : nullptr;
    in->post_written[o.dest] = 1;
    in->post_pending_scale[o.dest] = in->deferred ? o.dest_scale : -1;
    if (o.dest_scale >= 0) in->scale_written[o.dest_scale] = 1;
  }
  std::vector<int> order(count);
  std::vector<int> level_start(n_levels + 1, 0);
  const bool walk = in->L.SP == 4 && nuc_use_walk(in, count, n_levels);
  if (walk || (cfg.flags & PLK_FLAG_NO_LEVEL_BATCH)) {
    for (int i = 0; i < count; ++i) order[i] = i;
  } else {
    for (int i = 0; i < count; ++i) ++level_start[level[i] + 1];
    for (int l = 0; l < n_levels; ++l) level_start[l + 1] += level_start[l];
    std::vector<int> fill(level_start.begin(), level_start.end() - 1);
    for (int i = 0; i < count; ++i) order[fill[level[i]]++] = i;
  }
  char *h, *d;
  int rc = ring_alloc(in, (size_t)count * sizeof(DevOp), &h, &d);
  if (rc) return rc;
  DevOp* hops = reinterpret_cast<DevOp*>(h);
  for (int i = 0; i < count; ++i) hops[i] = items[order[i]];
  rc = copy_ring(in, h, d, (size_t)count * sizeof(DevOp));
  if (rc) return rc;
  const DevOp* dops = reinterpret_cast<const DevOp*>(d);
  auto launch = [&](int first, int n) {
    return by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      if (in->L.SP != 4) return launch_post64<T>(in, dops + first, n);
      return nuc_use_tma(in) ? launch_post4_tma<T>(in, dops + first, n, false) : launch_post4<T>(in, dops + first, n);
    });
  };
  if (walk) {  // one launch, list order (plk_nuc.cuh "walk")
    rc = by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      return nuc_use_tma(in, true) ? launch_post4_tma<T>(in, dops, count, true) : launch_post4_walk<T>(in, dops, count);
    });
    if (rc) return rc;
  } else if (cfg.flags & PLK_FLAG_NO_LEVEL_BATCH) {
    for (int i = 0; i < count; ++i) {
      rc = launch(i, 1);
      if (rc) return rc;
    }
  } else {
    for (int l = 0; l < n_levels; ++l) {
      const int n = level_start[l + 1] - level_start[l];
      for (int first = 0; first < n; first += 32768) {  // grid.y / grid.z limit
        rc = launch(level_start[l] + first, n - first < 32768 ? n - first : 32768);
        if (rc) return rc;
      }
    }
  }
  if (cfg.flags & PLK_FLAG_CACHE_RATE_PRODUCTS) {  // cache Q p_k while the traversal has p_k at hand
    std::vector<int32_t> dests(count);
    for (int i = 0; i < count; ++i) {
      dests[i] = ops[i].dest;
      in->qp_valid[ops[i].dest] = 0;
    }
    if (in->q_written[0]) return cache_rate_products_impl(in, 0, dests.data(), count);
  }
  return PLK_SUCCESS;
}


// ---- step 4: root ---------------------------------------------------------------------------------------------------

static int root_impl(plk_instance* in, int root, const int32_t* scale_idx, int scale_count, double* d_sum,
                     double* d_site) {
  const Layout& L = in->L;
  const plk_config& cfg = in->cfg;
  if (scale_count < 0 || (scale_count > 0 && scale_idx == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  int rc = check_model_ready(in, false);
  if (rc) return rc;
  const void* rptr;
  const void* pending;
  int kind;
  rc = operand_of(in, root, &rptr, &kind, &pending);
  if (rc) return rc;
  if (kind == KIND_STATES) return PLK_ERR_OUT_OF_RANGE;
  for (int i = 0; i < scale_count; ++i) {
    if (scale_idx[i] < 0 || scale_idx[i] >= cfg.scale_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (!in->scale_written[scale_idx[i]]) return PLK_ERR_UNINITIALIZED;
  }
  // deferred rescaling: the root's own pending factor is not applied to the stored values, so it must not be
  // counted: drop it from the list
  std::vector<const void*> list;
  const int own = in->deferred ? in->post_pending_scale[root] : -1;
  bool own_listed = false;
  for (int i = 0; i < scale_count; ++i) {
    if (scale_idx[i] == own && !own_listed) {
      own_listed = true;
      continue;
    }
    list.push_back(in->scale_ptr(scale_idx[i]));
  }
  if (own >= 0 && !own_listed) return PLK_ERR_UNSUPPORTED;  // would need the factor applied with negative sign
  char *h = nullptr, *d = nullptr;
  if (!list.empty()) {
    rc = ring_alloc(in, list.size() * sizeof(void*), &h, &d);
    if (rc) return rc;
    std::memcpy(h, list.data(), list.size() * sizeof(void*));
    rc = copy_ring(in, h, d, list.size() * sizeof(void*));
    if (rc) return rc;
  }
  const int G = L.SP == 4 ? 1 : L.SP / 4;  // threads per pattern, 4 states each
  const int n_blocks = (int)blocks_for((size_t)L.P * G, 128);
  // one block (a few patterns: the latency-bound end of configs[4], single-pattern large-S problems): its partial sum IS
  // the result, written straight to the output -- one launch less per evaluation
  double* bp = n_blocks == 1 ? d_sum : in->at<double>(L.off_block_partial);
  by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    const T* r = static_cast<const T*>(rptr);
    if (L.SP == 4)
      k_root<T, 4, 1><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, in->at<double>(L.off_pi),
                                                        in->at<double>(L.off_catw),
                                                        reinterpret_cast<const void* const*>(d), (int)list.size(),
                                                        in->at<double>(L.off_weights), d_site, bp);
    else if (L.SP == 32)
      k_root<T, 32, 8><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, in->at<double>(L.off_pi),
                                                         in->at<double>(L.off_catw),
                                                         reinterpret_cast<const void* const*>(d), (int)list.size(),
                                                         in->at<double>(L.off_weights), d_site, bp);
    else
      k_root<T, 64, 16><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, in->at<double>(L.off_pi),
                                                          in->at<double>(L.off_catw),
                                                          reinterpret_cast<const void* const*>(d), (int)list.size(),
                                                          in->at<double>(L.off_weights), d_site, bp);
    return PLK_SUCCESS;
  });
  CHECK_LAUNCH(in);
  if (n_blocks > 1) {
    k_sum_rows<<<1, 128, 0, in->stream>>>(bp, nullptr, n_blocks, n_blocks, d_sum);
    CHECK_LAUNCH(in);
  }
  return PLK_SUCCESS;
}

int plk_root_log_likelihoods_device(plk_instance* in, int root, const int32_t* scale_idx, int scale_count,
                                    double* d_out_sum, double* d_out_site) {
  if (in == nullptr || d_out_sum == nullptr) return PLK_ERR_OUT_OF_RANGE;
  return root_impl(in, root, scale_idx, scale_count, d_out_sum, d_out_site);
}

int plk_root_log_likelihoods(plk_instance* in, int root, const int32_t* scale_idx, int scale_count, double* out_sum,
                             double* out_site) {
  if (in == nullptr || out_sum == nullptr) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  double* d_sum = in->at<double>(L.off_logl);
  double* d_site = in->at<double>(L.off_site);
  int rc = root_impl(in, root, scale_idx, scale_count, d_sum, d_site);
  if (rc) return rc;
  if (out_site != nullptr) CU(cudaMemcpyAsync(out_site, d_site, (size_t)L.P * 8, cudaMemcpyDeviceToHost, in->stream));
  rc = download(in, out_sum, d_sum, 1);
  if (rc) return rc;
  return std::isfinite(*out_sum) ? PLK_SUCCESS : PLK_ERR_FLOATING_POINT;
}

// ---- steps 5-6: pre-order and derivatives --------------------------------------------------------------------------

static int fill_root_pre(plk_instance* in, int root_pre) {
  const Layout& L = in->L;
  if (root_pre < 0 || root_pre >= in->cfg.preorder_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->have_pi) return PLK_ERR_UNINITIALIZED;
  int rc = bind_pre(in, root_pre);
  if (rc) return rc;
  if (in->root_pre_filled != root_pre || !in->pre_written[root_pre]) {
    const size_t n = (size_t)L.C * L.P * L.SP;
    by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      k_fill_root_pre<T><<<blocks_for(n, 256), 256, 0, in->stream>>>(static_cast<T*>(in->pre_ptr(root_pre)),
                                                                     in->at<double>(L.off_pi), n, L.SP);
      return PLK_SUCCESS;
    });
    CHECK_LAUNCH(in);
    in->root_pre_filled = root_pre;
  }
  in->pre_written[root_pre] = 1;
  in->pre_has_mx[root_pre] = 0;
  return PLK_SUCCESS;
}

// Shared by plk_update_pre_partials (want_grad = false) and plk_pre_order_gradient.
static int pre_impl(plk_instance* in, int eigen, int root_pre, const plk_pre_op* ops, int count, bool want_grad,
                    double* d_grad, double* d_site) {
  const Layout& L = in->L;
  const plk_config& cfg = in->cfg;
  if (count < 0) return PLK_ERR_OUT_OF_RANGE;
  if (cfg.preorder_buffer_count == 0) return PLK_ERR_UNSUPPORTED;
  if (want_grad) {
    if (eigen < 0 || eigen >= cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (!in->q_written[eigen]) return PLK_ERR_UNINITIALIZED;
    int rc = check_model_ready(in, true);
    if (rc) return rc;
    if (count > L.max_grad) return PLK_ERR_OUT_OF_RANGE;
  }
  std::vector<int> level, partner;
  const int n_levels = schedule_pre(ops, count, level, partner);
  if (n_levels < 0) return n_levels;
  for (int i = 0; i < count; ++i) {
    const plk_pre_op& o = ops[i];
    if (o.dest_pre >= cfg.preorder_buffer_count || o.parent_pre >= cfg.preorder_buffer_count ||
        o.matrix >= cfg.matrix_buffer_count || o.sibling_matrix >= cfg.matrix_buffer_count ||
        o.sibling_post >= cfg.partials_buffer_count || o.node_post >= cfg.partials_buffer_count || o.node_post < -1)
      return PLK_ERR_OUT_OF_RANGE;
    if (want_grad && o.node_post < 0) return PLK_ERR_OUT_OF_RANGE;
    if (!want_grad && o.dest_pre < 0) return PLK_ERR_OUT_OF_RANGE;
    if (!in->matrix_written[o.matrix] || !in->matrix_written[o.sibling_matrix]) return PLK_ERR_UNINITIALIZED;
  }
  int rc = fill_root_pre(in, root_pre);
  if (rc) return rc;
  {  // parents must be written already or produced earlier in this list; count fresh slots
    std::vector<char> will(cfg.preorder_buffer_count, 0);
    int fresh = 0;
    for (int i = 0; i < count; ++i) {
      const plk_pre_op& o = ops[i];
      if (!(in->pre_written[o.parent_pre] || will[o.parent_pre])) return PLK_ERR_UNINITIALIZED;
      if (o.dest_pre >= 0) {
        if (in->pre_slot[o.dest_pre] < 0 && !will[o.dest_pre]) ++fresh;
        will[o.dest_pre] = 1;
      }
    }
    if (in->next_pre_slot + fresh > L.pre_slots) return PLK_ERR_OUT_OF_MEMORY;
  }
  // build items in list order (bookkeeping), one per pair / unpaired op
  struct HostItem { DevPreItem it; int level; int cls; };  // cls 0..2: plk_nuc_lean.cuh classes; 3: general kernel
  const bool lean = want_grad && (nuc_lean_ok(in) || tc5_classes_ok(in));
  std::vector<HostItem> items;
  items.reserve(count);
  for (int i = 0; i < count; ++i) {
    if (partner[i] >= 0 && partner[i] < i) continue;  // emitted with its partner
    const plk_pre_op& a = ops[i];
    DevPreItem it;
    std::memset(&it, 0, sizeof(it));
    it.qm = in->pre_ptr(a.parent_pre);
    it.qm_scale = (in->deferred && in->pre_has_mx[a.parent_pre]) ? in->pre_mx_ptr(a.parent_pre) : nullptr;
    const plk_pre_op* pair[2] = {&a, partner[i] >= 0 ? &ops[partner[i]] : nullptr};
    const int op_index[2] = {i, partner[i]};
    // operands: child 0 = a's node, child 1 = a's sibling (= partner's node)
    int post_idx[2] = {a.node_post, a.sibling_post};
    if (pair[1] != nullptr) {
      if (post_idx[0] < 0) post_idx[0] = pair[1]->sibling_post;
      if (pair[1]->node_post >= 0 && pair[1]->node_post != a.sibling_post) return PLK_ERR_OUT_OF_RANGE;
      if (a.node_post >= 0 && pair[1]->sibling_post != a.node_post) return PLK_ERR_OUT_OF_RANGE;
    }
    const int mats[2] = {a.matrix, a.sibling_matrix};
    for (int k = 0; k < 2; ++k) {
      it.mat[k] = in->matrix_ptr(mats[k]);
      if (post_idx[k] >= 0) {
        rc = operand_of(in, post_idx[k], &it.p[k], &it.kind[k], &it.p_scale[k]);
        if (rc) return rc;
      } else {
        it.p[k] = nullptr;
        it.kind[k] = KIND_NONE;
        it.p_scale[k] = nullptr;
      }
      it.slot[k] = -1;
      it.q[k] = nullptr;
      it.q_scale[k] = nullptr;
      if (pair[k] != nullptr) {
        if (want_grad) it.slot[k] = op_index[k];
        if (pair[k]->dest_pre >= 0) {
          rc = bind_pre(in, pair[k]->dest_pre);
          if (rc) return rc;
          it.q[k] = in->pre_ptr(pair[k]->dest_pre);
          it.q_scale[k] = in->deferred ? in->pre_mx_ptr(pair[k]->dest_pre) : nullptr;
        }
      }
    }
    int cls = 3;
    if (lean && it.slot[0] >= 0 && it.slot[1] >= 0) {
      auto internal = [&](int k) { return it.kind[k] == KIND_PARTIALS && it.q[k] != nullptr; };
      auto tip = [&](int k) { return it.kind[k] == KIND_STATES && it.q[k] == nullptr; };
      if (tip(0) && internal(1)) {  // the update is symmetric in the two children: internal child first
        std::swap(it.q[0], it.q[1]);
        std::swap(it.q_scale[0], it.q_scale[1]);
        std::swap(it.p[0], it.p[1]);
        std::swap(it.p_scale[0], it.p_scale[1]);
        std::swap(it.mat[0], it.mat[1]);
        std::swap(it.kind[0], it.kind[1]);
        std::swap(it.slot[0], it.slot[1]);
      }
      if (internal(0) && internal(1)) cls = 0;
      else if (internal(0) && tip(1)) cls = 1;
      else if (tip(0) && tip(1)) cls = 2;
    }
    items.push_back({it, level[i], cls});
    // bookkeeping after the item's inputs were resolved
    for (int k = 0; k < 2; ++k)
      if (pair[k] != nullptr && pair[k]->dest_pre >= 0) {
        in->pre_written[pair[k]->dest_pre] = 1;
        in->pre_has_mx[pair[k]->dest_pre] = in->deferred ? 1 : 0;
        if (in->root_pre_filled == pair[k]->dest_pre) in->root_pre_filled = -1;
      }
  }
  const int n_items = (int)items.size();
  // Both-tips items (class 2) read q_parent and write no partials: nothing in the pass depends on them, so all of them
  // run as ONE launch after the last level instead of one small launch per level (a level's few cherries do not fill
  // the GPU: 9 launches of 66 MB at configs[1]).  They are placed in a pseudo-level behind the real ones.  Not done
  // when the list overwrites a buffer that an earlier op reads as its parent (the deferred read would see the new
  // contents).
  int n_lv = n_levels;
  if (lean) {
    bool war = false;
    std::vector<char> read_as_parent(cfg.preorder_buffer_count, 0);
    for (int i = 0; i < count && !war; ++i) {
      if (ops[i].dest_pre >= 0 && read_as_parent[ops[i].dest_pre]) war = true;
      read_as_parent[ops[i].parent_pre] = 1;
    }
    if (!war) {
      bool any = false;
      for (HostItem& hi : items)
        if (hi.cls == 2) {
          hi.level = n_levels;
          any = true;
        }
      if (any) n_lv = n_levels + 1;
    }
  }
  std::vector<int> slot_parts(count > 0 ? count : 0, 0);  // partial sums per gradient slot (0: nothing written)
  if (n_items > 0) {
    std::vector<int> level_start(n_lv + 1, 0);
    for (const HostItem& hi : items) ++level_start[hi.level + 1];
    for (int l = 0; l < n_lv; ++l) level_start[l + 1] += level_start[l];
    std::vector<int> fill(level_start.begin(), level_start.end() - 1);
    char *h, *d;
    rc = ring_alloc(in, (size_t)n_items * sizeof(DevPreItem), &h, &d);
    if (rc) return rc;
    DevPreItem* hit = reinterpret_cast<DevPreItem*>(h);
    const bool walk = L.SP == 4 && nuc_use_walk(in, n_items, n_levels, want_grad);
    std::vector<int> class_start((size_t)n_lv * 5, 0);  // per level: first item of class 0..3, end
    if (walk) {
      for (int i = 0; i < n_items; ++i) hit[i] = items[i].it;  // list order (plk_nuc.cuh "walk")
    } else {  // by level, and inside a level by class
      for (const HostItem& hi : items) ++class_start[(size_t)hi.level * 5 + hi.cls + 1];
      for (int l = 0; l < n_lv; ++l) {
        class_start[(size_t)l * 5] = level_start[l];
        for (int k = 0; k < 4; ++k) class_start[(size_t)l * 5 + k + 1] += class_start[(size_t)l * 5 + k];
      }
      std::vector<int> cfill(class_start);
      for (const HostItem& hi : items) hit[cfill[(size_t)hi.level * 5 + hi.cls]++] = hi.it;
    }
    rc = copy_ring(in, h, d, (size_t)n_items * sizeof(DevPreItem));
    if (rc) return rc;
    const DevPreItem* dit = reinterpret_cast<const DevPreItem*>(d);
    const void* Q = want_grad ? in->eig_QT(eigen) : in->eig_QT(0);
#ifdef PLK_WITH_TENSOR
    std::vector<int> fin_slots;  // gradient slots served by the class-specialised tcgen05 kernels (per-category scratch)
    if (L.SP == 64 && in->f32 && (in->cfg.flags & PLK_FLAG_TENSOR_CORES) && !(in->cfg.flags & PLK_FLAG_NO_TCGEN05)) {
      // step B of the tcgen05 pre-order kernels contracts over the ROW index of M: it reads transposed copies; the
      // class-specialised kernels also read D = M Q and D^T (plk_tc5_pre2.cuh).  Every matrix buffer, once per pass.
      if (want_grad) {
        rc = tc5::pre2::launch_prep(in->stream, in->at<float>(L.off_matrix), static_cast<const float*>(Q),
                                    in->at<float>(L.off_matrix_d), in->at<float>(L.off_matrix_t),
                                    in->at<float>(L.off_matrix_dt), in->cfg.matrix_buffer_count * L.C, &in->launches);
        if (rc) return rc;
      } else {
        tc5::pre::k_transpose64<<<in->cfg.matrix_buffer_count * L.C, 256, 0, in->stream>>>(
            in->at<float>(L.off_matrix), in->at<float>(L.off_matrix_t));
        CHECK_LAUNCH(in);
      }
    }
#endif
    // Every gradient kernel writes its own number of partial sums per slot (tile geometry differs between the
    // class-specialised, the general TMA and the register-staged kernels): remember it per slot for k_sum_rows.
    auto mark_parts = [&](int first, int n) {
      for (int i = first; i < first + n; ++i)
        for (int k = 0; k < 2; ++k)
          if (hit[i].slot[k] >= 0) slot_parts[hit[i].slot[k]] = in->grad_parts;
    };
    if (walk) {
      rc = by_precision(in, [&](auto tag) -> int {
        using T = decltype(tag);
        return nuc_use_tma(in, true) ? launch_pre4_tma<T>(in, dit, n_items, static_cast<const T*>(Q), d_site, true)
                               : launch_pre4_walk<T>(in, dit, n_items, static_cast<const T*>(Q), d_site);
      });
      if (rc) return rc;
      mark_parts(0, n_items);
    }
    if (!walk && L.SP == 4 && class_start[(size_t)(n_lv - 1) * 5 + 3] > 0) {
      // some items run on the class-specialised kernels: their compact-tip children read D = M Q (one 4 x 4 product
      // per matrix and category, every matrix buffer; unwritten buffers give unused garbage)
      rc = by_precision(in, [&](auto tag) -> int {
        using T = decltype(tag);
        const int n_buf = in->cfg.matrix_buffer_count;
        k_deriv_matrices4<T><<<(n_buf * L.C * 16 + 255) / 256, 256, 0, in->stream>>>(
            in->at<T>(L.off_matrix), static_cast<const T*>(Q), in->at<T>(L.off_matrix_d), n_buf, L.C,
            L.matrix_bytes / sizeof(T));
        CHECK_LAUNCH(in);
        return PLK_SUCCESS;
      });
      if (rc) return rc;
    }
    for (int l = 0; l < (walk ? 0 : n_lv); ++l) {
      bool first_launch = true;  // of this level: see launch_pre4_lean_c
      for (int k = 0; k < 3; ++k) {  // specialised classes
        const int c0 = class_start[(size_t)l * 5 + k], m = class_start[(size_t)l * 5 + k + 1] - c0;
        if (m == 0) continue;
#ifdef PLK_WITH_TENSOR
        if (L.SP == 64) {  // tcgen05 classes: results go through the per-category scratch, finished after the last level
          const tc5::pre2::MatDeltas mdl{(long long)L.off_matrix_d - (long long)L.off_matrix,
                                         (long long)L.off_matrix_t - (long long)L.off_matrix,
                                         (long long)L.off_matrix_dt - (long long)L.off_matrix};
          float* scr = in->at<float>(L.off_cat_scratch);
          if (k == 0)
            rc = tc5::pre2::launch_class<0>(in->stream, dit + c0, m, L.P, L.S, L.C, mdl, scr, in->sm_count, &in->launches);
          else if (k == 1)
            rc = tc5::pre2::launch_class<1>(in->stream, dit + c0, m, L.P, L.S, L.C, mdl, scr, in->sm_count, &in->launches);
          else
            rc = tc5::pre2::launch_tips(in->stream, dit + c0, m, L.P, L.S, L.C, mdl, scr, in->sm_count, &in->launches);
          if (rc) return rc;
          for (int i = c0; i < c0 + m; ++i) {
            fin_slots.push_back(hit[i].slot[0]);
            fin_slots.push_back(hit[i].slot[1]);
          }
          continue;
        }
#endif
        rc = by_precision(in, [&](auto tag) -> int {
          using T = decltype(tag);
          return launch_pre4_lean<T>(in, k, dit + c0, m, in->h_q4.data() + (size_t)(want_grad ? eigen : 0) * 16, d_site,
                                     first_launch);
        });
        if (rc) return rc;
        mark_parts(c0, m);
        first_launch = false;
      }
      const int g0 = class_start[(size_t)l * 5 + 3];
      const int n = level_start[l + 1] - g0;
      for (int first = 0; first < n; first += 32768) {
        const int m = n - first < 32768 ? n - first : 32768;
        rc = by_precision(in, [&](auto tag) -> int {
          using T = decltype(tag);
          const DevPreItem* p0 = dit + g0 + first;
          if (L.SP != 4) return launch_pre64<T>(in, p0, m, static_cast<const T*>(Q), d_site);
          return nuc_use_tma(in) ? launch_pre4_tma<T>(in, p0, m, static_cast<const T*>(Q), d_site, false)
                                 : launch_pre4<T>(in, p0, m, static_cast<const T*>(Q), d_site);
        });
        if (rc) return rc;
        mark_parts(g0 + first, m);
      }
    }
#ifdef PLK_WITH_TENSOR
    if (!fin_slots.empty()) {  // d_k[p] = sum_c w_c r_c num / sum_c w_c den and the weighted pattern sums of those slots
      char *hs, *ds;
      rc = ring_alloc(in, fin_slots.size() * sizeof(int), &hs, &ds);
      if (rc) return rc;
      std::memcpy(hs, fin_slots.data(), fin_slots.size() * sizeof(int));
      rc = copy_ring(in, hs, ds, fin_slots.size() * sizeof(int));
      if (rc) return rc;
      int parts = 0;
      rc = tc5::pre2::launch_finish(in->stream, in->at<float>(L.off_cat_scratch), reinterpret_cast<const int*>(ds),
                                    (int)fin_slots.size(), L.P, L.C, in->at<double>(L.off_catw), in->at<double>(L.off_rates),
                                    in->at<double>(L.off_weights), in->at<double>(L.off_grad_partial), L.n_tiles, d_site,
                                    &parts, &in->launches);
      if (rc) return rc;
      for (int sl : fin_slots) slot_parts[sl] = parts;
    }
#endif
  }
  if (want_grad && count > 0) {
    char *h, *d;
    rc = ring_alloc(in, (size_t)count * sizeof(int), &h, &d);
    if (rc) return rc;
    std::memcpy(h, slot_parts.data(), (size_t)count * sizeof(int));
    rc = copy_ring(in, h, d, (size_t)count * sizeof(int));
    if (rc) return rc;
    k_sum_rows<<<count, 128, 0, in->stream>>>(in->at<double>(L.off_grad_partial), reinterpret_cast<const int*>(d), 0,
                                              L.n_tiles, d_grad);
    CHECK_LAUNCH(in);
  }
  return PLK_SUCCESS;
}

int plk_update_pre_partials(plk_instance* in, int root_pre, const plk_pre_op* ops, int count) {
  if (in == nullptr) return PLK_ERR_OUT_OF_RANGE;
  return pre_impl(in, 0, root_pre, ops, count, false, nullptr, nullptr);
}

int plk_pre_order_gradient_device(plk_instance* in, int eigen, int root_pre, const plk_pre_op* ops, int count,
                                  double* d_out_gradient, double* d_out_site) {
  if (in == nullptr || (count > 0 && d_out_gradient == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  return pre_impl(in, eigen, root_pre, ops, count, true, d_out_gradient, d_out_site);
}

static int finish_gradient(plk_instance* in, int count, double* out_gradient, double* out_site, double* d_site) {
  const Layout& L = in->L;
  if (count == 0) return PLK_SUCCESS;
  if (out_site != nullptr)
    CU(cudaMemcpyAsync(out_site, d_site, (size_t)count * L.P * 8, cudaMemcpyDeviceToHost, in->stream));
  int rc = download(in, out_gradient, in->at<double>(L.off_grad_out), count);
  if (rc) return rc;
  for (int i = 0; i < count; ++i)
    if (!std::isfinite(out_gradient[i])) return PLK_ERR_FLOATING_POINT;
  return PLK_SUCCESS;
}

int plk_pre_order_gradient(plk_instance* in, int eigen, int root_pre, const plk_pre_op* ops, int count,
                           double* out_gradient, double* out_site) {
  if (in == nullptr || (count > 0 && out_gradient == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  if (out_site != nullptr && !(in->cfg.flags & PLK_FLAG_SITE_DERIVATIVES)) return PLK_ERR_UNSUPPORTED;
  double* d_site = out_site != nullptr ? in->at<double>(L.off_site_deriv) : nullptr;
  int rc = pre_impl(in, eigen, root_pre, ops, count, true, in->at<double>(L.off_grad_out), d_site);
  if (rc) return rc;
  return finish_gradient(in, count, out_gradient, out_site, d_site);
}

// P:101 variant (a), gradient side: the sandwich from the cached Q p_k (k_deriv*_cached) -- no matrix is applied.
static int branch_derivatives_cached(plk_instance* in, int eigen, const int32_t* post_idx, const int32_t* pre_idx,
                                     int count, double* out_gradient, double* out_site) {
  const Layout& L = in->L;
  const plk_config& cfg = in->cfg;
  char *h, *d;
  int rc = ring_alloc(in, (size_t)count * sizeof(DevBranchQp), &h, &d);
  if (rc) return rc;
  DevBranchQp* hb = reinterpret_cast<DevBranchQp*>(h);
  for (int i = 0; i < count; ++i) {
    if (pre_idx[i] < 0 || pre_idx[i] >= cfg.preorder_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (in->pre_slot[pre_idx[i]] < 0 || !in->pre_written[pre_idx[i]]) return PLK_ERR_UNINITIALIZED;
    const void* pending;
    rc = operand_of(in, post_idx[i], &hb[i].p, &hb[i].kind, &pending);
    if (rc) return rc;
    if (hb[i].kind != KIND_STATES && !in->qp_valid[post_idx[i]]) return PLK_ERR_UNINITIALIZED;  // plk_cache_rate_products first
    hb[i].qp = hb[i].kind == KIND_STATES ? nullptr : in->qp_ptr(post_idx[i]);
    hb[i].q = in->pre_ptr(pre_idx[i]);
    hb[i].slot = i;
  }
  rc = copy_ring(in, h, d, (size_t)count * sizeof(DevBranchQp));
  if (rc) return rc;
  double* d_site = out_site != nullptr ? in->at<double>(L.off_site_deriv) : nullptr;
  const DevBranchQp* db = reinterpret_cast<const DevBranchQp*>(d);
  const double* cw = in->at<double>(L.off_catw);
  const double* cr = in->at<double>(L.off_rates);
  const double* wt = in->at<double>(L.off_weights);
  double* gp = in->at<double>(L.off_grad_partial);
  for (int first = 0; first < count; first += 32768) {
    const int m = count - first < 32768 ? count - first : 32768;
    rc = by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      const T* Q = static_cast<const T*>(in->eig_QT(eigen));
      if (L.SP == 4) {
        dim3 grid(blocks_for(L.P, NUC_THREADS), m);
        switch (L.C) {
#define CASE(CC) case CC: k_deriv4_cached<T, CC><<<grid, NUC_THREADS, 0, in->stream>>>(db + first, L.P, Q, cw, cr, wt, gp, L.n_tiles, d_site); break;
          CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
          default: return PLK_ERR_UNSUPPORTED;
        }
        in->grad_parts = (int)grid.x;
      } else {
        dim3 grid(L.n_tiles, m);
        if (L.SP == 32)
          k_deriv64_cached<T, 32><<<grid, GEN_THREADS, 0, in->stream>>>(db + first, L.P, L.S, L.C, Q, cw, cr, wt, gp, L.n_tiles, d_site);
        else
          k_deriv64_cached<T, 64><<<grid, GEN_THREADS, 0, in->stream>>>(db + first, L.P, L.S, L.C, Q, cw, cr, wt, gp, L.n_tiles, d_site);
        in->grad_parts = L.n_tiles;
      }
      return PLK_SUCCESS;
    });
    if (rc) return rc;
    CHECK_LAUNCH(in);
  }
  k_sum_rows<<<count, 128, 0, in->stream>>>(gp, nullptr, in->grad_parts, L.n_tiles, in->at<double>(L.off_grad_out));
  CHECK_LAUNCH(in);
  return finish_gradient(in, count, out_gradient, out_site, d_site);
}

int plk_cache_rate_products(plk_instance* in, int eigen, const int32_t* post_idx, int count) {
  if (in == nullptr) return PLK_ERR_OUT_OF_RANGE;
  return cache_rate_products_impl(in, eigen, post_idx, count);
}

// P:101 variant (b): the whole post-order list in one launch, transition matrices applied on the fly (k_post_otf).
int plk_update_partials_on_the_fly(plk_instance* in, int eigen, const plk_op* ops, int count, const double* branch_lengths) {
  if (in == nullptr || count < 0) return PLK_ERR_OUT_OF_RANGE;
  const plk_config& cfg = in->cfg;
  const Layout& L = in->L;
  if (!(cfg.flags & PLK_FLAG_ON_THE_FLY_MATRICES)) return PLK_ERR_UNSUPPORTED;
  if (count == 0) return PLK_SUCCESS;
  if (ops == nullptr || branch_lengths == nullptr || count > cfg.partials_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (eigen < 0 || eigen >= cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->eigen_written[eigen] || !in->have_rates) return PLK_ERR_UNINITIALIZED;
  std::vector<int> level;
  const int n_levels = schedule_post(ops, count, level);
  if (n_levels < 0) return n_levels;
  std::vector<int> producer(cfg.partials_buffer_count, -1);
  int fresh = 0;
  for (int i = 0; i < count; ++i) {
    const plk_op& o = ops[i];
    if (o.dest >= cfg.partials_buffer_count || o.child1 >= cfg.partials_buffer_count || o.child2 >= cfg.partials_buffer_count ||
        o.dest_scale >= cfg.scale_buffer_count || o.dest_scale < -1)
      return PLK_ERR_OUT_OF_RANGE;
    if (in->post_slot[o.dest] >= 0 && in->post_kind[o.dest] == KIND_STATES) return PLK_ERR_OUT_OF_RANGE;
    for (int k = 0; k < 2; ++k) {
      const double t = branch_lengths[2 * i + k];
      if (!(t >= 0.0 && std::isfinite(t))) return PLK_ERR_OUT_OF_RANGE;
      const int ch = k == 0 ? o.child1 : o.child2;
      if (!(in->post_written[ch] || producer[ch] >= 0)) return PLK_ERR_UNINITIALIZED;
    }
    if (in->post_slot[o.dest] < 0 && producer[o.dest] < 0) ++fresh;
    producer[o.dest] = i;
  }
  if (in->next_post_slot + fresh > L.post_slots) return PLK_ERR_OUT_OF_MEMORY;
  char *h, *d;
  int rc = ring_alloc(in, (size_t)count * sizeof(DevOtfOp), &h, &d);
  if (rc) return rc;
  DevOtfOp* ho = reinterpret_cast<DevOtfOp*>(h);
  std::fill(producer.begin(), producer.end(), -1);
  for (int i = 0; i < count; ++i) {  // list order: every dependency has a lower index
    const plk_op& o = ops[i];
    rc = bind_post_full(in, o.dest, KIND_PARTIALS);
    if (rc) return rc;
    DevOtfOp& x = ho[i];
    x.dest = in->post_ptr(o.dest);
    x.scale = o.dest_scale >= 0 ? in->scale_ptr(o.dest_scale) : nullptr;
    const int ch[2] = {o.child1, o.child2};
    for (int k = 0; k < 2; ++k) {
      rc = operand_of(in, ch[k], &x.child[k], &x.kind[k], &x.cscale[k]);
      if (rc) return rc;
      x.t[k] = branch_lengths[2 * i + k];
      x.dep[k] = producer[ch[k]];
    }
    producer[o.dest] = i;
    in->post_written[o.dest] = 1;
    in->qp_valid[o.dest] = 0;
    in->post_pending_scale[o.dest] = o.dest_scale;
    if (o.dest_scale >= 0) in->scale_written[o.dest_scale] = 1;
  }
  rc = copy_ring(in, h, d, (size_t)count * sizeof(DevOtfOp));
  if (rc) return rc;
  if (++in->otf_epoch == 0) {  // wrapped: clear the flags so that an old value cannot match
    CU(cudaMemsetAsync(in->arena + L.off_otf_ready, 0, (size_t)cfg.partials_buffer_count * L.P * 4, in->stream));
    in->otf_epoch = 1;
  }
  const long long total = (long long)count * L.P;
  rc = by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    auto go = [&](auto kernel, size_t smem) -> int {
      int r2 = opt_in_smem(kernel, smem);
      if (r2) return r2;
      int bps = 0;
      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, OTF_THREADS, smem));
      if (bps < 1) return PLK_ERR_CUDA;
      long long g = (long long)in->sm_count * bps;
      if (g > total) g = total;
      kernel<<<(unsigned)g, OTF_THREADS, smem, in->stream>>>(
          reinterpret_cast<const DevOtfOp*>(d), count, L.P, L.S, L.C, in->eig_U(eigen), in->eig_Uinv(eigen),
          in->eig_lam(eigen), in->at<double>(L.off_rates), in->at<OtfSync>(L.off_otf_sync),
          in->at<unsigned int>(L.off_otf_ready), in->otf_epoch);
      return PLK_SUCCESS;
    };
    return L.SP == 32 ? go(k_post_otf<T, 32>, otf_smem<32>()) : go(k_post_otf<T, 64>, otf_smem<64>());
  });
  if (rc) return rc;
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}

int plk_branch_derivatives(plk_instance* in, int eigen, const int32_t* post_idx, const int32_t* pre_idx, int count,
                           double* out_gradient, double* out_site) {
  if (in == nullptr || count < 0) return PLK_ERR_OUT_OF_RANGE;
  if (count == 0) return PLK_SUCCESS;
  if (post_idx == nullptr || pre_idx == nullptr || out_gradient == nullptr) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  const plk_config& cfg = in->cfg;
  if (cfg.preorder_buffer_count == 0) return PLK_ERR_UNSUPPORTED;
  if (out_site != nullptr && !(cfg.flags & PLK_FLAG_SITE_DERIVATIVES)) return PLK_ERR_UNSUPPORTED;
  if (eigen < 0 || eigen >= cfg.eigen_buffer_count || count > L.max_grad) return PLK_ERR_OUT_OF_RANGE;
  if (!in->q_written[eigen]) return PLK_ERR_UNINITIALIZED;
  int rc = check_model_ready(in, true);
  if (rc) return rc;
  if (cfg.flags & PLK_FLAG_CACHE_RATE_PRODUCTS)
    return branch_derivatives_cached(in, eigen, post_idx, pre_idx, count, out_gradient, out_site);
  char *h, *d;
  rc = ring_alloc(in, (size_t)count * sizeof(DevBranch), &h, &d);
  if (rc) return rc;
  DevBranch* hb = reinterpret_cast<DevBranch*>(h);
  for (int i = 0; i < count; ++i) {
    if (pre_idx[i] < 0 || pre_idx[i] >= cfg.preorder_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (in->pre_slot[pre_idx[i]] < 0 || !in->pre_written[pre_idx[i]]) return PLK_ERR_UNINITIALIZED;
    const void* pending;
    rc = operand_of(in, post_idx[i], &hb[i].p, &hb[i].kind, &pending);
    if (rc) return rc;
    hb[i].q = in->pre_ptr(pre_idx[i]);
    hb[i].slot = i;
  }
  rc = copy_ring(in, h, d, (size_t)count * sizeof(DevBranch));
  if (rc) return rc;
  double* d_site = out_site != nullptr ? in->at<double>(L.off_site_deriv) : nullptr;
  const DevBranch* db = reinterpret_cast<const DevBranch*>(d);
  for (int first = 0; first < count; first += 32768) {
    const int m = count - first < 32768 ? count - first : 32768;
    rc = by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      const T* Q = static_cast<const T*>(in->eig_QT(eigen));
      return L.SP == 4 ? launch_deriv4<T>(in, db + first, m, Q, d_site) : launch_deriv64<T>(in, db + first, m, Q, d_site);
    });
    if (rc) return rc;
  }
  k_sum_rows<<<count, 128, 0, in->stream>>>(in->at<double>(L.off_grad_partial), nullptr, in->grad_parts, L.n_tiles,
                                            in->at<double>(L.off_grad_out));
  CHECK_LAUNCH(in);
  return finish_gradient(in, count, out_gradient, out_site, d_site);
}

// ---- steps 1-6 in one call, replayed from a cached CUDA graph ---------------------------------------------------------
// Small problems (configs[0], the low end of configs[4]) are bound by launch latency, not by the GPU: an evaluation is
// 10-20 dependent launches plus their descriptor uploads (SURVEY section 7 hard part 7).  plk_evaluate_device runs the
// four steps through the very same code as the separate calls, but from its third use with an unchanged signature it
// replays them as ONE cudaGraphLaunch: the first use runs eagerly (it binds slots and sets kernel attributes), the
// second use is run once more under stream capture with the launch descriptors placed in a region of the arena that
// belongs to the graph (uploaded once, after the capture), and every later use is the instantiated graph.

namespace {

uint64_t fnv1a(uint64_t h, const void* data, size_t bytes) {
  const unsigned char* p = static_cast<const unsigned char*>(data);
  for (size_t i = 0; i < bytes; ++i) h = (h ^ p[i]) * 1099511628211ull;
  return h;
}

struct EvalArgs {
  int eigen;
  const int32_t* matrix_idx;
  const double* d_t;
  int matrix_count;
  const plk_op* ops;
  int op_count;
  int root;
  const int32_t* scale_idx;
  int scale_count;
  int root_pre;
  const plk_pre_op* pre_ops;
  int pre_count;
  double* d_out;
};

int evaluate_steps(plk_instance* in, const EvalArgs& a) {
  int rc = update_matrices_impl(in, a.eigen, a.matrix_idx, nullptr, a.d_t, a.matrix_count);
  if (rc) return rc;
  rc = plk_update_partials(in, a.ops, a.op_count);
  if (rc) return rc;
  rc = root_impl(in, a.root, a.scale_idx, a.scale_count, a.d_out, nullptr);
  if (rc) return rc;
  return pre_impl(in, a.eigen, a.root_pre, a.pre_ops, a.pre_count, true, a.d_out + 1, nullptr);
}

void drop_plans(plk_instance* in) {
  cudaStreamSynchronize(in->stream);  // a graph still in flight reads its descriptor block
  for (auto& pl : in->plans)
    if (pl.exec != nullptr) cudaGraphExecDestroy(pl.exec);
  in->plans.clear();
  in->plan_pos = 0;
}

int evaluate_impl(plk_instance* in, const EvalArgs& a) {
  if (a.matrix_count < 0 || a.op_count < 0 || a.scale_count < 0 || a.pre_count < 0) return PLK_ERR_OUT_OF_RANGE;
  if ((a.matrix_count > 0 && (a.matrix_idx == nullptr || a.d_t == nullptr)) || (a.op_count > 0 && a.ops == nullptr) ||
      (a.scale_count > 0 && a.scale_idx == nullptr) || (a.pre_count > 0 && a.pre_ops == nullptr) || a.d_out == nullptr)
    return PLK_ERR_OUT_OF_RANGE;
  uint64_t key = 1469598103934665603ull;
  const int head[8] = {a.eigen, a.matrix_count, a.op_count, a.root, a.scale_count, a.root_pre, a.pre_count,
                       in->root_pre_filled == a.root_pre ? 1 : 0};
  key = fnv1a(key, head, sizeof(head));
  key = fnv1a(key, a.matrix_idx, (size_t)a.matrix_count * 4);
  key = fnv1a(key, a.ops, (size_t)a.op_count * sizeof(plk_op));
  key = fnv1a(key, a.scale_idx, (size_t)a.scale_count * 4);
  key = fnv1a(key, a.pre_ops, (size_t)a.pre_count * sizeof(plk_pre_op));
  const uint64_t tail[4] = {(uint64_t)(uintptr_t)a.d_t, (uint64_t)(uintptr_t)a.d_out, in->model_epoch, in->binding_epoch};
  key = fnv1a(key, tail, sizeof(tail));
  plk_instance::EvalPlan* pl = nullptr;
  for (auto& q : in->plans)
    if (q.key == key) pl = &q;
  if (pl != nullptr && pl->exec != nullptr) {  // replay
    CU(cudaGraphLaunch(pl->exec, in->stream));
    in->launches += pl->launches;
    ++pl->uses;
    return PLK_SUCCESS;
  }
  if (pl == nullptr) {  // first use: eager
    if ((int)in->plans.size() >= PLAN_MAX) drop_plans(in);
    in->plans.emplace_back();
    in->plans.back().key = key;
    in->plans.back().uses = 1;
    return evaluate_steps(in, a);
  }
  ++pl->uses;
  if (pl->failed) return evaluate_steps(in, a);
  // second use: the same steps under stream capture, descriptors in the plan region
  if (in->plan_host.empty()) in->plan_host.assign(PLAN_BYTES, 0);
  const size_t plan_from = in->plan_pos;
  const int64_t launches_before = in->launches;
  if (cudaStreamBeginCapture(in->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
    cudaGetLastError();  // e.g. the legacy default stream cannot be captured
    pl->failed = true;
    return evaluate_steps(in, a);
  }
  in->planning = true;
  const int rc = evaluate_steps(in, a);
  in->planning = false;
  cudaGraph_t graph = nullptr;
  const cudaError_t ce = cudaStreamEndCapture(in->stream, &graph);
  const int64_t captured = in->launches - launches_before;
  in->launches = launches_before;
  cudaGraphExec_t exec = nullptr;
  if (rc == PLK_SUCCESS && ce == cudaSuccess && graph != nullptr &&
      cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess) {
    cudaGraphDestroy(graph);
    // the descriptor block, once; stream order puts it before the first replay
    if (in->plan_pos > plan_from)
      CU(cudaMemcpyAsync(in->arena + in->L.off_plan + plan_from, in->plan_host.data() + plan_from, in->plan_pos - plan_from,
                         cudaMemcpyHostToDevice, in->stream));
    pl->exec = exec;
    pl->launches = captured;
    CU(cudaGraphLaunch(exec, in->stream));
    in->launches += captured;
    return PLK_SUCCESS;
  }
  if (graph != nullptr) cudaGraphDestroy(graph);
  cudaGetLastError();
  in->plan_pos = plan_from;
  pl->failed = true;
  if (rc != PLK_SUCCESS && rc != PLK_ERR_OUT_OF_MEMORY) return rc;  // a genuine argument error
  return evaluate_steps(in, a);
}

}  // namespace

int plk_evaluate_device(plk_instance* in, int eigen, const int32_t* matrix_idx, const double* d_branch_lengths,
                        int matrix_count, const plk_op* ops, int op_count, int root_buffer, const int32_t* scale_idx,
                        int scale_count, int root_pre_buffer, const plk_pre_op* pre_ops, int pre_count, double* d_out) {
  if (in == nullptr) return PLK_ERR_OUT_OF_RANGE;
  const EvalArgs a{eigen, matrix_idx, d_branch_lengths, matrix_count, ops, op_count, root_buffer, scale_idx, scale_count,
                   root_pre_buffer, pre_ops, pre_count, d_out};
  return evaluate_impl(in, a);
}

int plk_evaluate(plk_instance* in, int eigen, const int32_t* matrix_idx, const double* branch_lengths, int matrix_count,
                 const plk_op* ops, int op_count, int root_buffer, const int32_t* scale_idx, int scale_count,
                 int root_pre_buffer, const plk_pre_op* pre_ops, int pre_count, double* out_logl, double* out_gradient) {
  if (in == nullptr || out_logl == nullptr || (pre_count > 0 && out_gradient == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  if (matrix_count < 0 || matrix_count > in->cfg.matrix_buffer_count || pre_count < 0 || pre_count > in->L.max_grad)
    return PLK_ERR_OUT_OF_RANGE;
  if (matrix_count > 0 && branch_lengths == nullptr) return PLK_ERR_OUT_OF_RANGE;
  for (int i = 0; i < matrix_count; ++i)
    if (!(branch_lengths[i] >= 0.0 && std::isfinite(branch_lengths[i]))) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  double* d_t = in->at<double>(L.off_eval_t);
  double* d_out = in->at<double>(L.off_eval_out);
  if (matrix_count > 0)
    CU(cudaMemcpyAsync(d_t, branch_lengths, (size_t)matrix_count * 8, cudaMemcpyHostToDevice, in->stream));
  const EvalArgs a{eigen, matrix_idx, d_t, matrix_count, ops, op_count, root_buffer, scale_idx, scale_count,
                   root_pre_buffer, pre_ops, pre_count, d_out};
  int rc = evaluate_impl(in, a);
  if (rc) return rc;
  std::vector<double> tmp(1 + (size_t)pre_count);
  rc = download(in, tmp.data(), d_out, tmp.size());
  if (rc) return rc;
  *out_logl = tmp[0];
  bool finite = std::isfinite(tmp[0]);
  for (int i = 0; i < pre_count; ++i) {
    out_gradient[i] = tmp[1 + i];
    finite = finite && std::isfinite(tmp[1 + i]);
  }
  return finite ? PLK_SUCCESS : PLK_ERR_FLOATING_POINT;
}

// ---- 8(f)-1: approximate gradient with respect to the rate-matrix elements --------------------------------------------

int plk_rate_matrix_gradient(plk_instance* in, const int32_t* post_idx, const int32_t* pre_idx,
                             const double* branch_lengths, int count, double* out_G) {
  if (in == nullptr || count < 0 || out_G == nullptr) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  const plk_config& cfg = in->cfg;
  if (cfg.preorder_buffer_count == 0) return PLK_ERR_UNSUPPORTED;
  if (count > 0 && (post_idx == nullptr || pre_idx == nullptr || branch_lengths == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  int rc = check_model_ready(in, true);
  if (rc) return rc;
  const int n_elem = L.SP * L.SP;
  double* d_out = in->at<double>(L.off_cross_out);
  if (count == 0) {
    for (int i = 0; i < L.S * L.S; ++i) out_G[i] = 0.0;
    return PLK_SUCCESS;
  }
  char *h, *d;
  rc = ring_alloc(in, (size_t)count * sizeof(DevCrossBranch), &h, &d);
  if (rc) return rc;
  DevCrossBranch* hb = reinterpret_cast<DevCrossBranch*>(h);
  for (int i = 0; i < count; ++i) {
    if (pre_idx[i] < 0 || pre_idx[i] >= cfg.preorder_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (in->pre_slot[pre_idx[i]] < 0 || !in->pre_written[pre_idx[i]]) return PLK_ERR_UNINITIALIZED;
    if (!(branch_lengths[i] >= 0.0 && std::isfinite(branch_lengths[i]))) return PLK_ERR_OUT_OF_RANGE;
    const void* pending;
    rc = operand_of(in, post_idx[i], &hb[i].p, &hb[i].kind, &pending);
    if (rc) return rc;
    hb[i].q = in->pre_ptr(pre_idx[i]);
    hb[i].t = branch_lengths[i];
    hb[i].pad = 0;
  }
  rc = copy_ring(in, h, d, (size_t)count * sizeof(DevCrossBranch));
  if (rc) return rc;
  const DevCrossBranch* db = reinterpret_cast<const DevCrossBranch*>(d);
  const double* cw = in->at<double>(L.off_catw);
  const double* cr = in->at<double>(L.off_rates);
  const double* wt = in->at<double>(L.off_weights);
  double* part = in->at<double>(L.off_cross_partial);
  if (L.SP == 4) {
    const int n_pblocks = (L.P + CROSS4_THREADS - 1) / CROSS4_THREADS;
    // branch ranges: enough blocks for ~64 warps per SM, at most CROSS4_SPLITS (the layout's bound) and one branch each
    int splits = 1;
    while (splits < CROSS4_SPLITS && splits * 2 <= count && (long long)n_pblocks * splits * (CROSS4_THREADS / 32) < 64LL * in->sm_count)
      splits *= 2;
    const int n_blocks = n_pblocks * splits;
    const dim3 grid4(n_pblocks, splits);
    rc = by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      switch (L.C) {
#define CASE(CC) case CC: k_cross4<T, CC><<<grid4, CROSS4_THREADS, 0, in->stream>>>(db, count, L.P, cw, cr, wt, part, n_blocks); break;
        CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
        default: return PLK_ERR_UNSUPPORTED;
      }
      return PLK_SUCCESS;
    });
    if (rc) return rc;
    CHECK_LAUNCH(in);
    k_sum_rows<<<16, 128, 0, in->stream>>>(part, nullptr, n_blocks, n_blocks, d_out);
    CHECK_LAUNCH(in);
  } else {
    const int n_blocks = (L.P + CROSS64_TP - 1) / CROSS64_TP;
    int n_sum = n_blocks;  // partial sums to add up
    rc = by_precision(in, [&](auto tag) -> int {
      using T = decltype(tag);
      if (L.SP == 32) {
        int r3 = opt_in_smem(k_cross64<T, 32>, cross64_smem<T, 32>());
        if (r3) return r3;
        k_cross64<T, 32><<<n_blocks, CROSS64_THREADS, cross64_smem<T, 32>(), in->stream>>>(db, count, L.P, L.S, L.C, cw, cr, wt, part);
        return PLK_SUCCESS;
      }
      if (cfg.flags & PLK_FLAG_TENSOR_CORES) {
        // tensor cores (plk_cross_tc.cuh): units = pattern tiles x branch ranges, dealt round-robin to a fixed grid
        const size_t smem = cross_tc_smem<T>(L.C);
        if (smem + 1024 > 232448) return PLK_ERR_UNSUPPORTED;
        auto kern = L.C == 4 ? k_cross_tc<T, 4> : k_cross_tc<T, 0>;
        int r4 = opt_in_smem(kern, smem);
        if (r4) return r4;
        const int per_sm = std::min(3, (int)(233472 / (smem + 1024)));
        const int slots = std::min(CROSS_TC_MAX_GRID, in->sm_count * per_sm);
        const int chunks = (L.P + CrossTc<T>::TP - 1) / CrossTc<T>::TP;
        const int n_split = std::max(1, std::min(count, (8 * slots + chunks - 1) / chunks));
        const long long units = (long long)chunks * n_split;
        n_sum = (int)std::min<long long>(units, slots);
        kern<<<n_sum, CROSS_TC_THREADS, smem, in->stream>>>(db, count, n_split, (int)units, L.P, L.S, L.C, cw, cr, wt, part);
        return PLK_SUCCESS;
      }
      int r2 = opt_in_smem(k_cross64<T>, cross64_smem<T>());
      if (r2) return r2;
      k_cross64<T><<<n_blocks, CROSS64_THREADS, cross64_smem<T>(), in->stream>>>(db, count, L.P, L.S, L.C, cw, cr, wt, part);
      return PLK_SUCCESS;
    });
    if (rc) return rc;
    CHECK_LAUNCH(in);
    k_sum_blocks<<<(n_elem + 255) / 256, 256, 0, in->stream>>>(part, n_sum, n_elem, d_out);
    CHECK_LAUNCH(in);
  }
  std::vector<double> tmp(n_elem);
  rc = download(in, tmp.data(), d_out, n_elem);
  if (rc) return rc;
  for (int i = 0; i < L.S; ++i)
    for (int j = 0; j < L.S; ++j) {
      out_G[i * L.S + j] = tmp[i * L.SP + j];
      if (!std::isfinite(out_G[i * L.S + j])) rc = PLK_ERR_FLOATING_POINT;
    }
  return rc;
}

int plk_chain_rule_rate_matrix(const double* G, const double* dQ, int state_count, int param_count, double* out) {
  if (G == nullptr || out == nullptr || state_count < 1 || param_count < 0 || (param_count > 0 && dQ == nullptr))
    return PLK_ERR_OUT_OF_RANGE;
  const size_t n = (size_t)state_count * state_count;
  for (int k = 0; k < param_count; ++k) {
    double s = 0.0;
    for (size_t e = 0; e < n; ++e) s += G[e] * dQ[(size_t)k * n + e];
    out[k] = s;
  }
  return PLK_SUCCESS;
}

// ---- read-back -------------------------------------------------------------------------------------------------------

int plk_get_partials(plk_instance* in, int buffer, int pre, double* out) {
  if (in == nullptr || out == nullptr) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  const size_t rows = (size_t)L.C * L.P;
  double* stage = in->at<double>(L.off_stage);
  const void* src;
  int kind = KIND_PARTIALS;
  if (pre == 2) {  // the cached rate product Q p_k of a post-order buffer (PLK_FLAG_CACHE_RATE_PRODUCTS)
    if (!(in->cfg.flags & PLK_FLAG_CACHE_RATE_PRODUCTS)) return PLK_ERR_UNSUPPORTED;
    const void* pending;
    int rc = operand_of(in, buffer, &src, &kind, &pending);
    if (rc) return rc;
    if (kind == KIND_STATES) return PLK_ERR_UNSUPPORTED;
    if (!in->qp_valid[buffer]) return PLK_ERR_UNINITIALIZED;
    src = in->qp_ptr(buffer);
  } else if (pre) {
    if (buffer < 0 || buffer >= in->cfg.preorder_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (in->pre_slot[buffer] < 0 || !in->pre_written[buffer]) return PLK_ERR_UNINITIALIZED;
    src = in->pre_ptr(buffer);
  } else {
    const void* pending;
    int rc = operand_of(in, buffer, &src, &kind, &pending);
    if (rc) return rc;
  }
  if (kind == KIND_STATES) {
    k_expand_states<<<blocks_for(rows * L.S, 256), 256, 0, in->stream>>>(static_cast<const uint8_t*>(src), stage, L.C,
                                                                        L.P, L.S);
    CHECK_LAUNCH(in);
  } else {
    const int reps = kind == KIND_BCAST ? L.C : 1;
    const size_t n_rows = kind == KIND_BCAST ? (size_t)L.P : rows;
    for (int r = 0; r < reps; ++r) {
      by_precision(in, [&](auto tag) -> int {
        using T = decltype(tag);
        k_unpad_rows<T><<<blocks_for(n_rows * L.S, 256), 256, 0, in->stream>>>(
            static_cast<const T*>(src), stage + (size_t)r * L.P * L.S, n_rows, L.S, L.SP);
        return PLK_SUCCESS;
      });
      CHECK_LAUNCH(in);
    }
  }
  return download(in, out, stage, rows * L.S);
}

int plk_get_scale_factors(plk_instance* in, int scale, double* out) {
  if (in == nullptr || out == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (scale < 0 || scale >= in->cfg.scale_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->scale_written[scale]) return PLK_ERR_UNINITIALIZED;
  const Layout& L = in->L;
  double* stage = in->at<double>(L.off_stage);
  by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    k_scale_logs<T><<<blocks_for(L.P, 256), 256, 0, in->stream>>>(in->scale_ptr(scale), stage, L.P, L.C,
                                                                  in->deferred ? 1 : 0);
    return PLK_SUCCESS;
  });
  CHECK_LAUNCH(in);
  return download(in, out, stage, L.P);
}

int plk_get_transition_matrix(plk_instance* in, int matrix, double* out) {
  if (in == nullptr || out == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (matrix < 0 || matrix >= in->cfg.matrix_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->matrix_written[matrix]) return PLK_ERR_UNINITIALIZED;
  const Layout& L = in->L;
  double* stage = in->at<double>(L.off_stage);
  by_precision(in, [&](auto tag) -> int {
    using T = decltype(tag);
    k_unpad_matrices<T><<<blocks_for((size_t)L.C * L.S * L.S, 256), 256, 0, in->stream>>>(
        static_cast<const T*>(in->matrix_ptr(matrix)), stage, L.C, L.S, L.SP);
    return PLK_SUCCESS;
  });
  CHECK_LAUNCH(in);
  return download(in, out, stage, (size_t)L.C * L.S * L.S);
}

int plk_get_rate_matrix(plk_instance* in, int eigen, double* out) {
  if (in == nullptr || out == nullptr) return PLK_ERR_OUT_OF_RANGE;
  if (eigen < 0 || eigen >= in->cfg.eigen_buffer_count) return PLK_ERR_OUT_OF_RANGE;
  if (!in->q_written[eigen]) return PLK_ERR_UNINITIALIZED;
  return download(in, out, in->eig_Q64(eigen), (size_t)in->L.S * in->L.S);
}

int plk_synchronize(plk_instance* in) {
  if (in == nullptr) return PLK_ERR_OUT_OF_RANGE;
  CU(cudaStreamSynchronize(in->stream));
  return PLK_SUCCESS;
}

int64_t plk_kernel_launch_count(const plk_instance* in) { return in == nullptr ? 0 : in->launches; }

// ---- host-only helpers -------------------------------------------------------------------------------------------------

int plk_schedule_levels(const plk_op* ops, int count, int32_t* out_level) {
  std::vector<int> level;
  const int n = schedule_post(ops, count, level);
  if (n >= 0 && out_level != nullptr)
    for (int i = 0; i < count; ++i) out_level[i] = level[i];
  return n;
}

int plk_schedule_pre_levels(const plk_pre_op* ops, int count, int32_t* out_level, int32_t* out_partner) {
  std::vector<int> level, partner;
  const int n = schedule_pre(ops, count, level, partner);
  if (n >= 0)
    for (int i = 0; i < count; ++i) {
      if (out_level != nullptr) out_level[i] = level[i];
      if (out_partner != nullptr) out_partner[i] = partner[i];
    }
  return n;
}

}  // extern "C"

// =================================================================================================================
// plk_root_log_likelihoods_static_device -- the root reduction (S8a step 4) for callers that must not allocate.
//
// Same kernels and arithmetic as plk_root_log_likelihoods_device; the one difference is where k_root's per-block
// partial sums go: not into the instance arena but into the file-scope array below, which every GPU that loads the
// library holds until the process exits (PLK_STATIC_SCRATCH_DOUBLES doubles = 64 KB).  The call allocates nothing on
// the device or on the host (no cudaMalloc / cudaFree, no allocating library routine, no std::vector): the scale list
// is assembled on the stack and travels through the instance's pinned parameter ring, which plk_create made.
// Limits (else PLK_ERR_STATIC_SCRATCH_LIMIT): k_root blocks = ceil(P * G / 128) <= PLK_STATIC_SCRATCH_DOUBLES (G = 1
// for 4 states, 8 for 5..32, 16 for 33..64: P <= 1 048 576 / 131 072 / 65 536) and scale_count <=
// PLK_STATIC_SCALE_MAX.  The array is shared by EVERY call on a device -- all instances, all streams -- and keeps the
// last call's contents: nothing in it has to start at zero (k_root writes each of the n_blocks entries k_sum_rows
// reads, in the same call), but two calls that overlap on the GPU (different streams, or graphs replayed concurrently)
// race on it and must be serialised by the caller.
// =================================================================================================================
static __device__ __align__(256) double g_plk_static_scratch[PLK_STATIC_SCRATCH_DOUBLES];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
double* g_static_scratch_ptr[STATIC_MAX_DEVICES] = {};  // device address of the array on each device (set once)

// In host code `g_plk_static_scratch` is a host-side stand-in, not a device address: resolve it once per device, with
// that device current, and hand the result to the kernels.
int static_scratch_address(int device, double** out) {
  if (device < 0 || device >= STATIC_MAX_DEVICES) return PLK_ERR_CUDA;
  if (g_static_scratch_ptr[device] == nullptr) {
    int current = -1;
    if (cudaGetDevice(&current) != cudaSuccess || current != device) return PLK_ERR_CUDA;
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_plk_static_scratch) != cudaSuccess || p == nullptr) return PLK_ERR_CUDA;
    g_static_scratch_ptr[device] = static_cast<double*>(p);
  }
  *out = g_static_scratch_ptr[device];
  return PLK_SUCCESS;
}
}  // namespace

extern "C" int plk_root_log_likelihoods_static_device(plk_instance* in, int root, const int32_t* scale_idx, int scale_count,
                                                      double* d_out_sum, double* d_out_site) {
  if (in == nullptr || d_out_sum == nullptr) return PLK_ERR_OUT_OF_RANGE;
  const Layout& L = in->L;
  const plk_config& cfg = in->cfg;
  if (scale_count < 0 || (scale_count > 0 && scale_idx == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  const int G = L.SP == 4 ? 1 : L.SP / 4;  // threads per pattern, 4 states each (as in root_impl)
  const size_t n_blocks_sz = ((size_t)L.P * G + 127) / 128;
  if (n_blocks_sz > (size_t)PLK_STATIC_SCRATCH_DOUBLES || scale_count > PLK_STATIC_SCALE_MAX)
    return PLK_ERR_STATIC_SCRATCH_LIMIT;
  const int n_blocks = (int)n_blocks_sz;
  int rc = check_model_ready(in, false);
  if (rc) return rc;
  const void* rptr;
  const void* pending;
  int kind;
  rc = operand_of(in, root, &rptr, &kind, &pending);
  if (rc) return rc;
  if (kind == KIND_STATES) return PLK_ERR_OUT_OF_RANGE;
  for (int i = 0; i < scale_count; ++i) {
    if (scale_idx[i] < 0 || scale_idx[i] >= cfg.scale_buffer_count) return PLK_ERR_OUT_OF_RANGE;
    if (!in->scale_written[scale_idx[i]]) return PLK_ERR_UNINITIALIZED;
  }
  // the arena's device must be the current one (the binding keeps it current around every call)
  cudaPointerAttributes pa;
  if (cudaPointerGetAttributes(&pa, in->arena) != cudaSuccess) return PLK_ERR_CUDA;
  double* bp = nullptr;
  rc = static_scratch_address(pa.device, &bp);
  if (rc) return rc;
  // deferred rescaling: the root's own pending factor is not applied to the stored values: drop it from the list
  const void* list[PLK_STATIC_SCALE_MAX];
  int n_list = 0;
  const int own = in->deferred ? in->post_pending_scale[root] : -1;
  bool own_listed = false;
  for (int i = 0; i < scale_count; ++i) {
    if (scale_idx[i] == own && !own_listed) {
      own_listed = true;
      continue;
    }
    list[n_list++] = in->scale_ptr(scale_idx[i]);
  }
  if (own >= 0 && !own_listed) return PLK_ERR_UNSUPPORTED;
  char *h = nullptr, *d = nullptr;
  if (n_list > 0) {
    rc = ring_alloc(in, (size_t)n_list * sizeof(void*), &h, &d);
    if (rc) return rc;
    std::memcpy(h, list, (size_t)n_list * sizeof(void*));
    rc = copy_ring(in, h, d, (size_t)n_list * sizeof(void*));
    if (rc) return rc;
  }
  const double* pi = in->at<double>(L.off_pi);
  const double* cw = in->at<double>(L.off_catw);
  const double* wt = in->at<double>(L.off_weights);
  const void* const* dl = reinterpret_cast<const void* const*>(d);
  if (in->f32) {
    const float* r = static_cast<const float*>(rptr);
    if (L.SP == 4) k_root<float, 4, 1><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, pi, cw, dl, n_list, wt, d_out_site, bp);
    else if (L.SP == 32) k_root<float, 32, 8><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, pi, cw, dl, n_list, wt, d_out_site, bp);
    else k_root<float, 64, 16><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, pi, cw, dl, n_list, wt, d_out_site, bp);
  } else {
    const double* r = static_cast<const double*>(rptr);
    if (L.SP == 4) k_root<double, 4, 1><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, pi, cw, dl, n_list, wt, d_out_site, bp);
    else if (L.SP == 32) k_root<double, 32, 8><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, pi, cw, dl, n_list, wt, d_out_site, bp);
    else k_root<double, 64, 16><<<n_blocks, 128, 0, in->stream>>>(r, kind, L.P, L.C, pi, cw, dl, n_list, wt, d_out_site, bp);
  }
  CHECK_LAUNCH(in);
  k_sum_rows<<<1, 128, 0, in->stream>>>(bp, nullptr, n_blocks, n_blocks, d_out_sum);
  CHECK_LAUNCH(in);
  return PLK_SUCCESS;
}
