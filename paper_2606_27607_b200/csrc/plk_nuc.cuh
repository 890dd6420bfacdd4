// plk_nuc.cuh -- 4-state (nucleotide) kernels: HBM-bandwidth-bound streaming kernels (~1-2 flop/B).
//
// Thread mapping.  A warp owns a "chunk" of PPW = 32 / LP consecutive patterns; LP lanes share one pattern and
// split its C rate categories (C = 4: LP = 4, one category per lane; lane = g * PPW + pl with g the category group
// and pl the pattern within the chunk).  A lane therefore holds only 4 states of ONE category in registers -- the
// occupancy that a one-thread-per-pattern kernel loses to its C x 4 x (2 children) live values is what kept the
// first version of the pre-order kernel at 18 % of peak warps (profiles/r01_nuc_fp64_baseline.md).  The per-pattern
// maximum (rescaling) and the category sums of the gradient are LP-lane xor-shuffles.
// Layout [c][p][s]: the PPW lanes of one category read PPW * 4 * sizeof(T) contiguous bytes (256 B fp64, 128 B
// fp32 at C = 4): whole 32-byte sectors, whole 128-byte lines.
//
// Two launch shapes share the per-chunk bodies post4_cell / pre4_cell:
//   level   (k_post4 / k_pre4)            blockIdx.y = operation of a dependency level, blockIdx.x = 4 chunks; one
//                                         launch per level.  Parallel over nodes x patterns: the shape for small P.
//   walk    (k_post4_walk / k_pre4_walk)  ONE launch for the whole operation list: a warp owns its chunks for the
//                                         whole traversal and walks the list in the client's (depth-first) order.
//                                         Patterns are independent ("conditionally independent"), and
//                                         cell (p, c) of every buffer is only ever touched by the lane that owns
//                                         (p, c), so program order is the only dependency: no grid barrier, no
//                                         level launches, and a parent reads the child it has just written from
//                                         L2 instead of HBM.  The grid is sized to ONE resident wave in which every
//                                         warp has the same number of chunks (no tail).
// Transition matrices of the current operation sit in shared memory, one padded slab per category (stride
// NucMat<T>::STRIDE) so that the LP distinct 16-byte addresses of one warp-wide read fall into distinct banks: one
// wavefront per read.  (Reading them through L1 instead costs one wavefront per distinct line and kept the L1 pipe
// 74 % busy: profiles/r01_nuc_walk_v1.md.)  The walk kernels stage the matrices and the descriptor of operation
// i + 1 while operation i is computed (double buffer, one __syncthreads per operation).
#pragma once
#include "plk_common.cuh"

namespace plk {

constexpr int NUC_THREADS = 128;
constexpr int NUC_WARPS = NUC_THREADS / 32;

template <int C>
struct NucMap {
  static constexpr int LP = (C % 4 == 0) ? 4 : (C % 2 == 0) ? 2 : 1;  // lanes per pattern
  static constexpr int CPT = C / LP;                                   // categories per lane
  static constexpr int PPW = 32 / LP;                                  // patterns per warp chunk
};

// shared-memory slab of one 4 x 4 matrix: 16 values + padding to the next 16-byte-bank group
template <typename T>
struct NucMat {
  static constexpr int STRIDE = 16 + 16 / (int)sizeof(T);  // fp64: 18 doubles (144 B); fp32: 20 floats (80 B)
};

// a[s] = sum_x M[s][x] v[x]
template <typename T>
__device__ __forceinline__ void mv4(const T* __restrict__ M, const T v[4], T a[4]) {
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    T r[4];
    ld4(M + 4 * s, r);
    a[s] = r[0] * v[0] + r[1] * v[1] + r[2] * v[2] + r[3] * v[3];
  }
}
// a[s] = sum_x M[x][s] v[x]
template <typename T>
__device__ __forceinline__ void mvt4(const T* __restrict__ M, const T v[4], T a[4]) {
  T r[4];
  ld4(M, r);
#pragma unroll
  for (int s = 0; s < 4; ++s) a[s] = r[s] * v[0];
#pragma unroll
  for (int x = 1; x < 4; ++x) {
    ld4(M + 4 * x, r);
#pragma unroll
    for (int s = 0; s < 4; ++s) a[s] = fma(r[s], v[x], a[s]);
  }
}

// the operand vector x of (child, category c, pattern p): partials, broadcast partials, or one-hot / all-ones.
// Plain (coherent) loads: in the walk kernels a buffer may have been written earlier by this very lane.
template <typename T>
__device__ __forceinline__ void operand4(int kind, const void* ptr, int c, int p, int P, T x[4]) {
  if (kind == KIND_PARTIALS) {
    ldg4c(static_cast<const T*>(ptr) + ((size_t)c * P + p) * 4, x);
  } else if (kind == KIND_BCAST) {
    ldg4c(static_cast<const T*>(ptr) + (size_t)p * 4, x);
  } else if (kind == KIND_STATES) {
    const int z = static_cast<const uint8_t*>(ptr)[p];
#pragma unroll
    for (int s = 0; s < 4; ++s) x[s] = (z >= 4 || z == s) ? T(1) : T(0);
  } else {
#pragma unroll
    for (int s = 0; s < 4; ++s) x[s] = T(0);
  }
}

// a = M . x for one child; compact states read a column of M (or 1 for a missing state)
template <typename T>
__device__ __forceinline__ void contrib4(int kind, const void* ptr, const T* __restrict__ M, int c, int p, int P, T a[4]) {
  if (kind == KIND_STATES) {
    const int z = static_cast<const uint8_t*>(ptr)[p];
#pragma unroll
    for (int s = 0; s < 4; ++s) a[s] = z < 4 ? M[s * 4 + z] : T(1);
  } else {
    T x[4];
    operand4<T>(kind, ptr, c, p, P, x);
    mv4<T>(M, x, a);
  }
}

template <typename T, int LP>
__device__ __forceinline__ T group_max(T v) {
#pragma unroll
  for (int o = 32 / LP; o < 32; o <<= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
template <int LP>
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
  for (int o = 32 / LP; o < 32; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// sum over the PPW pattern lanes of category group 0 (values of the other groups must be 0); result in lane 0
template <int LP>
__device__ __forceinline__ double chunk_sum(double v) {
#pragma unroll
  for (int o = 16 / LP; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

// ---------------------------------------------------------------------------------------------------------------
// staging of one operation's matrices: dst[k][c * STRIDE + e] <- mat_k[c * 16 + e]  (k = 0, 1; all threads)
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C>
struct NucStage {
  static constexpr int N = 2 * C * 16;                                  // values per operation
  static constexpr int PER = (N + NUC_THREADS - 1) / NUC_THREADS;      // values per thread
  T v[PER];
  __device__ __forceinline__ void load(const void* m0, const void* m1) {
#pragma unroll
    for (int j = 0; j < PER; ++j) {
      const int idx = threadIdx.x + j * NUC_THREADS;
      if (idx < N) v[j] = __ldg(static_cast<const T*>(idx < C * 16 ? m0 : m1) + (idx % (C * 16)));
    }
  }
  __device__ __forceinline__ void store(T* dst /* [2][C * STRIDE] */) const {
#pragma unroll
    for (int j = 0; j < PER; ++j) {
      const int idx = threadIdx.x + j * NUC_THREADS;
      if (idx < N) {
        const int k = idx / (C * 16), r = idx % (C * 16);
        dst[k * C * NucMat<T>::STRIDE + (r / 16) * NucMat<T>::STRIDE + (r % 16)] = v[j];
      }
    }
  }
};

// ---------------------------------------------------------------------------------------------------------------
// post-order update + immediate per-pattern rescaling of one chunk
// sM: this operation's matrices in shared memory, [2][C * STRIDE]
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C>
__device__ __forceinline__ void post4_cell(const DevOp& op, const T* __restrict__ sM, int P, int p, int g) {
  using Mp = NucMap<C>;
  constexpr int MS = NucMat<T>::STRIDE;
  const bool live = p < P;
  T r[Mp::CPT][4];
  T mx = T(0);
  if (live) {
#pragma unroll
    for (int i = 0; i < Mp::CPT; ++i) {
      const int c = g * Mp::CPT + i;
      T a[4], b[4];
      contrib4<T>(op.kind[0], op.child[0], sM + c * MS, c, p, P, a);
      contrib4<T>(op.kind[1], op.child[1], sM + (C + c) * MS, c, p, P, b);
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        r[i][s] = a[s] * b[s];
        mx = fmax(mx, r[i][s]);
      }
    }
  }
  if (op.scale != nullptr) {
    mx = group_max<T, Mp::LP>(mx);
    const int e = exp_of(mx);
    if (e != 0) {
      const Pow2Pair<T> f = pow2_pair(-e, T(0));
#pragma unroll
      for (int i = 0; i < Mp::CPT; ++i)
#pragma unroll
        for (int s = 0; s < 4; ++s) r[i][s] = (r[i][s] * f.f1) * f.f2;
    }
    if (live && g == 0) static_cast<int16_t*>(op.scale)[p] = (int16_t)e;
  }
  if (live) {
    T* dest = static_cast<T*>(op.dest);
#pragma unroll
    for (int i = 0; i < Mp::CPT; ++i) stg4c(dest + ((size_t)(g * Mp::CPT + i) * P + p) * 4, r[i]);
  }
}

// U chunks at once (the walk kernels, fp32): the operand loads of all U patterns are issued before any arithmetic, and
// a matrix row read from shared memory serves all U of them -- fewer instructions per byte, which is what bounds the
// 4-byte kernels (same instruction count per cell as fp64 for half the bytes).
template <typename T, int U>
__device__ __forceinline__ void contrib4_multi(int kind, const void* ptr, const T* __restrict__ M, int c, const int (&p)[U],
                                               int P, T (&a)[U][4]) {
  if (kind == KIND_STATES) {
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int z = p[u] < P ? static_cast<const uint8_t*>(ptr)[p[u]] : 4;
#pragma unroll
      for (int s = 0; s < 4; ++s) a[u][s] = z < 4 ? M[s * 4 + z] : T(1);
    }
  } else {
    T x[U][4];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (p[u] < P) {
        operand4<T>(kind, ptr, c, p[u], P, x[u]);
      } else {
#pragma unroll
        for (int s = 0; s < 4; ++s) x[u][s] = T(0);
      }
    }
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      T r[4];
      ld4(M + 4 * s, r);
#pragma unroll
      for (int u = 0; u < U; ++u) a[u][s] = r[0] * x[u][0] + r[1] * x[u][1] + r[2] * x[u][2] + r[3] * x[u][3];
    }
  }
}
template <typename T, int C, int U>
__device__ __forceinline__ void post4_cells(const DevOp& op, const T* __restrict__ sM, int P, const int (&p)[U], int g) {
  using Mp = NucMap<C>;
  constexpr int MS = NucMat<T>::STRIDE;
  T r[U][Mp::CPT][4];
  T mx[U];
#pragma unroll
  for (int u = 0; u < U; ++u) mx[u] = T(0);
#pragma unroll
  for (int i = 0; i < Mp::CPT; ++i) {
    const int c = g * Mp::CPT + i;
    T a[U][4], b[U][4];
    contrib4_multi<T, U>(op.kind[0], op.child[0], sM + c * MS, c, p, P, a);
    contrib4_multi<T, U>(op.kind[1], op.child[1], sM + (C + c) * MS, c, p, P, b);
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        r[u][i][s] = p[u] < P ? a[u][s] * b[u][s] : T(0);
        mx[u] = fmax(mx[u], r[u][i][s]);
      }
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const bool live = p[u] < P;
    if (op.scale != nullptr) {
      const int e = exp_of(group_max<T, Mp::LP>(mx[u]));
      if (e != 0) {
        const Pow2Pair<T> f = pow2_pair(-e, T(0));
#pragma unroll
        for (int i = 0; i < Mp::CPT; ++i)
#pragma unroll
          for (int s = 0; s < 4; ++s) r[u][i][s] = (r[u][i][s] * f.f1) * f.f2;
      }
      if (live && g == 0) static_cast<int16_t*>(op.scale)[p[u]] = (int16_t)e;
    }
    if (live) {
      T* dest = static_cast<T*>(op.dest);
#pragma unroll
      for (int i = 0; i < Mp::CPT; ++i) st4(dest + ((size_t)(g * Mp::CPT + i) * P + p[u]) * 4, r[u][i]);
    }
  }
}

template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_post4(const DevOp* __restrict__ ops, int P) {
  using Mp = NucMap<C>;
  __shared__ __align__(16) T sM[2 * C * NucMat<T>::STRIDE];
  const DevOp op = ops[blockIdx.y];
  NucStage<T, C> st;
  st.load(op.mat[0], op.mat[1]);
  st.store(sM);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int chunk = blockIdx.x * NUC_WARPS + (threadIdx.x >> 5);
  post4_cell<T, C>(op, sM, P, chunk * Mp::PPW + lane % Mp::PPW, lane / Mp::PPW);
}

template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_post4_walk(const DevOp* __restrict__ ops, int n_ops, int P,
                                                            int n_chunks, int total_warps) {
  using Mp = NucMap<C>;
  constexpr int SLAB = 2 * C * NucMat<T>::STRIDE;
  __shared__ __align__(16) T sM[2][SLAB];
  __shared__ DevOp sOp[2];
  const int lane = threadIdx.x & 31;
  const int g = lane / Mp::PPW, pl = lane % Mp::PPW;
  const int warp = blockIdx.x * NUC_WARPS + (threadIdx.x >> 5);
  constexpr int OP_WORDS = (int)(sizeof(DevOp) / 4);
  NucStage<T, C> st;
  uint32_t opw = 0;
  if (n_ops > 0) {
    st.load(ops[0].mat[0], ops[0].mat[1]);
    if (threadIdx.x < OP_WORDS) opw = reinterpret_cast<const uint32_t*>(ops)[threadIdx.x];
    st.store(sM[0]);
    if (threadIdx.x < OP_WORDS) reinterpret_cast<uint32_t*>(&sOp[0])[threadIdx.x] = opw;
  }
  __syncthreads();
  for (int i = 0; i < n_ops; ++i) {
    const int cur = i & 1;
    if (i + 1 < n_ops) {  // operation i + 1 -> registers while operation i is computed
      st.load(ops[i + 1].mat[0], ops[i + 1].mat[1]);
      if (threadIdx.x < OP_WORDS) opw = reinterpret_cast<const uint32_t*>(ops + i + 1)[threadIdx.x];
    }
    const DevOp op = sOp[cur];
    int chunk = warp < total_warps ? warp : n_chunks;
    if (sizeof(T) == 4) {  // three / two chunks per pass (see post4_cells)
      for (; chunk + 2 * total_warps < n_chunks; chunk += 3 * total_warps) {
        const int pp[3] = {chunk * Mp::PPW + pl, (chunk + total_warps) * Mp::PPW + pl, (chunk + 2 * total_warps) * Mp::PPW + pl};
        post4_cells<T, C, 3>(op, sM[cur], P, pp, g);
      }
      for (; chunk + total_warps < n_chunks; chunk += 2 * total_warps) {
        const int pp[2] = {chunk * Mp::PPW + pl, (chunk + total_warps) * Mp::PPW + pl};
        post4_cells<T, C, 2>(op, sM[cur], P, pp, g);
      }
    }
    for (; chunk < n_chunks; chunk += total_warps) post4_cell<T, C>(op, sM[cur], P, chunk * Mp::PPW + pl, g);
    if (i + 1 < n_ops) {
      st.store(sM[cur ^ 1]);
      if (threadIdx.x < OP_WORDS) reinterpret_cast<uint32_t*>(&sOp[cur ^ 1])[threadIdx.x] = opw;
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------------------------
// root: site log-likelihoods + weighted block partial sums; works for any padded state count
//   G = threads per pattern (1 for SP = 4, 16 for SP = 64); each thread reads SP / G contiguous states.
// scale list: S = 4 -> int16 [P] exponents; SP = 64 -> T [C][P] maxima whose per-pattern exponent is recomputed.
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int SP, int G>
__global__ void __launch_bounds__(128) k_root(const T* __restrict__ root, int kind, int P, int C,
                                              const double* __restrict__ pi, const double* __restrict__ catw,
                                              const void* const* __restrict__ scales, int n_scales,
                                              const double* __restrict__ weights, double* __restrict__ site,
                                              double* __restrict__ block_partial) {
  constexpr int PER = SP / G;  // states per thread
  __shared__ double red[4];
  const int g = threadIdx.x % G;
  const int p = (blockIdx.x * 128 + threadIdx.x) / G;
  double term = 0.0;
  double lik = 0.0;
  if (p < P) {
    for (int c = 0; c < C; ++c) {
      const T* src = kind == KIND_BCAST ? root + (size_t)p * SP : root + ((size_t)c * P + p) * SP;
      double acc = 0.0;
#pragma unroll
      for (int i = 0; i < PER; i += 4) {
        T v[4];
        ld4(src + g * PER + i, v);
#pragma unroll
        for (int j = 0; j < 4; ++j) acc += pi[g * PER + i + j] * (double)v[j];
      }
      lik += catw[c] * acc;
    }
  }
  // the scale buffers of a pattern are shared out over its G lanes (configs[3]: 255 buffers x 4 categories per pattern)
  int esum = 0;
  if (p < P) {
    for (int k = g; k < n_scales; k += G) {
      if (SP == 4) {
        esum += static_cast<const int16_t*>(scales[k])[p];
      } else {
        const T* mxs = static_cast<const T*>(scales[k]);
        T m = T(0);
        for (int c = 0; c < C; ++c) m = fmax(m, mxs[(size_t)c * P + p]);
        esum += exp_of(m);
      }
    }
  }
#pragma unroll
  for (int o = G / 2; o > 0; o >>= 1) {
    lik += __shfl_xor_sync(0xffffffffu, lik, o);
    esum += __shfl_xor_sync(0xffffffffu, esum, o);
  }
  if (p < P) {
    if (g == 0) {
      const double ll = log(lik) + 0.6931471805599453094 * (double)esum;
      if (site != nullptr) site[p] = ll;
      term = weights[p] * ll;
    }
  }
  const double s = block_sum(term, red);
  if (threadIdx.x == 0) block_partial[blockIdx.x] = s;
}

// out[slot] = sum_i partial[slot][i] in a fixed order (deterministic: SURVEY section 7 hard part 8)
// n_per_row[r] (or n when n_per_row == NULL) = how many partial sums the kernel that served row r has written.
__global__ void __launch_bounds__(128) k_sum_rows(const double* __restrict__ partial, const int* __restrict__ n_per_row,
                                                  int n, int stride, double* __restrict__ out) {
  __shared__ double red[4];
  const double* row = partial + (size_t)blockIdx.x * stride;
  if (n_per_row != nullptr) n = n_per_row[blockIdx.x];
  double v = 0.0;
  for (int i = threadIdx.x; i < n; i += 128) v += row[i];
  const double s = block_sum(v, red);
  if (threadIdx.x == 0) out[blockIdx.x] = s;
}

// ---------------------------------------------------------------------------------------------------------------
// pre-order update of both children of one parent, fused with both branch derivatives, one chunk
// (SURVEY 8(a) steps 5-6).  d[k] = omega_p * num_p / den_p of child k on the lanes of category
// group 0, 0 elsewhere.  sM: the matrices of the two branches [2][C * STRIDE]; sQ: the rate matrix [16].
// den is the same for both children: q_k^T x_k = (q_m o a_{1-k})^T M_k x_k = sum_s q_m[s] a_0[s] a_1[s].
// ---------------------------------------------------------------------------------------------------------------
struct NucModel {
  const double* catw;
  const double* catr;
  const double* weights;
  double* site_out;  // [slots][P] or NULL
};

template <typename T, int C>
__device__ __forceinline__ void pre4_cell(const DevPreItem& it, const T* __restrict__ sM, const T* __restrict__ sQ,
                                          int P, int p, int g, const NucModel& md, double d[2]) {
  using Mp = NucMap<C>;
  constexpr int MS = NucMat<T>::STRIDE;
  const bool live = p < P;
  const bool want_grad = it.slot[0] >= 0 || it.slot[1] >= 0;
  T q[2][Mp::CPT][4];
  T mxq[2] = {T(0), T(0)};
  double num[2] = {0.0, 0.0}, den = 0.0;
  if (live) {
#pragma unroll
    for (int i = 0; i < Mp::CPT; ++i) {
      const int c = g * Mp::CPT + i;
      T qm[4], x[2][4], a[2][4];
      ld4(static_cast<const T*>(it.qm) + ((size_t)c * P + p) * 4, qm);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        operand4<T>(it.kind[k], it.p[k], c, p, P, x[k]);
        mv4<T>(sM + (k * C + c) * MS, x[k], a[k]);
      }
      const double cw = __ldg(md.catw + c), cwr = cw * __ldg(md.catr + c);
      if (want_grad) {
        T dd = T(0);
#pragma unroll
        for (int s = 0; s < 4; ++s) dd += qm[s] * (a[0][s] * a[1][s]);
        den += cw * (double)dd;
      }
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        T u[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) u[s] = qm[s] * a[1 - k][s];
        mvt4<T>(sM + (k * C + c) * MS, u, q[k][i]);
#pragma unroll
        for (int s = 0; s < 4; ++s) mxq[k] = fmax(mxq[k], q[k][i][s]);
        if (it.slot[k] >= 0) {
          T qx[4];
          mv4<T>(sQ, x[k], qx);
          T n = T(0);
#pragma unroll
          for (int s = 0; s < 4; ++s) n += q[k][i][s] * qx[s];
          num[k] += cwr * (double)n;
        }
      }
    }
  }
  if (want_grad) den = group_sum<Mp::LP>(den);
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    d[k] = 0.0;
    if (it.q[k] != nullptr) {  // uniform over the grid
      const int e = exp_of(group_max<T, Mp::LP>(mxq[k]));
      if (live) {
        const Pow2Pair<T> f = pow2_pair(-e, T(0));
        T* dst = static_cast<T*>(it.q[k]);
#pragma unroll
        for (int i = 0; i < Mp::CPT; ++i) {
          T v[4];
#pragma unroll
          for (int s = 0; s < 4; ++s) v[s] = (q[k][i][s] * f.f1) * f.f2;
          st4(dst + ((size_t)(g * Mp::CPT + i) * P + p) * 4, v);
        }
      }
    }
    if (it.slot[k] >= 0) {
      const double nn = group_sum<Mp::LP>(num[k]);
      if (live && g == 0) {
        const double r = nn / den;
        if (md.site_out != nullptr) md.site_out[(size_t)it.slot[k] * P + p] = r;
        d[k] = md.weights[p] * r;
      }
    }
  }
}

// level shape: blockIdx.y = item, blockIdx.x = 4 chunks; grad_partial[slot][blockIdx.x], row stride n_part
template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS, sizeof(T) == 8 ? 4 : 6) k_pre4(const DevPreItem* __restrict__ items, int P,
                                                      const T* __restrict__ Qg, NucModel md,
                                                      double* __restrict__ grad_partial, int n_part) {
  using Mp = NucMap<C>;
  __shared__ __align__(16) T sM[2 * C * NucMat<T>::STRIDE];
  __shared__ __align__(16) T sQ[16];
  __shared__ double red[2][NUC_WARPS];
  const DevPreItem it = items[blockIdx.y];
  NucStage<T, C> st;
  st.load(it.mat[0], it.mat[1]);
  st.store(sM);
  if (threadIdx.x < 16) sQ[threadIdx.x] = Qg[threadIdx.x];
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int chunk = blockIdx.x * NUC_WARPS + warp;
  double d[2];
  pre4_cell<T, C>(it, sM, sQ, P, chunk * Mp::PPW + lane % Mp::PPW, lane / Mp::PPW, md, d);
  if (it.slot[0] < 0 && it.slot[1] < 0) return;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const double s = chunk_sum<Mp::LP>(d[k]);
    if (lane == 0) red[k][warp] = s;
  }
  __syncthreads();
  if (threadIdx.x < 2) {
    const int slot = threadIdx.x == 0 ? it.slot[0] : it.slot[1];
    if (slot >= 0) {
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < NUC_WARPS; ++w) s += red[threadIdx.x][w];
      grad_partial[(size_t)slot * n_part + blockIdx.x] = s;
    }
  }
}

// walk shape: one launch for all items; grad_partial[slot][warp], row stride n_part
template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS, sizeof(T) == 8 ? 4 : 6) k_pre4_walk(const DevPreItem* __restrict__ items, int n_items, int P,
                                                           int n_chunks, int total_warps, const T* __restrict__ Qg,
                                                           NucModel md, double* __restrict__ grad_partial,
                                                           int n_part) {
  using Mp = NucMap<C>;
  constexpr int SLAB = 2 * C * NucMat<T>::STRIDE;
  __shared__ __align__(16) T sM[2][SLAB];
  __shared__ __align__(16) T sQ[16];
  __shared__ DevPreItem sIt[2];
  const int lane = threadIdx.x & 31;
  const int g = lane / Mp::PPW, pl = lane % Mp::PPW;
  const int warp = blockIdx.x * NUC_WARPS + (threadIdx.x >> 5);
  constexpr int IT_WORDS = (int)(sizeof(DevPreItem) / 4);
  static_assert(IT_WORDS <= NUC_THREADS, "descriptor staging uses one word per thread");
  NucStage<T, C> st;
  uint32_t itw = 0;
  if (threadIdx.x < 16) sQ[threadIdx.x] = Qg[threadIdx.x];
  if (n_items > 0) {
    st.load(items[0].mat[0], items[0].mat[1]);
    if (threadIdx.x < IT_WORDS) itw = reinterpret_cast<const uint32_t*>(items)[threadIdx.x];
    st.store(sM[0]);
    if (threadIdx.x < IT_WORDS) reinterpret_cast<uint32_t*>(&sIt[0])[threadIdx.x] = itw;
  }
  __syncthreads();
  for (int i = 0; i < n_items; ++i) {
    const int cur = i & 1;
    if (i + 1 < n_items) {  // item i + 1 -> registers while item i is computed
      st.load(items[i + 1].mat[0], items[i + 1].mat[1]);
      if (threadIdx.x < IT_WORDS) itw = reinterpret_cast<const uint32_t*>(items + i + 1)[threadIdx.x];
    }
    const DevPreItem& it = sIt[cur];
    double acc[2] = {0.0, 0.0};
    for (int chunk = warp < total_warps ? warp : n_chunks; chunk < n_chunks; chunk += total_warps) {
      double d[2];
      pre4_cell<T, C>(it, sM[cur], sQ, P, chunk * Mp::PPW + pl, g, md, d);
      acc[0] += d[0];
      acc[1] += d[1];
    }
    if (warp < total_warps) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (it.slot[k] < 0) continue;
        const double s = chunk_sum<Mp::LP>(acc[k]);
        if (lane == 0) grad_partial[(size_t)it.slot[k] * n_part + warp] = s;
      }
    }
    if (i + 1 < n_items) {
      st.store(sM[cur ^ 1]);
      if (threadIdx.x < IT_WORDS) reinterpret_cast<uint32_t*>(&sIt[cur ^ 1])[threadIdx.x] = itw;
    }
    __syncthreads();
  }
}

// root pre-order partials: q_root[c][p][.] = pi
template <typename T>
__global__ void k_fill_root_pre(T* __restrict__ q, const double* __restrict__ pi, size_t n, int SP) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) q[i] = (T)pi[i % SP];
}

// ---------------------------------------------------------------------------------------------------------------
// unfused branch derivatives from stored pre- and post-order partials; one thread per pattern
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_deriv4(const DevBranch* __restrict__ br, int P,
                                                        const T* __restrict__ Qg, const double* __restrict__ catw,
                                                        const double* __restrict__ catr,
                                                        const double* __restrict__ weights,
                                                        double* __restrict__ grad_partial, int n_tiles,
                                                        double* __restrict__ site_out) {
  const DevBranch b = br[blockIdx.y];
  __shared__ double red[NUC_THREADS / 32];
  const int p = blockIdx.x * NUC_THREADS + threadIdx.x;
  double d = 0.0;
  if (p < P) {
    double num = 0.0, den = 0.0;
#pragma unroll
    for (int c = 0; c < C; ++c) {
      T q[4], x[4], qx[4];
      ld4(static_cast<const T*>(b.q) + ((size_t)c * P + p) * 4, q);
      operand4<T>(b.kind, b.p, c, p, P, x);
      mv4<T>(Qg, x, qx);
      T n = T(0), dd = T(0);
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        n += q[s] * qx[s];
        dd += q[s] * x[s];
      }
      num += catw[c] * catr[c] * (double)n;
      den += catw[c] * (double)dd;
    }
    const double r = num / den;
    if (site_out != nullptr) site_out[(size_t)b.slot * P + p] = r;
    d = weights[p] * r;
  }
  const double s = block_sum(d, red);
  if (threadIdx.x == 0) grad_partial[(size_t)b.slot * n_tiles + blockIdx.x] = s;
}

}  // namespace plk
