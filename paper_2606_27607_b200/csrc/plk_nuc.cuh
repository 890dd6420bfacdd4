// plk_nuc.cuh -- 4-state (nucleotide) kernels: HBM-bandwidth-bound streaming kernels (~1-2 flop/B).
//
// One thread owns one pattern and all C categories of it, so the per-pattern maximum (rescaling, SURVEY 8(a)
// step 3) and the category sums (root, gradient) never leave registers.  Layout [c][p][s]: thread p reads
// 4*sizeof(T) contiguous bytes per category, a warp reads 32 * 4 * sizeof(T) contiguous bytes (1 KB fp64, 512 B
// fp32) per category -- fully coalesced, C independent streams per operand.  Transition matrices of the operation
// sit in shared memory (broadcast reads).  blockIdx.y = operation of the level, blockIdx.x = pattern tile.
#pragma once
#include "plk_common.cuh"

namespace plk {

constexpr int NUC_THREADS = 128;

// a[s] = sum_x M[s][x] v[x]
template <typename T>
__device__ __forceinline__ void mv4(const T* __restrict__ M, const T v[4], T a[4]) {
#pragma unroll
  for (int s = 0; s < 4; ++s) a[s] = M[s * 4 + 0] * v[0] + M[s * 4 + 1] * v[1] + M[s * 4 + 2] * v[2] + M[s * 4 + 3] * v[3];
}
// a[s] = sum_x M[x][s] v[x]
template <typename T>
__device__ __forceinline__ void mvt4(const T* __restrict__ M, const T v[4], T a[4]) {
#pragma unroll
  for (int s = 0; s < 4; ++s) a[s] = M[0 * 4 + s] * v[0] + M[1 * 4 + s] * v[1] + M[2 * 4 + s] * v[2] + M[3 * 4 + s] * v[3];
}

// the operand vector x of (child, category c, pattern p): partials, broadcast partials, or one-hot / all-ones
template <typename T>
__device__ __forceinline__ void operand4(int kind, const void* ptr, int c, int p, int P, T x[4]) {
  if (kind == KIND_PARTIALS) {
    ld4(static_cast<const T*>(ptr) + ((size_t)c * P + p) * 4, x);
  } else if (kind == KIND_BCAST) {
    ld4(static_cast<const T*>(ptr) + (size_t)p * 4, x);
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

// ---------------------------------------------------------------------------------------------------------------
// post-order update + immediate per-pattern rescaling
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_post4(const DevOp* __restrict__ ops, int P) {
  const DevOp op = ops[blockIdx.y];
  __shared__ T sM[2][C * 16];
  for (int i = threadIdx.x; i < C * 16; i += NUC_THREADS) {
    sM[0][i] = static_cast<const T*>(op.mat[0])[i];
    sM[1][i] = static_cast<const T*>(op.mat[1])[i];
  }
  __syncthreads();
  const int p = blockIdx.x * NUC_THREADS + threadIdx.x;
  if (p >= P) return;
  T r[C][4];
  T mx = T(0);
#pragma unroll
  for (int c = 0; c < C; ++c) {
    T a[4], b[4];
    contrib4<T>(op.kind[0], op.child[0], sM[0] + c * 16, c, p, P, a);
    contrib4<T>(op.kind[1], op.child[1], sM[1] + c * 16, c, p, P, b);
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      r[c][s] = a[s] * b[s];
      mx = fmax(mx, r[c][s]);
    }
  }
  if (op.scale != nullptr) {
    const int e = exp_of(mx);
    if (e != 0) {
      const Pow2Pair<T> f = pow2_pair(-e, T(0));
#pragma unroll
      for (int c = 0; c < C; ++c)
#pragma unroll
        for (int s = 0; s < 4; ++s) r[c][s] = (r[c][s] * f.f1) * f.f2;
    }
    static_cast<int16_t*>(op.scale)[p] = (int16_t)e;
  }
  T* dest = static_cast<T*>(op.dest);
#pragma unroll
  for (int c = 0; c < C; ++c) st4(dest + ((size_t)c * P + p) * 4, r[c]);
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
#pragma unroll
  for (int o = G / 2; o > 0; o >>= 1) lik += __shfl_xor_sync(0xffffffffu, lik, o);
  if (p < P) {
    if (g == 0) {
      long esum = 0;
      for (int k = 0; k < n_scales; ++k) {
        if (SP == 4) {
          esum += static_cast<const int16_t*>(scales[k])[p];
        } else {
          const T* mxs = static_cast<const T*>(scales[k]);
          T m = T(0);
          for (int c = 0; c < C; ++c) m = fmax(m, mxs[(size_t)c * P + p]);
          esum += exp_of(m);
        }
      }
      const double ll = log(lik) + 0.6931471805599453094 * (double)esum;
      if (site != nullptr) site[p] = ll;
      term = weights[p] * ll;
    }
  }
  const double s = block_sum(term, red);
  if (threadIdx.x == 0) block_partial[blockIdx.x] = s;
}

// out[slot] = sum_i partial[slot][i] in a fixed order (deterministic: SURVEY section 7 hard part 8)
__global__ void __launch_bounds__(128) k_sum_rows(const double* __restrict__ partial, int n, int stride,
                                                  double* __restrict__ out) {
  __shared__ double red[4];
  const double* row = partial + (size_t)blockIdx.x * stride;
  double v = 0.0;
  for (int i = threadIdx.x; i < n; i += 128) v += row[i];
  const double s = block_sum(v, red);
  if (threadIdx.x == 0) out[blockIdx.x] = s;
}

// ---------------------------------------------------------------------------------------------------------------
// pre-order update of both children of one parent, fused with both branch derivatives
//
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_pre4(const DevPreItem* __restrict__ items, int P,
                                                      const T* __restrict__ Qg, const double* __restrict__ catw,
                                                      const double* __restrict__ catr,
                                                      const double* __restrict__ weights,
                                                      double* __restrict__ grad_partial, int n_tiles,
                                                      double* __restrict__ site_out) {
  const DevPreItem it = items[blockIdx.y];
  __shared__ T sM[2][C * 16];
  __shared__ T sQ[16];
  __shared__ double red[NUC_THREADS / 32];
  for (int i = threadIdx.x; i < C * 16; i += NUC_THREADS) {
    sM[0][i] = static_cast<const T*>(it.mat[0])[i];
    sM[1][i] = static_cast<const T*>(it.mat[1])[i];
  }
  if (threadIdx.x < 16) sQ[threadIdx.x] = Qg[threadIdx.x];
  __syncthreads();
  const int p = blockIdx.x * NUC_THREADS + threadIdx.x;
  const bool live = p < P;
  const bool want_grad = it.slot[0] >= 0 || it.slot[1] >= 0;
  double d[2] = {0.0, 0.0};
  if (live) {
    T q[2][C][4];
    T mxq[2] = {T(0), T(0)};
    double num[2] = {0.0, 0.0}, den[2] = {0.0, 0.0};
#pragma unroll
    for (int c = 0; c < C; ++c) {
      T qm[4], x[2][4], a[2][4];
      ld4(static_cast<const T*>(it.qm) + ((size_t)c * P + p) * 4, qm);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        operand4<T>(it.kind[k], it.p[k], c, p, P, x[k]);
        mv4<T>(sM[k] + c * 16, x[k], a[k]);
      }
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        T u[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) u[s] = qm[s] * a[1 - k][s];
        mvt4<T>(sM[k] + c * 16, u, q[k][c]);
#pragma unroll
        for (int s = 0; s < 4; ++s) mxq[k] = fmax(mxq[k], q[k][c][s]);
        if (want_grad) {
          T qx[4];
          mv4<T>(sQ, x[k], qx);
          T n = T(0), dd = T(0);
#pragma unroll
          for (int s = 0; s < 4; ++s) {
            n += q[k][c][s] * qx[s];
            dd += q[k][c][s] * x[k][s];
          }
          num[k] += catw[c] * catr[c] * (double)n;
          den[k] += catw[c] * (double)dd;
        }
      }
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      if (it.q[k] != nullptr) {
        const int e = exp_of(mxq[k]);
        const Pow2Pair<T> f = pow2_pair(-e, T(0));
        T* dst = static_cast<T*>(it.q[k]);
#pragma unroll
        for (int c = 0; c < C; ++c) {
          T v[4];
#pragma unroll
          for (int s = 0; s < 4; ++s) v[s] = (q[k][c][s] * f.f1) * f.f2;
          st4(dst + ((size_t)c * P + p) * 4, v);
        }
      }
      if (it.slot[k] >= 0) {
        const double r = num[k] / den[k];
        if (site_out != nullptr) site_out[(size_t)it.slot[k] * P + p] = r;
        d[k] = weights[p] * r;
      }
    }
  }
  if (want_grad) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      if (it.slot[k] < 0) continue;  // uniform over the block
      const double s = block_sum(d[k], red);
      if (threadIdx.x == 0) grad_partial[(size_t)it.slot[k] * n_tiles + blockIdx.x] = s;
    }
  }
}

// root pre-order partials: q_root[c][p][.] = pi
template <typename T>
__global__ void k_fill_root_pre(T* __restrict__ q, const double* __restrict__ pi, size_t n, int SP) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) q[i] = (T)pi[i % SP];
}

// ---------------------------------------------------------------------------------------------------------------
// unfused branch derivatives from stored pre- and post-order partials
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_deriv4(const DevBranch* __restrict__ br, int P,
                                                        const T* __restrict__ Qg, const double* __restrict__ catw,
                                                        const double* __restrict__ catr,
                                                        const double* __restrict__ weights,
                                                        double* __restrict__ grad_partial, int n_tiles,
                                                        double* __restrict__ site_out) {
  const DevBranch b = br[blockIdx.y];
  __shared__ T sQ[16];
  __shared__ double red[NUC_THREADS / 32];
  if (threadIdx.x < 16) sQ[threadIdx.x] = Qg[threadIdx.x];
  __syncthreads();
  const int p = blockIdx.x * NUC_THREADS + threadIdx.x;
  double d = 0.0;
  if (p < P) {
    double num = 0.0, den = 0.0;
#pragma unroll
    for (int c = 0; c < C; ++c) {
      T q[4], x[4], qx[4];
      ld4(static_cast<const T*>(b.q) + ((size_t)c * P + p) * 4, q);
      operand4<T>(b.kind, b.p, c, p, P, x);
      mv4<T>(sQ, x, qx);
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
