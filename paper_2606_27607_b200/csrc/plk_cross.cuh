// plk_cross.cuh -- approximate gradient of logL with respect to the ELEMENTS of the rate matrix (
// "the gradient w.r.t. elements of the rate matrix ... exploiting a first-order approximation of
// the derivative of the matrix exponential").  With d exp(Q tau) / d Q_ij ~= tau exp(Q tau) E_ij the sandwich of a
// branch collapses into an outer product of the pre- and post-order partials of the SAME node (DESIGN.md section 2,
// reading 14):
//     G[i][j] = sum_b t_b sum_p omega_p ( sum_c w_c r_c q_b[c,p,i] p_b[c,p,j] ) / ( sum_c w_c q_b[c,p]^T p_b[c,p] )
// the same pre- and post-order buffers the branch-length gradient uses; per-pattern scale factors cancel in the
// quotient.  Pattern sums are fp64 in both precisions and reduced in a fixed order (bitwise repeatable).
//   4 states   HBM-bound: 2 W bytes per branch; a thread owns a pattern, the 16 sums live in registers.
//   64 states  a contraction over the pattern axis (G_c = Q_c^T diag(s) P_c, 64 x 64 x patterns): a CTA owns a chunk of
//              patterns, a thread a 4 x 4 block of G; first pass over the categories for den, second for the outer
//              products (the tiles of a chunk stay in L2 between the two).
#pragma once
#include "plk_common.cuh"
#include "plk_gen.cuh"
#include "plk_nuc.cuh"

namespace plk {

struct DevCrossBranch {
  const void* q;  // pre-order partials of the node, T [C][P][SP]
  const void* p;  // post-order operand of the node
  double t;       // branch length above the node
  int32_t kind;
  int32_t pad;
};

constexpr int CROSS4_THREADS = 128, CROSS4_SPLITS = 8;

// grid.x = pattern blocks, grid.y = branch ranges (a thread's walk over the branches is one dependent chain of loads:
// with one range the 782 blocks of configs[1] gave an SM 21 warps and the kernel ran at a third of the HBM rate).
// partial[e][blockIdx.y * gridDim.x + blockIdx.x], e = 4 i + j; n_blocks = gridDim.x * gridDim.y.
template <typename T, int C>
__global__ void __launch_bounds__(CROSS4_THREADS) k_cross4(const DevCrossBranch* __restrict__ br, int n_br, int P,
                                                           const double* __restrict__ catw, const double* __restrict__ catr,
                                                           const double* __restrict__ weights, double* __restrict__ partial,
                                                           int n_blocks) {
  __shared__ double red[CROSS4_THREADS / 32];
  const int p = blockIdx.x * CROSS4_THREADS + threadIdx.x;
  double g[16];
#pragma unroll
  for (int e = 0; e < 16; ++e) g[e] = 0.0;
  if (p < P) {
    const double wp = weights[p];
    const int b_lo = (int)((long long)blockIdx.y * n_br / gridDim.y), b_hi = (int)((long long)(blockIdx.y + 1) * n_br / gridDim.y);
    for (int b = b_lo; b < b_hi; ++b) {
      const DevCrossBranch B = br[b];
      // category sums in the working precision, widened once per branch (16 fp64 FMAs and conversions per category
      // made the fp32 instantiation as slow as fp64)
      T num[16], den = T(0);
#pragma unroll
      for (int e = 0; e < 16; ++e) num[e] = T(0);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        T q[4], x[4];
        ld4(static_cast<const T*>(B.q) + ((size_t)c * P + p) * 4, q);
        operand4<T>(B.kind, B.p, c, p, P, x);
        const T cw = (T)catw[c], cwr = (T)(catw[c] * catr[c]);
        T d = T(0);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          d += q[i] * x[i];
          const T qi = cwr * q[i];  // 4 products + 16 FMAs per category instead of 16 + 16
#pragma unroll
          for (int j = 0; j < 4; ++j) num[4 * i + j] = fma(qi, x[j], num[4 * i + j]);
        }
        den = fma(cw, d, den);
      }
      const double s = wp * B.t / (double)den;
#pragma unroll
      for (int e = 0; e < 16; ++e) g[e] = fma(s, (double)num[e], g[e]);
    }
  }
#pragma unroll
  for (int e = 0; e < 16; ++e) {
    const double s = block_sum(g[e], red);
    if (threadIdx.x == 0) partial[(size_t)e * n_blocks + blockIdx.y * gridDim.x + blockIdx.x] = s;
  }
}

// ---- 32 / 64 padded states ----------------------------------------------------------------------------------------
constexpr int CROSS64_TP = 32, CROSS64_THREADS = 256;
template <typename T, int SP = SP64>
constexpr size_t cross64_smem() {
  return (size_t)2 * CROSS64_TP * Gen<T, SP>::TS * sizeof(T) + (size_t)2 * CROSS64_TP * sizeof(double);
}

// grid.x = pattern chunks of 32; thread (ti, tj) = (tid >> 4, tid & 15) owns the B x B block G[B ti ..][B tj ..],
// B = SP / 16.  partial[block][i * SP + j] (padded rows / columns stay 0).
template <typename T, int SP = SP64>
__global__ void __launch_bounds__(CROSS64_THREADS) k_cross64(const DevCrossBranch* __restrict__ br, int n_br, int P, int S,
                                                             int C, const double* __restrict__ catw,
                                                             const double* __restrict__ catr,
                                                             const double* __restrict__ weights,
                                                             double* __restrict__ partial) {
  constexpr int TS = Gen<T, SP>::TS, B = SP / 16, NPT = SP / 8;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* tQ = reinterpret_cast<T*>(smem_raw);
  T* tX = tQ + CROSS64_TP * TS;
  double* sDen = reinterpret_cast<double*>(tX + CROSS64_TP * TS);
  double* sScale = sDen + CROSS64_TP;
  static_assert(CROSS64_TP == GEN_TP && CROSS64_THREADS == GEN_THREADS, "load_tile geometry");
  const int p0 = blockIdx.x * CROSS64_TP;
  const int ti = threadIdx.x >> 4, tj = threadIdx.x & 15;
  const int pp = threadIdx.x >> 3, sb = threadIdx.x & 7;  // den pass: 8 lanes per pattern, NPT states each
  double g[B * B];
#pragma unroll
  for (int e = 0; e < B * B; ++e) g[e] = 0.0;
  for (int b = 0; b < n_br; ++b) {
    const DevCrossBranch Br = br[b];
    // pass 1: den_p = sum_c w_c q^T p
    if (threadIdx.x < CROSS64_TP) sDen[threadIdx.x] = 0.0;
    for (int c = 0; c < C; ++c) {
      __syncthreads();
      load_tile<T, SP>(tQ, KIND_PARTIALS, Br.q, c, p0, P, S);
      load_tile<T, SP>(tX, Br.kind, Br.p, c, p0, P, S);
      __syncthreads();
      T d = T(0);
#pragma unroll
      for (int k = 0; k < NPT; ++k) d = fma(tQ[pp * TS + NPT * sb + k], tX[pp * TS + NPT * sb + k], d);
      d = lane8_sum(d);
      if (sb == 0) sDen[pp] += catw[c] * (double)d;
    }
    // pass 2: G += sum_c sum_p (omega_p w_c r_c t_b / den_p) q[p, i] p[p, j]   (the chunk's tiles come back from L2)
    for (int c = 0; c < C; ++c) {
      __syncthreads();
      load_tile<T, SP>(tQ, KIND_PARTIALS, Br.q, c, p0, P, S);
      load_tile<T, SP>(tX, Br.kind, Br.p, c, p0, P, S);
      if (threadIdx.x < CROSS64_TP) {
        const int p = p0 + threadIdx.x;
        sScale[threadIdx.x] = p < P ? weights[p] * catw[c] * catr[c] * Br.t / sDen[threadIdx.x] : 0.0;
      }
      __syncthreads();
      T acc[B * B];  // working-precision sum over the 32 patterns of the chunk, widened once per (branch, category)
#pragma unroll
      for (int e = 0; e < B * B; ++e) acc[e] = T(0);
#pragma unroll 4
      for (int r = 0; r < CROSS64_TP; ++r) {
        const T sc = (T)sScale[r];
        T qi[B], xj[B];
#pragma unroll
        for (int k = 0; k < B; ++k) {
          qi[k] = tQ[r * TS + B * ti + k] * sc;
          xj[k] = tX[r * TS + B * tj + k];
        }
#pragma unroll
        for (int i = 0; i < B; ++i)
#pragma unroll
          for (int j = 0; j < B; ++j) acc[B * i + j] = fma(qi[i], xj[j], acc[B * i + j]);
      }
#pragma unroll
      for (int e = 0; e < B * B; ++e) g[e] += (double)acc[e];
    }
    __syncthreads();
  }
  double* out = partial + (size_t)blockIdx.x * SP * SP;
#pragma unroll
  for (int i = 0; i < B; ++i)
#pragma unroll
    for (int j = 0; j < B; ++j) out[(B * ti + i) * SP + B * tj + j] = g[B * i + j];
}

// out[e] = sum over blocks of partial[block][e] in block order (fixed order)
__global__ void __launch_bounds__(256) k_sum_blocks(const double* __restrict__ partial, int n_blocks, int n_elem,
                                                    double* __restrict__ out) {
  const int e = blockIdx.x * 256 + threadIdx.x;
  if (e >= n_elem) return;
  double s = 0.0;
  for (int b = 0; b < n_blocks; ++b) s += partial[(size_t)b * n_elem + e];
  out[e] = s;
}

}  // namespace plk
