// plk_misc.cuh -- transition matrices from the eigendecomposition and the layout
// conversion kernels behind the setters / getters (host fp64 [..][S]  <->  device T [..][SP], SP = padded states).
#pragma once
#include "plk_common.cuh"

namespace plk {

// One block per branch: M_c = U diag(f(lambda, r_c, t)) U^-1 for every category c, fp64 arithmetic, stored as T in
// the padded layout [C][SP][SP] (padding stays zero).  mode 0: f = exp(lambda * (r_c * t)) (transition matrices);
// mode 1: f = lambda (rebuilds the rate matrix Q; C = 1, also written in fp64 to out64 [S][S]).
// Shared memory: U and U^-1 (2 S^2 doubles) + the C*S diagonal factors.
// One block per (matrix, category): W = U diag(f) (S x S, formed once per block) and U^-1 with its rows padded to a
// multiple of four columns sit in shared memory; a thread owns a strip of four consecutive columns of one row, so an
// inner-loop step is one broadcast load of W[i][k], one 32-byte load of U^-1[k][4 js ..] and four fp64 FMAs (the first
// version spent five instructions per FMA on three scalar shared-memory loads and a multiplication, and gave a
// 62-branch tree 62 blocks for 148 SMs: 139 us at configs[2], 382 us at configs[3]).  Same products, same summation
// order over k as before: results are unchanged bit for bit.
inline size_t transition_smem(int S) { return ((size_t)S * S + (size_t)S * 4 * ((S + 3) / 4) + S) * sizeof(double); }

template <typename T>
__global__ void __launch_bounds__(256) k_transition(const double* __restrict__ U, const double* __restrict__ Uinv,
                                                    const double* __restrict__ lam, const double* __restrict__ rates,
                                                    const double* __restrict__ t, void* const* __restrict__ mats,
                                                    double* __restrict__ out64, int S, int SP, int C, int mode) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NS = (S + 3) / 4, LD = 4 * NS;  // strips per row, padded row length of U^-1
  double* sV = reinterpret_cast<double*>(smem_raw);  // [S][LD]  U^-1[k][.], zero padded; within a row the columns are
                                                     // stored as [strip js: cols 4js, 4js+1] x NS, then [cols 4js+2, 4js+3] x NS,
                                                     // so that the lanes of a quarter warp read consecutive 16-byte chunks
  double* sW = sV + S * LD;                          // [S][S]   U[i][k] f[k]
  double* sF = sW + S * S;                           // [S]
  const int c = blockIdx.y;
  const double tb = mode == 0 ? t[blockIdx.x] : 0.0;
  for (int k = threadIdx.x; k < S; k += blockDim.x) sF[k] = mode == 0 ? exp(lam[k] * (rates[c] * tb)) : lam[k];
  for (int i = threadIdx.x; i < S * LD; i += blockDim.x) {
    const int k = i / LD, j = i - k * LD;  // column j of row k -> strip j / 4, element j % 4
    const int js = j >> 2, e = j & 3;
    sV[k * LD + (e >> 1) * 2 * NS + 2 * js + (e & 1)] = j < S ? Uinv[k * S + j] : 0.0;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < S * S; i += blockDim.x) sW[i] = U[i] * sF[i % S];
  __syncthreads();
  T* out = static_cast<T*>(mats[blockIdx.x]) + (size_t)c * SP * SP;
  const int NR = (S + 1) / 2;  // row pairs: a thread owns rows 2 ip, 2 ip + 1 x four columns (8 FMAs per two 32-byte loads)
  for (int idx = threadIdx.x; idx < NR * NS; idx += blockDim.x) {
    const int ip = idx / NS, js = idx - ip * NS, i0 = 2 * ip, i1 = i0 + 1 < S ? i0 + 1 : i0, j0 = 4 * js;
    const double* w0 = sW + i0 * S;
    const double* w1 = sW + i1 * S;
    const double* v = sV + 2 * js;
    double a[2][4] = {{0.0, 0.0, 0.0, 0.0}, {0.0, 0.0, 0.0, 0.0}};
#pragma unroll 4
    for (int k = 0; k < S; ++k) {
      const double x0 = w0[k], x1 = w1[k];
      const double2 v01 = *reinterpret_cast<const double2*>(v + k * LD);
      const double2 v23 = *reinterpret_cast<const double2*>(v + k * LD + 2 * NS);
      a[0][0] = fma(x0, v01.x, a[0][0]);
      a[0][1] = fma(x0, v01.y, a[0][1]);
      a[0][2] = fma(x0, v23.x, a[0][2]);
      a[0][3] = fma(x0, v23.y, a[0][3]);
      a[1][0] = fma(x1, v01.x, a[1][0]);
      a[1][1] = fma(x1, v01.y, a[1][1]);
      a[1][2] = fma(x1, v23.x, a[1][2]);
      a[1][3] = fma(x1, v23.y, a[1][3]);
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int i = i0 + r;
      if (i >= S) break;
#pragma unroll
      for (int e = 0; e < 4; ++e)
        if (j0 + e < S) {
          out[(size_t)i * SP + j0 + e] = (T)a[r][e];
          if (out64 != nullptr) out64[(size_t)c * S * S + i * S + j0 + e] = a[r][e];
        }
    }
  }
}

// dst[r][0..SP) <- src[r][0..S) (zero padding), r < rows
template <typename T>
__global__ void k_pad_rows(const double* __restrict__ src, T* __restrict__ dst, size_t rows, int S, int SP) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows * SP) return;
  const size_t r = i / SP;
  const int s = (int)(i % SP);
  dst[i] = s < S ? (T)src[r * S + s] : T(0);
}
// dst[r][0..S) <- src[r][0..S) of a padded buffer
template <typename T>
__global__ void k_unpad_rows(const T* __restrict__ src, double* __restrict__ dst, size_t rows, int S, int SP) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows * S) return;
  const size_t r = i / S;
  const int s = (int)(i % S);
  dst[i] = (double)src[r * SP + s];
}
// [C][S][S] host layout -> [C][SP][SP]
template <typename T>
__global__ void k_pad_matrices(const double* __restrict__ src, T* __restrict__ dst, int n, int S, int SP) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)n * SP * SP) return;
  const int m = (int)(i / ((size_t)SP * SP)), rem = (int)(i % ((size_t)SP * SP)), r = rem / SP, c = rem % SP;
  dst[i] = (r < S && c < S) ? (T)src[((size_t)m * S + r) * S + c] : T(0);
}
template <typename T>
__global__ void k_unpad_matrices(const T* __restrict__ src, double* __restrict__ dst, int n, int S, int SP) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)n * S * S) return;
  const int m = (int)(i / ((size_t)S * S)), rem = (int)(i % ((size_t)S * S)), r = rem / S, c = rem % S;
  dst[i] = (double)src[((size_t)m * SP + r) * SP + c];
}
// compact states int32 -> uint8, anything outside 0..S-1 becomes S (missing)
__global__ void k_pack_states(const int32_t* __restrict__ src, uint8_t* __restrict__ dst, int P, int S) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < P) dst[i] = (uint8_t)((src[i] < 0 || src[i] >= S) ? S : src[i]);
}
// rows of `width` bytes from a dense block (row r at src + r * width) into pitched rows (dst + r * pitch); blockIdx.y = row.
// (A pitched device-to-device cudaMemcpy2DAsync of 128 rows took 0.5 ms: the copy engine handles it row by row.)
__global__ void k_scatter_rows(const uint8_t* __restrict__ src, uint8_t* __restrict__ dst, size_t width, size_t pitch) {
  const uint8_t* s = src + (size_t)blockIdx.y * width;
  uint8_t* d = dst + (size_t)blockIdx.y * pitch;
  const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 16;
  if (i >= width) return;
  if (i + 16 <= width && ((reinterpret_cast<uintptr_t>(s + i) | reinterpret_cast<uintptr_t>(d + i)) & 15) == 0) {
    *reinterpret_cast<uint4*>(d + i) = *reinterpret_cast<const uint4*>(s + i);
  } else {
    for (size_t j = i; j < width && j < i + 16; ++j) d[j] = s[j];
  }
}
// expand compact states into fp64 partials [C][P][S] (plk_get_partials on a compact tip)
__global__ void k_expand_states(const uint8_t* __restrict__ st, double* __restrict__ dst, int C, int P, int S) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)C * P * S) return;
  const int s = (int)(i % S);
  const int p = (int)((i / S) % P);
  const int z = st[p];
  dst[i] = (z >= S || z == s) ? 1.0 : 0.0;
}
// natural-log scale factors of one scale buffer
template <typename T>
__global__ void k_scale_logs(const void* __restrict__ scale, double* __restrict__ dst, int P, int C, int deferred) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  int e;
  if (!deferred) {
    e = static_cast<const int16_t*>(scale)[p];
  } else {
    const T* m = static_cast<const T*>(scale);
    T v = T(0);
    for (int c = 0; c < C; ++c) v = fmax(v, m[(size_t)c * P + p]);
    e = exp_of(v);
  }
  dst[p] = 0.6931471805599453094 * (double)e;
}

}  // namespace plk
