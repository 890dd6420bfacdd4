// plk_misc.cuh -- transition matrices from the eigendecomposition and the layout
// conversion kernels behind the setters / getters (host fp64 [..][S]  <->  device T [..][SP], SP = padded states).
#pragma once
#include "plk_common.cuh"

namespace plk {

// One block per branch: M_c = U diag(f(lambda, r_c, t)) U^-1 for every category c, fp64 arithmetic, stored as T in
// the padded layout [C][SP][SP] (padding stays zero).  mode 0: f = exp(lambda * (r_c * t)) (transition matrices);
// mode 1: f = lambda (rebuilds the rate matrix Q; C = 1, also written in fp64 to out64 [S][S]).
// Shared memory: U and U^-1 (2 S^2 doubles) + the C*S diagonal factors.
template <typename T>
__global__ void __launch_bounds__(256) k_transition(const double* __restrict__ U, const double* __restrict__ Uinv,
                                                    const double* __restrict__ lam, const double* __restrict__ rates,
                                                    const double* __restrict__ t, void* const* __restrict__ mats,
                                                    double* __restrict__ out64, int S, int SP, int C, int mode) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* sU = reinterpret_cast<double*>(smem_raw);
  double* sV = sU + S * S;
  double* sF = sV + S * S;
  for (int i = threadIdx.x; i < S * S; i += blockDim.x) {
    sU[i] = U[i];
    sV[i] = Uinv[i];
  }
  const double tb = mode == 0 ? t[blockIdx.x] : 0.0;
  for (int i = threadIdx.x; i < C * S; i += blockDim.x) {
    const int c = i / S, k = i % S;
    sF[i] = mode == 0 ? exp(lam[k] * (rates[c] * tb)) : lam[k];
  }
  __syncthreads();
  T* out = static_cast<T*>(mats[blockIdx.x]);
  for (int idx = threadIdx.x; idx < C * S * S; idx += blockDim.x) {
    const int c = idx / (S * S), rem = idx % (S * S), i = rem / S, j = rem % S;
    double acc = 0.0;
    for (int k = 0; k < S; ++k) acc = fma(sU[i * S + k] * sF[c * S + k], sV[k * S + j], acc);
    out[((size_t)c * SP + i) * SP + j] = (T)acc;
    if (out64 != nullptr) out64[idx] = acc;
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
