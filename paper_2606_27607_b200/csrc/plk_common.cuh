// plk_common.cuh -- device-side descriptors and small numeric helpers shared by the kernels of libplk.
//
// Launch items are plain structs of device pointers, built on the host by plk_api.cu, copied to device memory and
// indexed by blockIdx.y.  Kinds of a child operand:
//   KIND_PARTIALS  full partials              T [C][P][SP]
//   KIND_BCAST     single-category partials   T [P][SP]        (tip partials, the same for every category)
//   KIND_STATES    compact tip states         uint8 [P]        (value >= S: missing, contributes 1 for every state)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace plk {

enum : int { KIND_PARTIALS = 0, KIND_BCAST = 1, KIND_STATES = 2, KIND_NONE = 3 /* operand absent: zeros */ };

// One post-order operation.
struct alignas(16) DevOp {
  void* dest;          // T [C][P][SP]
  const void* child[2];
  const void* mat[2];  // T [C][SP][SP]
  void* scale;         // S=4: int16 [P] exponents (immediate rescaling).  SP=64: T [C][P] maxima (deferred rescaling)
  const void* cscale[2];  // SP=64 only: pending maxima T [C][P] of each child (NULL: none)
  int32_t kind[2];
};

// Both children of one parent in the pre-order pass (SURVEY 8(a) steps 5-6 fused).
struct alignas(16) DevPreItem {
  const void* qm;       // parent pre-order partials T [C][P][SP]
  const void* qm_scale; // SP=64: pending maxima of qm (T [C][P]) or NULL
  void* q[2];           // pre-order partials written for child 0 / 1 (NULL: not stored)
  void* q_scale[2];     // SP=64: maxima written next to q (T [C][P])
  const void* p[2];     // post-order operand of child 0 / 1
  const void* p_scale[2];
  const void* mat[2];   // transition matrices of the branches above child 0 / 1
  int32_t kind[2];
  int32_t slot[2];      // gradient output slot of child 0 / 1, or -1
};

// One branch of the unfused derivative call.
struct DevBranch {
  const void* q;  // pre-order partials of the node, T [C][P][SP]
  const void* p;  // post-order operand of the node
  int32_t kind;
  int32_t slot;
};

// ---------------------------------------------------------------------------------------------------------------
// power-of-two rescaling helpers: e = exponent with m * 2^-e in [0.5, 1); exact multiplications only
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int exp_of(double m) {
  if (!(m > 0.0) || m > 1.7e308) return 0;  // zero, negative, NaN, Inf: leave unscaled
  int e;
  frexp(m, &e);
  return e;
}
__device__ __forceinline__ int exp_of(float m) {
  if (!(m > 0.0f) || m > 3.0e38f) return 0;
  int e;
  frexpf(m, &e);
  return e;
}
__device__ __forceinline__ double pow2i(int k, double) {  // 2^k, k in [-1022, 1023]
  return __hiloint2double((k + 1023) << 20, 0);
}
__device__ __forceinline__ float pow2i(int k, float) {  // 2^k, k in [-126, 127]
  return __int_as_float((k + 127) << 23);
}
// factor pair (f1, f2) with f1 * f2 = 2^k for any k that can occur (|k| <= 2 * max exponent)
template <typename T>
struct Pow2Pair {
  T f1, f2;
};
__device__ __forceinline__ Pow2Pair<double> pow2_pair(int k, double) {
  int k1 = k > 1000 ? 1000 : (k < -1000 ? -1000 : k);
  int k2 = k - k1;
  k2 = k2 > 1000 ? 1000 : (k2 < -1000 ? -1000 : k2);
  return {pow2i(k1, 0.0), pow2i(k2, 0.0)};
}
__device__ __forceinline__ Pow2Pair<float> pow2_pair(int k, float) {
  int k1 = k > 120 ? 120 : (k < -120 ? -120 : k);
  int k2 = k - k1;
  k2 = k2 > 120 ? 120 : (k2 < -120 ? -120 : k2);
  return {pow2i(k1, 0.0f), pow2i(k2, 0.0f)};
}

// ---------------------------------------------------------------------------------------------------------------
// 4-wide vector access (one pattern-category cell of a 4-state partials buffer)
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void ld4(const double* p, double v[4]) {
  const double2 a = reinterpret_cast<const double2*>(p)[0];
  const double2 b = reinterpret_cast<const double2*>(p)[1];
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ void ld4(const float* p, float v[4]) {
  const float4 a = *reinterpret_cast<const float4*>(p);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
}
// the same from GLOBAL memory in one 256-bit request per lane (sm_100: ld.global.v4.f64; 32-byte aligned): a warp whose
// lanes take consecutive cells then touches every 128-byte line once instead of twice (two 16-byte halves at a
// 32-byte stride).  volatile: stays behind griddepcontrol.wait.
__device__ __forceinline__ void ldg4(const double* p, double v[4]) {
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
}
__device__ __forceinline__ void ldg4(const float* p, float v[4]) { ld4(p, v); }
// coherent variants for buffers that the same launch also writes (walk kernels): ordered against every other access
__device__ __forceinline__ void ldg4c(const double* p, double v[4]) {
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3])
               : "l"(p)
               : "memory");
}
__device__ __forceinline__ void ldg4c(const float* p, float v[4]) { ld4(p, v); }
__device__ __forceinline__ void stg4c(double* p, const double v[4]) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
}
__device__ __forceinline__ void stg4c(float* p, const float v[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void st4(double* p, const double v[4]) {
  reinterpret_cast<double2*>(p)[0] = make_double2(v[0], v[1]);
  reinterpret_cast<double2*>(p)[1] = make_double2(v[2], v[3]);
}
__device__ __forceinline__ void st4(float* p, const float v[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}

// deterministic block sum of one double per thread; result valid in thread 0.  `red` holds >= blockDim.x/32 doubles.
__device__ __forceinline__ double block_sum(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (l == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0)
    for (int i = 0; i < nw; ++i) s += red[i];
  return s;
}

}  // namespace plk
