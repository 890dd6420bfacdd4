// plk_cache.cuh -- the two caching variants of PAPER.md:101 (section 4).
//
// (a) Cached rate products.  "the product of the infinitesimal rate matrix and the post-order partial likelihood vector
//     at each node could be cached directly thus reducing memory burden from S^2 elements of the infinitesimal rate
//     matrix to S partial likelihoods": k_rate_products* store Qp_k[c,p,.] = Q p_k[c,p,.] next to every post-order
//     buffer (same layout, same pending rescaling factor as p_k), and k_deriv*_cached evaluate the sandwich of SURVEY
//     8(a) step 6 from it -- num = sum_c w_c r_c q_k . Qp_k, den = sum_c w_c q_k . p_k -- reading S values per (node,
//     pattern, category) instead of applying Q (2 S^2 flops).  A compact tip needs no cache: Q e_z is column z of Q.
//
// (b) Transition matrices on the fly.  "for phylogeographic problems that typically have a large state-space size but
//     only a single site pattern, the transition probability matrices are not reused, and it is more efficient to form
//     the transition probability matrix on-the-fly": k_post_otf applies P = U diag(exp(lambda r_c t)) U^-1 to a child's
//     partial as  U (e o (U^-1 x))  -- two matrix-vector products, 4 S^2 flops per (edge, pattern, category), no S x S
//     matrix formed (2 S^3), stored or re-read -- and runs the WHOLE operation list in one launch: CTAs take (operation,
//     pattern) tickets in list order from an atomic counter and wait on the ready flags of the operations that produce
//     their children.  A ticket only ever waits for lower tickets, whose CTAs are already running, so the dataflow
//     cannot deadlock whatever the grid size, and independent subtrees run concurrently on different SMs: the latency of
//     an evaluation is the tree depth, not the node count.  Arithmetic is fp64 whatever the instance precision (the
//     eigenvector matrices are not rounded); storage and deferred rescaling are those of the padded-state kernels
//     (plk_gen.cuh), so the buffers it writes are interchangeable with theirs.
#pragma once
#include "plk_common.cuh"
#include "plk_gen.cuh"
#include "plk_nuc.cuh"

namespace plk {

struct DevQpItem {  // one post-order buffer whose rate product is cached
  const void* p;    // T [C][P][SP] (KIND_PARTIALS) or T [P][SP] (KIND_BCAST)
  void* qp;         // same shape
  int32_t kind;
  int32_t pad;
};
struct DevBranchQp {  // one branch of the cached derivative call
  const void* q;      // pre-order partials of the node
  const void* p;      // post-order operand of the node
  const void* qp;     // cached Q p (unused for KIND_STATES)
  int32_t kind;
  int32_t slot;
};

// ---- (a) 4 states: one thread per (category, pattern) cell -------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_rate_products4(const DevQpItem* __restrict__ items, int P, int C,
                                                        const T* __restrict__ Qg) {
  const DevQpItem it = items[blockIdx.y];
  const size_t rows = it.kind == KIND_BCAST ? (size_t)P : (size_t)C * P;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows) return;
  T x[4], y[4];
  ld4(static_cast<const T*>(it.p) + i * 4, x);
  mv4<T>(Qg, x, y);
  st4(static_cast<T*>(it.qp) + i * 4, y);
}

template <typename T, int C>
__global__ void __launch_bounds__(NUC_THREADS) k_deriv4_cached(const DevBranchQp* __restrict__ br, int P,
                                                               const T* __restrict__ Qg, const double* __restrict__ catw,
                                                               const double* __restrict__ catr,
                                                               const double* __restrict__ weights,
                                                               double* __restrict__ grad_partial, int n_tiles,
                                                               double* __restrict__ site_out) {
  const DevBranchQp b = br[blockIdx.y];
  __shared__ double red[NUC_THREADS / 32];
  const int p = blockIdx.x * NUC_THREADS + threadIdx.x;
  double d = 0.0;
  if (p < P) {
    double num = 0.0, den = 0.0;
    int z = 4;
    if (b.kind == KIND_STATES) z = static_cast<const uint8_t*>(b.p)[p];
#pragma unroll
    for (int c = 0; c < C; ++c) {
      T q[4], x[4], qx[4];
      ld4(static_cast<const T*>(b.q) + ((size_t)c * P + p) * 4, q);
      if (b.kind == KIND_STATES) {  // Q e_z = column z of Q; a missing state: Q 1 = 0
#pragma unroll
        for (int s = 0; s < 4; ++s) {
          x[s] = z >= 4 ? T(1) : (s == z ? T(1) : T(0));
          qx[s] = z >= 4 ? T(0) : Qg[s * 4 + z];
        }
      } else {
        const size_t row = b.kind == KIND_BCAST ? (size_t)p : (size_t)c * P + p;
        ld4(static_cast<const T*>(b.p) + row * 4, x);
        ld4(static_cast<const T*>(b.qp) + row * 4, qx);
      }
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

// ---- (a) padded state counts (SP = 32, 64): one (tile of 32 patterns, category, buffer) per block ------------------------
template <typename T, int SP = SP64>
constexpr size_t rate_products64_smem() {
  return (SP * SP + GEN_TP * Gen<T, SP>::TS) * sizeof(T);
}
template <typename T, int SP = SP64>
__global__ void __launch_bounds__(GEN_THREADS) k_rate_products64(const DevQpItem* __restrict__ items, int P, int S, int C,
                                                                 const T* __restrict__ Qg) {
  constexpr int TS = Gen<T, SP>::TS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* BQ = reinterpret_cast<T*>(smem_raw);
  T* tX = BQ + SP * SP;
  const DevQpItem it = items[blockIdx.z];
  const int c = blockIdx.y, p0 = blockIdx.x * GEN_TP;
  if (it.kind == KIND_BCAST && c > 0) return;  // one category's worth of rows
  const int pp = threadIdx.x >> 3, sb = threadIdx.x & 7, p = p0 + pp;
  fill_matrix<T, SP>(BQ, Qg, true);
  load_tile<T, SP>(tX, it.kind, it.p, c, p0, P, S);
  __syncthreads();
  T qx[Gen<T, SP>::NPT];
  mv64<T, SP>(BQ, tX + pp * TS, sb, qx);
  if (p < P) {
    const size_t row = it.kind == KIND_BCAST ? (size_t)p : (size_t)c * P + p;
    store_states<T, SP>(static_cast<T*>(it.qp) + row * SP, sb, qx);
  }
}

template <typename T, int SP = SP64>
__global__ void __launch_bounds__(GEN_THREADS) k_deriv64_cached(const DevBranchQp* __restrict__ br, int P, int S, int C,
                                                                const T* __restrict__ Qg,
                                                                const double* __restrict__ catw,
                                                                const double* __restrict__ catr,
                                                                const double* __restrict__ weights,
                                                                double* __restrict__ grad_partial, int n_tiles,
                                                                double* __restrict__ site_out) {
  constexpr int VEC = Gen<T, SP>::VEC, NCH = Gen<T, SP>::NCH;
  using V = typename VecOf<T>::type;
  __shared__ double sRatio[GEN_TP];
  const DevBranchQp b = br[blockIdx.y];
  const int p0 = blockIdx.x * GEN_TP;
  const int pp = threadIdx.x >> 3, sb = threadIdx.x & 7, p = p0 + pp;
  double num = 0.0, den = 0.0;
  {  // every lane takes part (the 8-lane sums are full-warp shuffles); rows past the end re-read the last pattern
    const int pr = p < P ? p : P - 1;
    int z = S;
    if (b.kind == KIND_STATES) z = static_cast<const uint8_t*>(b.p)[pr];
    for (int c = 0; c < C; ++c) {
      const T* qrow = static_cast<const T*>(b.q) + ((size_t)c * P + pr) * SP;
      const size_t row = b.kind == KIND_BCAST ? (size_t)pr : (size_t)c * P + pr;
      T n = T(0), d = T(0);
#pragma unroll
      for (int i = 0; i < NCH; ++i) {
        T q[VEC], x[VEC], qx[VEC];
        const int s0 = (VEC * 8) * i + VEC * sb;
        unpack(*reinterpret_cast<const V*>(qrow + s0), q);
        if (b.kind == KIND_STATES) {
#pragma unroll
          for (int j = 0; j < VEC; ++j) {
            const int s = s0 + j;
            x[j] = z >= S ? (s < S ? T(1) : T(0)) : (s == z ? T(1) : T(0));
            qx[j] = z >= S ? T(0) : Qg[s * SP + z];
          }
        } else {
          unpack(*reinterpret_cast<const V*>(static_cast<const T*>(b.p) + row * SP + s0), x);
          unpack(*reinterpret_cast<const V*>(static_cast<const T*>(b.qp) + row * SP + s0), qx);
        }
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
          n = fma(q[j], qx[j], n);
          d = fma(q[j], x[j], d);
        }
      }
      n = lane8_sum(n);
      d = lane8_sum(d);
      num += catw[c] * catr[c] * (double)n;
      den += catw[c] * (double)d;
    }
  }
  if (sb == 0) sRatio[pp] = p < P ? num / den : 0.0;
  __syncthreads();
  if (threadIdx.x < GEN_TP) {
    const int r = threadIdx.x;
    double v = 0.0;
    if (p0 + r < P) {
      if (site_out != nullptr) site_out[(size_t)b.slot * P + p0 + r] = sRatio[r];
      v = weights[p0 + r] * sRatio[r];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (r == 0) grad_partial[(size_t)b.slot * n_tiles + blockIdx.x] = v;
  }
}

// ---- (b) transition matrices on the fly: the whole post-order list in one launch ---------------------------------------
struct DevOtfOp {
  void* dest;             // T [C][P][SP], stored unscaled (deferred rescaling, plk_gen.cuh)
  void* scale;            // T [C][P] maxima of dest, or NULL
  const void* child[2];
  const void* cscale[2];  // pending maxima of child k (T [C][P]) or NULL
  double t[2];            // length of the branch above child k
  int32_t kind[2];
  int32_t dep[2];         // index in this list of the operation that writes child k, or -1 (already in memory)
};
struct OtfSync {          // lives in the arena, zero at creation, left zero by every launch
  unsigned int ticket, done;
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

constexpr int OTF_THREADS = 256;
template <int SP>
constexpr size_t otf_smem() {
  return ((size_t)2 * SP * SP + SP + 2 * OTF_THREADS + 2 * (OTF_THREADS / 32)) * sizeof(double);
}

// One (operation, pattern) per ticket; thread (cg = tid / SP, s = tid % SP) owns state s of category c0 + cg.
template <typename T, int SP>
__global__ void __launch_bounds__(OTF_THREADS) k_post_otf(const DevOtfOp* __restrict__ ops, int n_ops, int P, int S, int C,
                                                          const double* __restrict__ U, const double* __restrict__ Uinv,
                                                          const double* __restrict__ lam, const double* __restrict__ rates,
                                                          OtfSync* sync, unsigned int* ready, unsigned int epoch) {
  constexpr int CG = OTF_THREADS / SP, WPC = SP / 32;  // categories in flight, warps per category
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* UT = reinterpret_cast<double*>(smem_raw);  // UT[i][s] = U[s][i]
  double* UiT = UT + SP * SP;                         // UiT[x][i] = Uinv[i][x]
  double* sLam = UiT + SP * SP;
  double* xs = sLam + SP;                             // [CG][SP]
  double* ys = xs + OTF_THREADS;
  double* sMx = ys + OTF_THREADS;                     // [CG][WPC] (padded to OTF_THREADS / 32 * 2)
  __shared__ unsigned int s_ticket;
  const int tid = threadIdx.x, cg = tid / SP, s = tid % SP;
  for (int idx = tid; idx < SP * SP; idx += OTF_THREADS) {
    const int r = idx / SP, col = idx % SP;  // UT[r][col] = U[col][r]
    const bool in = r < S && col < S;
    UT[idx] = in ? U[col * S + r] : 0.0;
    UiT[idx] = in ? Uinv[col * S + r] : 0.0;
  }
  if (tid < SP) sLam[tid] = tid < S ? lam[tid] : 0.0;
  const unsigned int total = (unsigned int)n_ops * (unsigned int)P;
  for (;;) {
    __syncthreads();  // smem tables ready / previous ticket's scratch no longer read
    if (tid == 0) s_ticket = atomicAdd(&sync->ticket, 1u);
    __syncthreads();
    const unsigned int tk = s_ticket;
    if (tk >= total) break;
    const int oi = (int)(tk / (unsigned int)P), p = (int)(tk - (unsigned int)oi * (unsigned int)P);
    const DevOtfOp& op = ops[oi];
    if (tid < 2) {  // children written by an earlier operation of this launch: wait for their ready flag
      const int d = op.dep[tid];
      if (d >= 0)
        while (ld_acquire_u32(ready + (size_t)d * P + p) != epoch) __nanosleep(40);
    }
    __syncthreads();
    for (int c0 = 0; c0 < C; c0 += CG) {
      const int c = c0 + cg;
      const bool live = c < C;
      double prod = 1.0;
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        double x = 0.0;
        if (live) {
          const int kind = op.kind[k];
          if (kind == KIND_STATES) {
            const int z = static_cast<const uint8_t*>(op.child[k])[p];
            x = z >= S ? (s < S ? 1.0 : 0.0) : (s == z ? 1.0 : 0.0);
          } else {
            const size_t row = kind == KIND_BCAST ? (size_t)p : (size_t)c * P + p;
            x = (double)__ldcg(static_cast<const T*>(op.child[k]) + row * SP + s);
            if (op.cscale[k] != nullptr) {  // pending power-of-two factor of the child (deferred rescaling)
              const T* m = static_cast<const T*>(op.cscale[k]);
              T v = T(0);
              for (int cc = 0; cc < C; ++cc) v = fmax(v, __ldcg(m + (size_t)cc * P + p));
              x = ldexp(x, -exp_of(v));
            }
          }
        }
        xs[tid] = x;
        __syncthreads();
        double y = 0.0;
#pragma unroll 8
        for (int i = 0; i < SP; ++i) y = fma(UiT[i * SP + s], xs[cg * SP + i], y);  // (U^-1 x)[s]
        y *= live ? exp(sLam[s] * rates[c] * op.t[k]) : 0.0;
        ys[tid] = y;
        __syncthreads();
        double a = 0.0;
#pragma unroll 8
        for (int i = 0; i < SP; ++i) a = fma(UT[i * SP + s], ys[cg * SP + i], a);    // (U y)[s]
        prod *= a;
      }
      const T out = (T)prod;
      T mx = s < S ? out : T(0);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
      if ((tid & 31) == 0) sMx[tid >> 5] = (double)mx;
      if (live) static_cast<T*>(op.dest)[((size_t)c * P + p) * SP + s] = s < S ? out : T(0);
      __syncthreads();
      if (live && s == 0 && op.scale != nullptr) {
        double m = 0.0;
#pragma unroll
        for (int w = 0; w < WPC; ++w) m = fmax(m, sMx[cg * WPC + w]);
        static_cast<T*>(op.scale)[(size_t)c * P + p] = (T)m;
      }
    }
    __syncthreads();  // every store of the ticket is issued
    if (tid == 0) {
      __threadfence();
      st_release_u32(ready + (size_t)oi * P + p, epoch);
    }
  }
  if (tid == 0) {  // the last CTA out leaves the counters at zero for the next launch
    const unsigned int d = atomicAdd(&sync->done, 1u);
    if (d == gridDim.x - 1) {
      sync->ticket = 0u;
      sync->done = 0u;
    }
  }
}

}  // namespace plk
