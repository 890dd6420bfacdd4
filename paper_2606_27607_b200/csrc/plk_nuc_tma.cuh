// plk_nuc_tma.cuh -- 4-state (nucleotide) kernels, TMA-staged: the bandwidth path of SURVEY 8(a) steps 2-6.
//
// Why.  The register-staged kernels of plk_nuc.cuh are latency-bound: every warp loads its operands, waits a DRAM
// round trip (stall_long_sb = 60 % of the stall samples, 16 resident warps per SM at 123 registers;
// profiles/r01_nuc_ldg.md) and only then computes.  Here the loads are decoupled from the arithmetic: ONE producer
// lane per CTA streams tiles into a ring of shared-memory stages with cp.async.bulk (the TMA engine, 1-D bulk
// copies, completion counted in bytes on an mbarrier), NS stages deep, so ~3 x (NS-1) x 12 KB are in flight per SM
// whatever the register count; four consumer warps wait on the stage's "full" barrier, compute out of shared
// memory, store straight from registers and release the stage through its "empty" barrier.
//
// Tile = (item, TP consecutive patterns); one stage holds, per tile:
//   hdr   {p0, n, state offsets}            written by the producer lane before its arrive.expect_tx (release)
//   desc  the item's descriptor (DevOp / DevPreItem), bulk-copied, so consumers never touch global memory for it
//   st    compact tip states of the tile (uint8), when a child is a compact tip
//   wts   pattern weights (fp64), pre-order only
//   mats  the 2 x C transition matrices, one bulk copy per category into padded slabs (bank-conflict-free reads)
//   ops   the operands: C segments of n x 4 reals per operand, each contiguous in the [c][p][s] layout
// Thread mapping inside a tile is that of plk_nuc.cuh: LP lanes share a pattern and split its categories.
//
// Two tile orders (the "launch shapes" of plk.h):
//   walk   ONE launch; CTA b owns a contiguous pattern range (sizes differ by at most PPW patterns) and walks the
//          whole item list over it.  Cell (p, c) of every buffer is produced and consumed by the same CTA, so list
//          order is the only dependency: the consumers fence (fence.proxy.async) before releasing a stage and the
//          producer never runs further ahead than the CTA's own tile count.  Fresh children are re-read from L2.
//   level  one launch per dependency level; tiles (item, pattern tile) are dealt round-robin to the CTAs.
#pragma once
#include "plk_common.cuh"
#include "plk_nuc.cuh"

namespace plk {

// ---- mbarrier / bulk-copy PTX ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// global -> shared bulk copy; src, dst 16-byte aligned, bytes a multiple of 16; completion on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
// programmatic dependent launch (griddepcontrol): `pdl_trigger` lets the next launch of the stream become resident
// as this grid's CTAs drain; `pdl_wait` blocks until the grids this launch depends on have completed and flushed.
// Both are no-ops in a launch without the programmatic-serialisation attribute.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- exponent of a non-negative maximum from its bit pattern (integer max instead of fp compares) ---------------
// key(v) is monotone in v for v >= 0; negative values and -0 give keys <= 0 and never win against 0.
__device__ __forceinline__ int max_key(double v) { return __double2hiint(v); }
__device__ __forceinline__ int max_key(float v) { return __float_as_int(v); }
// e with max * 2^-e in [0.5, 1) (frexp convention), clamped so that 2^-e is a normal number; 0 = leave unscaled
__device__ __forceinline__ int exp_of_key(int key, double) {
  const int be = key >> 20;
  if (key <= 0 || be >= 2047) return 0;
  const int e = be - 1022;
  return e < -1000 ? -1000 : (e > 1000 ? 1000 : e);
}
__device__ __forceinline__ int exp_of_key(int key, float) {
  const int be = key >> 23;
  if (key <= 0 || be >= 255) return 0;
  const int e = be - 126;
  return e < -120 ? -120 : (e > 120 ? 120 : e);
}
__device__ __forceinline__ double pow2_neg(int e, double) { return __hiloint2double((1023 - e) << 20, 0); }
__device__ __forceinline__ float pow2_neg(int e, float) { return __int_as_float((127 - e) << 23); }

template <int LP>
__device__ __forceinline__ int group_max_int(int v) {
#pragma unroll
  for (int o = 32 / LP; o < 32; o <<= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// sum over each segment of PPW consecutive lanes; every lane of a segment gets the segment's sum
template <int PPW>
__device__ __forceinline__ double segment_sum(double v) {
#pragma unroll
  for (int o = PPW / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- configuration ---------------------------------------------------------------------------------------------
constexpr int NT_CW = 4;                    // consumer warps per CTA
constexpr int NT_THREADS = (NT_CW + 1) * 32;  // + one producer warp
constexpr int NT_NS = 4;                    // pipeline stages
constexpr int NT_DESC = 128;                // bytes reserved for the descriptor copy
static_assert(sizeof(DevOp) % 16 == 0 && sizeof(DevOp) <= NT_DESC, "DevOp must be bulk-copyable");
static_assert(sizeof(DevPreItem) % 16 == 0 && sizeof(DevPreItem) <= NT_DESC, "DevPreItem must be bulk-copyable");

struct NtHdr {
  int32_t p0, n, soff0, soff1;  // first pattern, pattern count, offset of pattern p0 inside st[0] / st[1]
};

template <typename T, int C, int NOPS, bool WTS, int R = 1>  // R = pattern rows per consumer lane
struct NtStage {
  using Mp = NucMap<C>;
  static constexpr int TP = Mp::PPW * NT_CW * R;   // patterns per tile
  static constexpr int SEG = TP * 4;               // reals per (operand, category) segment
  static constexpr int MS = NucMat<T>::STRIDE;
  static constexpr int OFF_HDR = 0;
  static constexpr int OFF_DESC = 16;
  static constexpr int OFF_ST = OFF_DESC + NT_DESC;             // 2 x (TP + 16) bytes
  static constexpr int OFF_WTS = OFF_ST + 2 * (TP + 16);        // TP doubles
  static constexpr int OFF_MATS = OFF_WTS + (WTS ? TP * 8 : 0);
  static constexpr int OFF_OPS = OFF_MATS + 2 * C * MS * (int)sizeof(T);
  static constexpr int BYTES = (OFF_OPS + NOPS * C * SEG * (int)sizeof(T) + 127) / 128 * 128;
  static_assert(OFF_MATS % 16 == 0 && OFF_OPS % 16 == 0, "stage regions must be 16-byte aligned");
};

// which tiles a CTA processes, in which order (identical arithmetic on the producer and the consumer side)
struct NtSched {
  int walk;     // 1: walk (own pattern range, item-major); 0: level (round-robin over item x pattern-tile)
  int n_items;
  int P;
  int n_rows;   // ceil(P / PPW)
};
template <int PPW, int TP>
struct NtTiles {
  int walk, J, n_own, lo, hi, n_tp, G, b;
  __device__ __forceinline__ void init(const NtSched& s) {
    walk = s.walk;
    G = gridDim.x;
    b = blockIdx.x;
    if (walk) {
      lo = (int)((long long)b * s.n_rows / G) * PPW;
      hi = (int)((long long)(b + 1) * s.n_rows / G) * PPW;
      if (hi > s.P) hi = s.P;
      n_own = (hi - lo + TP - 1) / TP;
      J = s.n_items * n_own;
      n_tp = 0;
    } else {
      n_tp = (s.P + TP - 1) / TP;
      const long long total = (long long)s.n_items * n_tp;
      J = total > b ? (int)((total - b + G - 1) / G) : 0;
      lo = 0;
      hi = s.P;
      n_own = 0;
    }
  }
  // tile j -> item, first pattern, pattern count, pattern-tile index (level) / own-tile index (walk)
  __device__ __forceinline__ void tile(int j, int& item, int& p0, int& n, int& t) const {
    if (walk) {
      item = j / n_own;
      t = j - item * n_own;
      p0 = lo + t * TP;
    } else {
      const long long idx = (long long)b + (long long)j * G;
      item = (int)(idx / n_tp);
      t = (int)(idx - (long long)item * n_tp);
      p0 = t * TP;
    }
    n = hi - p0 < TP ? hi - p0 : TP;
  }
};

// ---- producer: fill one stage with one tile (single lane) ------------------------------------------------------
// operand o of NOPS: ptr[o], kind[o]; operands NOPS-2 and NOPS-1 are the two children (their compact states go to
// st[0] / st[1]); an operand before them (the parent's pre-order partials) is always KIND_PARTIALS.
template <typename T, int C, int NOPS, bool WTS, int R = 1>
__device__ __forceinline__ void nt_fill(unsigned char* stage, uint64_t* full, const void* desc, uint32_t desc_bytes,
                                        const void* const* ptr, const int* kind, const void* const* mat,
                                        const double* weights, int P, int p0, int n, long long dmat_delta = 0) {
  // dmat_delta != 0 (class-specialised gradient kernels): a child given as compact states leaves its operand segment of
  // the stage unused; the derivative matrices D = M Q of its branch ([C][16], at mat + dmat_delta bytes) are copied there
  using St = NtStage<T, C, NOPS, WTS, R>;
  const uint32_t seg_bytes = (uint32_t)n * 4 * sizeof(T);
  const uint32_t mat_bytes = 16 * sizeof(T);
  NtHdr h;
  h.p0 = p0;
  h.n = n;
  h.soff0 = h.soff1 = 0;
  // pass 1: byte count
  uint32_t bytes = desc_bytes + 2 * C * mat_bytes;
  if (WTS) bytes += ((uint32_t)n * 8 + 15) & ~15u;
#pragma unroll
  for (int o = 0; o < NOPS; ++o) {
    if (kind[o] == KIND_PARTIALS) bytes += C * seg_bytes;
    else if (kind[o] == KIND_BCAST) bytes += seg_bytes;
    else if (kind[o] == KIND_STATES) bytes += (((uint32_t)(n + (p0 & 15)) + 15) & ~15u) + (dmat_delta != 0 ? C * mat_bytes : 0u);
  }
  if (kind[NOPS - 2] == KIND_STATES) h.soff0 = p0 & 15;
  if (kind[NOPS - 1] == KIND_STATES) h.soff1 = p0 & 15;
  *reinterpret_cast<NtHdr*>(stage + St::OFF_HDR) = h;
  mbar_expect_tx(full, bytes);
  // pass 2: copies
  bulk_g2s(stage + St::OFF_DESC, desc, desc_bytes, full);
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int c = 0; c < C; ++c)
      bulk_g2s(stage + St::OFF_MATS + (k * C + c) * St::MS * sizeof(T), static_cast<const T*>(mat[k]) + c * 16,
               mat_bytes, full);
  if (WTS) bulk_g2s(stage + St::OFF_WTS, weights + p0, ((uint32_t)n * 8 + 15) & ~15u, full);
#pragma unroll
  for (int o = 0; o < NOPS; ++o) {
    unsigned char* dst = stage + St::OFF_OPS + (size_t)o * C * St::SEG * sizeof(T);
    if (kind[o] == KIND_PARTIALS) {
#pragma unroll
      for (int c = 0; c < C; ++c)
        bulk_g2s(dst + (size_t)c * St::SEG * sizeof(T), static_cast<const T*>(ptr[o]) + ((size_t)c * P + p0) * 4,
                 seg_bytes, full);
    } else if (kind[o] == KIND_BCAST) {
      bulk_g2s(dst, static_cast<const T*>(ptr[o]) + (size_t)p0 * 4, seg_bytes, full);
    } else if (kind[o] == KIND_STATES) {
      const int k = o - (NOPS - 2);
      bulk_g2s(stage + St::OFF_ST + k * (St::TP + 16), static_cast<const uint8_t*>(ptr[o]) + (p0 & ~15),
               ((uint32_t)(n + (p0 & 15)) + 15) & ~15u, full);
      if (dmat_delta != 0)
        bulk_g2s(dst, static_cast<const char*>(mat[k]) + dmat_delta, C * mat_bytes, full);
    }
  }
}

// producer-side wait before tile j may be issued: the stage must be free, and in the walk order the tile of the
// same patterns of the previous item (j - n_own) must have been consumed and fenced (it may have produced what
// this tile reads).  With n_own >= NS the first condition implies the second.
template <bool WALK>
__device__ __forceinline__ void nt_producer_wait(uint64_t* empty, int j, int n_own) {
  if (j >= NT_NS) mbar_wait(&empty[j % NT_NS], (uint32_t)((j / NT_NS - 1) & 1));
  if (WALK && n_own < NT_NS && j >= n_own) {
    const int d = j - n_own;
    mbar_wait(&empty[d % NT_NS], (uint32_t)((d / NT_NS) & 1));
  }
  if (WALK) fence_proxy_async();
}

// contribution a[s] = sum_x M[s][x] x[x] of one child to its parent, operand taken from the stage
//   KIND_STATES: column z of M (1 for a missing state)
template <typename T>
__device__ __forceinline__ void nt_contrib(int kind, const T* __restrict__ opnd, const uint8_t* __restrict__ st,
                                           const T* __restrict__ M, T a[4]) {
  if (kind == KIND_STATES) {
    const int z = *st;
#pragma unroll
    for (int s = 0; s < 4; ++s) a[s] = z < 4 ? M[s * 4 + z] : T(1);
  } else if (kind == KIND_NONE) {
#pragma unroll
    for (int s = 0; s < 4; ++s) a[s] = T(0);
  } else {
    T x[4];
    ld4(opnd, x);
    mv4<T>(M, x, a);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// post-order update + per-pattern rescaling
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C, bool WALK>
__global__ void __launch_bounds__(NT_THREADS) k_post4_tma(const DevOp* __restrict__ ops, NtSched sched) {
  using Mp = NucMap<C>;
  using St = NtStage<T, C, 2, false>;
  extern __shared__ __align__(128) unsigned char nt_smem[];
  __shared__ __align__(8) uint64_t full[NT_NS], empty[NT_NS];
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < NT_NS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], NT_CW);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  __syncthreads();
  NtTiles<Mp::PPW, St::TP> tl;
  tl.init(sched);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == NT_CW) {  // ---- producer
    if (lane == 0) {
      for (int j = 0; j < tl.J; ++j) {
        int item, p0, n, t;
        tl.tile(j, item, p0, n, t);
        nt_producer_wait<WALK>(empty, j, tl.n_own);
        const DevOp* op = ops + item;
        const void* ptr[2] = {op->child[0], op->child[1]};
        const int kind[2] = {op->kind[0], op->kind[1]};
        const void* mat[2] = {op->mat[0], op->mat[1]};
        nt_fill<T, C, 2, false>(nt_smem + (size_t)(j % NT_NS) * St::BYTES, &full[j % NT_NS], op, sizeof(DevOp), ptr,
                                kind, mat, nullptr, sched.P, p0, n);
      }
    }
    return;
  }
  // ---- consumers
  const int g = lane / Mp::PPW, pl = lane % Mp::PPW;
  const int r = warp * Mp::PPW + pl;  // pattern within the tile
  for (int j = 0; j < tl.J; ++j) {
    const int s = j % NT_NS;
    unsigned char* stage = nt_smem + (size_t)s * St::BYTES;
    mbar_wait(&full[s], (uint32_t)((j / NT_NS) & 1));
    const NtHdr h = *reinterpret_cast<const NtHdr*>(stage + St::OFF_HDR);
    const DevOp& op = *reinterpret_cast<const DevOp*>(stage + St::OFF_DESC);
    const T* sM = reinterpret_cast<const T*>(stage + St::OFF_MATS);
    const T* sX = reinterpret_cast<const T*>(stage + St::OFF_OPS);
    const uint8_t* st0 = stage + St::OFF_ST + h.soff0 + r;
    const uint8_t* st1 = stage + St::OFF_ST + (St::TP + 16) + h.soff1 + r;
    const bool live = r < h.n;
    const int p = h.p0 + r;
    const int kind0 = op.kind[0], kind1 = op.kind[1];
    T res[Mp::CPT][4];
    int key = 0;
    if (live) {
#pragma unroll
      for (int i = 0; i < Mp::CPT; ++i) {
        const int c = g * Mp::CPT + i;
        T a[4], b[4];
        nt_contrib<T>(kind0, sX + ((kind0 == KIND_BCAST ? 0 : c) * St::TP + r) * 4, st0, sM + c * St::MS, a);
        nt_contrib<T>(kind1, sX + ((C + (kind1 == KIND_BCAST ? 0 : c)) * St::TP + r) * 4, st1, sM + (C + c) * St::MS,
                      b);
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          res[i][x] = a[x] * b[x];
          key = max(key, max_key(res[i][x]));
        }
      }
    }
    void* scale = op.scale;
    T* dest = static_cast<T*>(op.dest);
    if (scale != nullptr) {
      key = group_max_int<Mp::LP>(key);
      const int e = exp_of_key(key, T(0));
      if (e != 0) {
        const T f = pow2_neg(e, T(0));
#pragma unroll
        for (int i = 0; i < Mp::CPT; ++i)
#pragma unroll
          for (int x = 0; x < 4; ++x) res[i][x] *= f;
      }
      if (live && g == 0) static_cast<int16_t*>(scale)[p] = (int16_t)e;
    }
    if (live) {
#pragma unroll
      for (int i = 0; i < Mp::CPT; ++i) st4(dest + ((size_t)(g * Mp::CPT + i) * sched.P + p) * 4, res[i]);
    }
    if (WALK) fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// pre-order update of both children of one parent fused with both branch derivatives (
// PAPER.md:43, :101).  With a_k = M_k x_k and u_k = q_m o a_{1-k}:
//   q_k = M_k^T u_k,   den = sum_c w_c q_m . (a_0 o a_1)  (the same for both children),
//   num_k = sum_c w_c r_c q_k . (Q x_k);   a compact tip takes column z of M_k and of Q instead of the products.
// Gradient partial sums: walk -> one per (item, CTA, warp), flushed after the CTA's last tile of the item;
//                        level -> one per (item, pattern tile, warp).
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int C, bool WALK>
__global__ void __launch_bounds__(NT_THREADS) k_pre4_tma(const DevPreItem* __restrict__ items, NtSched sched,
                                                         const T* __restrict__ Qg, NucModel md,
                                                         double* __restrict__ grad_partial, int n_part) {
  using Mp = NucMap<C>;
  using St = NtStage<T, C, 3, true>;
  extern __shared__ __align__(128) unsigned char nt_smem[];
  __shared__ __align__(8) uint64_t full[NT_NS], empty[NT_NS];
  __shared__ __align__(16) T sQ[16];
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < NT_NS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], NT_CW);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
  }
  if (threadIdx.x < 16) sQ[threadIdx.x] = Qg[threadIdx.x];
  __syncthreads();
  NtTiles<Mp::PPW, St::TP> tl;
  tl.init(sched);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == NT_CW) {  // ---- producer
    if (lane == 0) {
      for (int j = 0; j < tl.J; ++j) {
        int item, p0, n, t;
        tl.tile(j, item, p0, n, t);
        nt_producer_wait<WALK>(empty, j, tl.n_own);
        const DevPreItem* it = items + item;
        const void* ptr[3] = {it->qm, it->p[0], it->p[1]};
        const int kind[3] = {KIND_PARTIALS, it->kind[0], it->kind[1]};
        const void* mat[2] = {it->mat[0], it->mat[1]};
        nt_fill<T, C, 3, true>(nt_smem + (size_t)(j % NT_NS) * St::BYTES, &full[j % NT_NS], it, sizeof(DevPreItem),
                               ptr, kind, mat, md.weights, sched.P, p0, n);
      }
    }
    return;
  }
  // ---- consumers
  const int g = lane / Mp::PPW, pl = lane % Mp::PPW;
  const int r = warp * Mp::PPW + pl;
  double cw[Mp::CPT], cwr[Mp::CPT];
#pragma unroll
  for (int i = 0; i < Mp::CPT; ++i) {
    cw[i] = md.catw[g * Mp::CPT + i];
    cwr[i] = cw[i] * md.catr[g * Mp::CPT + i];
  }
  // which child's derivative this lane finishes: category group 0 -> child 0, group 1 -> child 1 (LP = 1: both)
  constexpr bool SPLIT = Mp::LP >= 2;
  double acc[2] = {0.0, 0.0};
  for (int j = 0; j < tl.J; ++j) {
    const int s = j % NT_NS;
    unsigned char* stage = nt_smem + (size_t)s * St::BYTES;
    int item, p0_, n_, t;
    tl.tile(j, item, p0_, n_, t);
    mbar_wait(&full[s], (uint32_t)((j / NT_NS) & 1));
    const NtHdr h = *reinterpret_cast<const NtHdr*>(stage + St::OFF_HDR);
    const DevPreItem& it = *reinterpret_cast<const DevPreItem*>(stage + St::OFF_DESC);
    const T* sM = reinterpret_cast<const T*>(stage + St::OFF_MATS);
    const T* sOp = reinterpret_cast<const T*>(stage + St::OFF_OPS);
    const double* sW = reinterpret_cast<const double*>(stage + St::OFF_WTS);
    const uint8_t* stp[2] = {stage + St::OFF_ST + h.soff0 + r, stage + St::OFF_ST + (St::TP + 16) + h.soff1 + r};
    const bool live = r < h.n;
    const int p = h.p0 + r;
    const int kind[2] = {it.kind[0], it.kind[1]};
    const int slot[2] = {it.slot[0], it.slot[1]};
    T* qdst[2] = {static_cast<T*>(it.q[0]), static_cast<T*>(it.q[1])};
    const bool want_grad = slot[0] >= 0 || slot[1] >= 0;
    const bool need_q[2] = {qdst[0] != nullptr || slot[0] >= 0, qdst[1] != nullptr || slot[1] >= 0};

    T q[2][Mp::CPT][4];
    int key[2] = {0, 0};
    double num[2] = {0.0, 0.0}, den = 0.0;
    if (live) {
#pragma unroll
      for (int i = 0; i < Mp::CPT; ++i) {
        const int c = g * Mp::CPT + i;
        T qm[4], a[2][4], qx[2][4];
        ld4(sOp + (c * St::TP + r) * 4, qm);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const T* Mk = sM + (k * C + c) * St::MS;
          if (kind[k] == KIND_STATES) {
            const int z = *stp[k];
#pragma unroll
            for (int x = 0; x < 4; ++x) {
              a[k][x] = z < 4 ? Mk[x * 4 + z] : T(1);
              qx[k][x] = z < 4 ? sQ[x * 4 + z] : T(0);
            }
          } else if (kind[k] == KIND_NONE) {
#pragma unroll
            for (int x = 0; x < 4; ++x) a[k][x] = qx[k][x] = T(0);
          } else {
            T x[4];
            ld4(sOp + (((k + 1) * C + (kind[k] == KIND_BCAST ? 0 : c)) * St::TP + r) * 4, x);
            mv4<T>(Mk, x, a[k]);
            if (slot[k] >= 0) mv4<T>(sQ, x, qx[k]);
          }
        }
        T u[2][4];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          u[0][x] = qm[x] * a[1][x];
          u[1][x] = qm[x] * a[0][x];
        }
        if (want_grad) {
          T dd = u[0][0] * a[0][0];
#pragma unroll
          for (int x = 1; x < 4; ++x) dd = fma(u[0][x], a[0][x], dd);
          den = fma(cw[i], (double)dd, den);
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          if (!need_q[k]) continue;
          mvt4<T>(sM + (k * C + c) * St::MS, u[k], q[k][i]);
#pragma unroll
          for (int x = 0; x < 4; ++x) key[k] = max(key[k], max_key(q[k][i][x]));
          if (slot[k] >= 0) {
            T nn = q[k][i][0] * qx[k][0];
#pragma unroll
            for (int x = 1; x < 4; ++x) nn = fma(q[k][i][x], qx[k][x], nn);
            num[k] = fma(cwr[i], (double)nn, num[k]);
          }
        }
      }
    }
    // stores of the rescaled pre-order partials (power-of-two factor, discarded: it cancels in num / den)
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      if (qdst[k] == nullptr) continue;  // uniform over the CTA
      const int e = exp_of_key(group_max_int<Mp::LP>(key[k]), T(0));
      if (live) {
        const T f = pow2_neg(e, T(0));
#pragma unroll
        for (int i = 0; i < Mp::CPT; ++i) {
          T v[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) v[x] = q[k][i][x] * f;
          st4(qdst[k] + ((size_t)(g * Mp::CPT + i) * sched.P + p) * 4, v);
        }
      }
    }
    if (want_grad) {
      den = group_sum<Mp::LP>(den);
      num[0] = group_sum<Mp::LP>(num[0]);
      num[1] = group_sum<Mp::LP>(num[1]);
      const double w = live ? sW[r] : 0.0;
      if (SPLIT) {
        const int k = g == 1 ? 1 : 0;
        const int sl = g == 1 ? slot[1] : slot[0];
        if (live && g < 2 && sl >= 0) {
          const double ratio = (g == 1 ? num[1] : num[0]) / den;
          if (md.site_out != nullptr) md.site_out[(size_t)sl * sched.P + p] = ratio;
          acc[k] = fma(w, ratio, acc[k]);
        }
      } else {
#pragma unroll
        for (int k = 0; k < 2; ++k)
          if (live && slot[k] >= 0) {
            const double ratio = num[k] / den;
            if (md.site_out != nullptr) md.site_out[(size_t)slot[k] * sched.P + p] = ratio;
            acc[k] = fma(w, ratio, acc[k]);
          }
      }
      // flush the warp's partial sums: level -> every tile; walk -> after the CTA's last tile of this item
      const bool flush = WALK ? (t == tl.n_own - 1) : true;
      if (flush) {
        const int col = WALK ? (int)blockIdx.x * NT_CW + warp : t * NT_CW + warp;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const double sum = segment_sum<Mp::PPW>(acc[k]);
          const int owner = SPLIT ? k * Mp::PPW : 0;  // first lane of the category group that accumulated child k
          if (lane == owner && slot[k] >= 0) grad_partial[(size_t)slot[k] * n_part + col] = sum;
          acc[k] = 0.0;
        }
      }
    }
    if (WALK) fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
  }
}

}  // namespace plk
