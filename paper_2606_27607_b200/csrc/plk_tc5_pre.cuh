// plk_tc5_pre.cuh -- fp32 codon (SP = 64) fused pre-order + branch-derivative kernel on tcgen05 / TMEM (sm_100a).
//
// What it computes (SURVEY 8(a) steps 5-6; PAPER.md:43 pre-order traversal, :101 "pre . Q . post" sandwich): for one
// unit (pre-order item = a parent with children 0 and 1, tile of 128 patterns), every category c, with x_k the
// post-order partials of child k, q_m the parent's pre-order partials, M_k the transition matrices, Q the rate matrix:
//     a_k = M_k x_k,  Qx_k = Q x_k                     (step A: tensor pipe, K-major B = M_k / Q)
//     u_0 = q_m o a_1,  u_1 = q_m o a_0,  den += w_c sum_s u_0[s] a_0[s]      (CUDA cores, thread = pattern row)
//     q_k = M_k^T u_k                                  (step B: tensor pipe, K-major B = M_k^T, staged from the transposed
//                                                       copies k_transpose64 writes once per pass; an MN-major TF32
//                                                       read of the M_k planes was tried and returned zeros)
//     num_k += w_c r_c sum_s q_k[s] Qx_k[s];  q_k and its per-pattern maximum are stored for internal children
// and after the last category  d_k[p] = num_k / den,  g_k += weight[p] d_k[p]  (fixed summation order).
// Arithmetic is that of k_pre_tc<float> (plk_tc.cuh): split TF32 (x = hi + lo, three products, fp32 accumulate),
// deferred power-of-two rescaling, fp64 category / pattern sums.
//
// Organisation.  One persistent CTA per SM walks a contiguous range of units.  Shared memory (192 KB): ONE operand
// stage (hi + lo planes of a 128 x 64 tile, 128-byte-swizzled K-major) that holds X_0, then X_1; M_0, M_1, Q as hi + lo
// planes (the M_k slots are re-staged with M_k^T between step A and step B); the q_m tile (raw fp32, same swizzle),
// each 4 KB slice loaded by the epilogue warp that reads it and reused as that warp's store stage.
// TMEM (512 columns): a_0, a_1, Qx_0, Qx_1, q_0, q_1 (64 each) + U_0 as hi / lo planes (128); the epilogue writes the
// split u_k with tcgen05.st -- U_1 over the a_0 / a_1 columns its thread has just consumed -- and step B reads its A
// operand from tensor memory.
// Roles (16 warps): 0-7 epilogue (warp 4h + q: patterns 32q.., states 32h..), 8-11 tile producers (X_0, X_1; the next
// tile is always in registers), 12-14 matrix stagers (Q once, M_k, M_k^T; L2 prefetch of the next round's tiles),
// 15 MMA issue.  The phases of one (unit, category) are ordered X_0 -> A -> X_1 -> A -> u -> B, B -> q_0, q_1; every
// hand-over is an mbarrier whose completions all roles count identically, and every phase arrives / commits even when
// it has nothing to do, so parities stay in step.
#pragma once
#include "plk_tc5.cuh"

namespace plk {
namespace tc5 {
namespace pre {

constexpr int EPI_W = 8, PROD_W = 4, AUX_W = 3, N_W = EPI_W + PROD_W + AUX_W + 1;  // tile producers, matrix / q_m stagers
constexpr int THREADS_PRE = N_W * 32;  // 512
constexpr int AT = AUX_W * 32;         // threads of the auxiliary stager group
constexpr uint32_t OFF_XS = 0;                        // operand stage: hi plane, lo plane
constexpr uint32_t OFF_MS = 2 * X_PLANE;              // M_0 hi, lo, M_1 hi, lo, Q hi, lo
constexpr uint32_t OFF_QM = OFF_MS + 6 * M_PLANE;     // q_m tile / store stage
constexpr uint32_t OFF_RED = OFF_QM + X_PLANE;        // doubles: [3][TP] half-1 partial sums, [2][TP] contributions
constexpr uint32_t OFF_MX = OFF_RED + 5 * TP * 8;     // floats: [TP] half-1 row maxima
constexpr uint32_t OFF_BARS = OFF_MX + TP * 4;
constexpr uint32_t SMEM_USED_PRE = OFF_BARS + 256;
constexpr size_t SMEM_BYTES_PRE = SMEM_USED_PRE + 1024;
enum { P_XFULL = 0, P_XFREE, P_UFULL, P_AFULL, P_QFULL, P_MFULL, P_MFREE, P_TFREE, P_ADONE, P_MTFULL,
       P_MTFULL1, P_MFULL1, P_M0FREE, P_TFREE0, P_TMEM_PTR, P_QFULL1 };
// TMEM columns.  U_0 (hi, lo) has its own 128 columns; U_1 (hi, lo) overwrites a_0 / a_1, which the thread that
// writes it has just consumed.
constexpr uint32_t T_A0 = 0, T_A1 = 64, T_QX0 = 128, T_QX1 = 192, T_Q0 = 256, T_Q1 = 320, T_U0 = 384;
constexpr uint32_t IDESC_BT = IDESC | (1u << 16);  // B operand MN-major: B(n = s, k = x) = M[x][s]

// MN-major B descriptor over a K-major-staged 64 x 64 plane read transposed: 32 n-values per 128-byte row, n-blocks
// LBO = 8192 B apart, 8-row k-groups SBO = 1024 B apart, 128-byte swizzle; k-step ks starts at + 1024 ks
__device__ __forceinline__ uint64_t make_desc_bt(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(8192 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
template <uint32_t ID>
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p, e;\n\t"
      "elect.sync _|e, 0xffffffff;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "@e tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(ID), "r"(accumulate)
      : "memory");
}

// out[m][x][s] = in[m][s][x] for every 64 x 64 fp32 matrix m (one block each; matrix buffers are [C][64][64] contiguous)
__global__ void __launch_bounds__(256) k_transpose64(const float* __restrict__ in, float* __restrict__ out) {
  __shared__ float tile[64][65];
  const float* src = in + (size_t)blockIdx.x * 4096;
  float* dst = out + (size_t)blockIdx.x * 4096;
  for (int i = threadIdx.x; i < 4096; i += 256) tile[i >> 6][i & 63] = src[i];
  __syncthreads();
  for (int i = threadIdx.x; i < 4096; i += 256) dst[i] = tile[i & 63][i >> 6];
}

struct PreCtx {
  const DevPreItem* items;
  int P, S, C, n_tiles;
  uint32_t n_units, u0;  // this CTA's units u0 .. u0 + n_units - 1; unit = item * n_tiles + tile
  uint32_t smem, bar;
  __device__ __forceinline__ uint32_t barrier(int slot) const { return bar + 8u * slot; }
};

// ---- producer pieces (128 threads; thread t takes chunk t % 16 of rows t / 16 + 8 j: swizzled offset off0 + 1024 j) --
__device__ __forceinline__ void pre_load_tile(const void* ptr, int kind, int c, int P, int p0, int n, int t, float4 (&r)[16]) {
  const int row0 = t >> 4;
  if (kind == KIND_PARTIALS || kind == KIND_BCAST) {
    const float* src = static_cast<const float*>(ptr) + ((kind == KIND_PARTIALS ? (size_t)c * P : 0) + p0) * SP64 + t * 4;
#pragma unroll
    for (int j = 0; j < 16; ++j) r[j] = row0 + 8 * j < n ? ldg_nc(src + j * 512) : make_float4(0.f, 0.f, 0.f, 0.f);
  } else if (kind == KIND_STATES) {
    const uint8_t* st = static_cast<const uint8_t*>(ptr) + p0 + row0;
#pragma unroll
    for (int j = 0; j < 16; ++j) r[j].x = __int_as_float(row0 + 8 * j < n ? (int)st[8 * j] : -1);
  }
}
// split into the hi / lo planes of the operand stage (one-hot rows for compact tips, hi only)
__device__ __forceinline__ void pre_store_x(uint32_t xs, int kind, int S, int t, const float4 (&r)[16]) {
  const uint32_t xhi = xs + swz_off(t >> 4, t & 15, TP), xlo = xhi + X_PLANE;
  if (kind == KIND_PARTIALS || kind == KIND_BCAST) {
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      float4 h, l;
      split4(r[j], h, l);
      sts128(xhi + 1024 * j, h);
      sts128(xlo + 1024 * j, l);
    }
  } else {
    const int x0 = (t & 15) * 4;
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const int z = kind == KIND_STATES ? __float_as_int(r[j].x) : -1;
      const bool miss = z >= S;
      float4 h;
      h.x = (z == x0 || (miss && x0 < S)) ? 1.f : 0.f;
      h.y = (z == x0 + 1 || (miss && x0 + 1 < S)) ? 1.f : 0.f;
      h.z = (z == x0 + 2 || (miss && x0 + 2 < S)) ? 1.f : 0.f;
      h.w = (z == x0 + 3 || (miss && x0 + 3 < S)) ? 1.f : 0.f;
      sts128(xhi + 1024 * j, h);
    }
  }
}
// a 64 x 64 matrix -> hi / lo planes at `ms` (1024 chunks, 8 per thread)
__device__ __forceinline__ void pre_stage_matrix(uint32_t ms, const float* M, int t) {
  float4 m[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) m[j] = ldg_nc(M + t * 4 + j * 512);
  const uint32_t mhi = ms + swz_off(t >> 4, t & 15, 64), mlo = mhi + M_PLANE;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    float4 h, l;
    split4(m[j], h, l);
    sts128(mhi + 1024 * j, h);
    sts128(mlo + 1024 * j, l);
  }
}
// the same with the 96 threads of the auxiliary group (chunks t, t + 96, ...), as a load half and a store half
__device__ __forceinline__ void aux_load_matrix(const float* M, int t, float4 (&m)[11]) {
#pragma unroll
  for (int j = 0; j < 11; ++j) {
    const int idx = t + AT * j;
    if (idx < 1024) m[j] = ldg_nc(M + idx * 4);
  }
}
__device__ __forceinline__ void aux_store_matrix(uint32_t ms, int t, const float4 (&m)[11]) {
#pragma unroll
  for (int j = 0; j < 11; ++j) {
    const int idx = t + AT * j;
    if (idx < 1024) {
      float4 h, l;
      split4(m[j], h, l);
      const uint32_t o = ms + swz_off(idx >> 4, idx & 15, 64);
      sts128(o, h);
      sts128(o + M_PLANE, l);
    }
  }
}
__device__ __forceinline__ void aux_stage_matrix(uint32_t ms, const float* M, int t) {
  float4 m[11];
  aux_load_matrix(M, t, m);
  aux_store_matrix(ms, t, m);
}
// raw fp32 tile rows p0 .. p0 + n - 1 of `src` ([.][64]) -> swizzled 128 x 64 plane at `dst` (rows beyond n: zeros)
__device__ __forceinline__ void aux_stage_tile(uint32_t dst, const float* src, int n, int t) {
#pragma unroll
  for (int b = 0; b < 2; ++b) {
    float4 v[11];
#pragma unroll
    for (int j = 0; j < 11; ++j) {
      const int idx = t + AT * (11 * b + j);
      v[j] = (idx < 2048 && (idx >> 4) < n) ? ldg_nc(src + idx * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int j = 0; j < 11; ++j) {
      const int idx = t + AT * (11 * b + j);
      if (idx < 2048) sts128(dst + swz_off(idx >> 4, idx & 15, TP), v[j]);
    }
  }
}
__device__ __forceinline__ void prefetch_tiles(const DevPreItem& it, int c, int P, int p0, int n) {
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    if (it.kind[k] == KIND_PARTIALS)
      l2_prefetch_bulk(static_cast<const float*>(it.p[k]) + ((size_t)c * P + p0) * SP64, (uint32_t)n * 256u);
    else if (it.kind[k] == KIND_BCAST)
      l2_prefetch_bulk(static_cast<const float*>(it.p[k]) + (size_t)p0 * SP64, (uint32_t)n * 256u);
  }
  l2_prefetch_bulk(static_cast<const float*>(it.qm) + ((size_t)c * P + p0) * SP64, (uint32_t)n * 256u);
}
__device__ __forceinline__ void prod_signal(uint32_t bar, int t) {
  fence_async_smem();
  __syncwarp();
  if ((t & 31) == 0) mbar_arrive(bar);
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]), "f"(v[8]), "f"(v[9]), "f"(v[10]),
      "f"(v[11]), "f"(v[12]), "f"(v[13]), "f"(v[14]), "f"(v[15])
      : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const float (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "f"(v[0]), "f"(v[1]),
               "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7])
               : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// D[tmem] (+)= A[tmem] . B[smem]^T : A = 128 lanes x 8 consecutive 32-bit columns (one k-step)
__device__ __forceinline__ void umma_ta(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p, e;\n\t"
      "elect.sync _|e, 0xffffffff;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "@e tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(IDESC), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ float scale2(uint32_t bits, const Pow2Pair<float>& f) { return (__uint_as_float(bits) * f.f1) * f.f2; }
__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, %0;" ::"n"(EPI_W * 32) : "memory"); }

// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(THREADS_PRE, 1)
    k_pre_tc5(const DevPreItem* __restrict__ items, int n_items, int P, int S, int C, const float* __restrict__ Qg,
              long long mat_t_delta,
              const double* __restrict__ catw, const double* __restrict__ catr, const double* __restrict__ weights,
              double* __restrict__ grad_partial, int n_part, double* __restrict__ site_out) {
  extern __shared__ unsigned char tc5p_smem_raw[];
  PreCtx cx;
  cx.items = items; cx.P = P; cx.S = S; cx.C = C;
  cx.n_tiles = (P + TP - 1) / TP;
  {
    const uint32_t total = (uint32_t)n_items * (uint32_t)cx.n_tiles;
    const uint32_t base = total / gridDim.x, rem = total % gridDim.x, b = blockIdx.x;
    cx.u0 = b * base + (b < rem ? b : rem);
    cx.n_units = base + (b < rem ? 1u : 0u);
  }
  if (cx.n_units == 0) return;
  cx.smem = (smem_u32(tc5p_smem_raw) + 1023u) & ~1023u;
  cx.bar = cx.smem + OFF_BARS;
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(cx.barrier(P_XFULL), PROD_W);
    mbar_init(cx.barrier(P_XFREE), 1);
    mbar_init(cx.barrier(P_UFULL), EPI_W);  // one completion per round: both U_0 and U_1 are in TMEM
    mbar_init(cx.barrier(P_AFULL), 1);
    mbar_init(cx.barrier(P_QFULL), 1);   // q_0 complete (one completion per round)
    mbar_init(cx.barrier(P_QFULL1), 1);  // q_1 complete.  Two barriers: when step B of child 1 has nothing to do both
                                         // commits land together, and a single barrier would run two phases ahead of
                                         // its waiter (an unpaired op hung here)
    mbar_init(cx.barrier(P_MFULL), AUX_W);
    mbar_init(cx.barrier(P_MFREE), 1);
    mbar_init(cx.barrier(P_TFREE), EPI_W);
    mbar_init(cx.barrier(P_ADONE), 1);
    mbar_init(cx.barrier(P_MTFULL), AUX_W);
    mbar_init(cx.barrier(P_MTFULL1), AUX_W);
    mbar_init(cx.barrier(P_MFULL1), AUX_W);
    mbar_init(cx.barrier(P_M0FREE), 1);
    mbar_init(cx.barrier(P_TFREE0), EPI_W);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == N_W - 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(cx.barrier(P_TMEM_PTR)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(cx.barrier(P_TMEM_PTR)) : "memory");
  const uint32_t xs = cx.smem + OFF_XS;

  if (warp >= EPI_W && warp < EPI_W + PROD_W) {
    // ===== tile producers: X_0 and X_1 of every (unit, category); the next tile is always in registers =====
    const int t = threadIdx.x - EPI_W * 32;
    uint32_t uc = 0;
    float4 r[16];
    {
      const DevPreItem& it = items[cx.u0 / cx.n_tiles];
      const int p0 = (int)(cx.u0 % cx.n_tiles) * TP, n = P - p0 < TP ? P - p0 : TP;
      pre_load_tile(it.p[0], it.kind[0], 0, P, p0, n, t, r);
    }
    for (uint32_t ui = 0; ui < cx.n_units; ++ui) {
      const uint32_t u = cx.u0 + ui;
      const DevPreItem& it = items[u / cx.n_tiles];
      const int p0 = (int)(u % cx.n_tiles) * TP, n = P - p0 < TP ? P - p0 : TP;
      for (int c = 0; c < C; ++c, ++uc) {
        if (uc > 0) mbar_wait(cx.barrier(P_XFREE), 1);  // completion 2 uc - 1: step B of child 1, previous round
        pre_store_x(xs, it.kind[0], S, t, r);
        prod_signal(cx.barrier(P_XFULL), t);
        pre_load_tile(it.p[1], it.kind[1], c, P, p0, n, t, r);
        mbar_wait(cx.barrier(P_XFREE), 0);  // completion 2 uc: step A of child 0
        pre_store_x(xs, it.kind[1], S, t, r);
        prod_signal(cx.barrier(P_XFULL), t);
        if (c + 1 < C) {
          pre_load_tile(it.p[0], it.kind[0], c + 1, P, p0, n, t, r);
        } else if (ui + 1 < cx.n_units) {
          const DevPreItem& nt = items[(u + 1) / cx.n_tiles];
          const int q0 = (int)((u + 1) % cx.n_tiles) * TP, m = P - q0 < TP ? P - q0 : TP;
          pre_load_tile(nt.p[0], nt.kind[0], 0, P, q0, m, t, r);
        }
      }
    }
  } else if (warp >= EPI_W + PROD_W && warp < N_W - 1) {
    // ===== auxiliary stagers: Q once, M_0 / M_1, the q_m tile, the transposed matrices; L2 prefetch of the next round =====
    const int t = threadIdx.x - (EPI_W + PROD_W) * 32;
    uint32_t uc = 0;
    for (uint32_t ui = 0; ui < cx.n_units; ++ui) {
      const uint32_t u = cx.u0 + ui;
      const DevPreItem& it = items[u / cx.n_tiles];
      const int p0 = (int)(u % cx.n_tiles) * TP, n = P - p0 < TP ? P - p0 : TP;
      for (int c = 0; c < C; ++c, ++uc) {
        if (t == 0) {
          if (c + 1 < C) {
            prefetch_tiles(it, c + 1, P, p0, n);
          } else if (ui + 1 < cx.n_units) {
            const int q0 = (int)((u + 1) % cx.n_tiles) * TP;
            prefetch_tiles(items[(u + 1) / cx.n_tiles], 0, P, q0, P - q0 < TP ? P - q0 : TP);
          }
        }
        // Slot of child 0: M_0 (step A) -> M_0^T (step B of child 0) -> M_0 of the next round as soon as that step B is
        // done (P_M0FREE), i.e. while child 1 is still in flight.  Slot of child 1: M_1 -> M_1^T -> next M_1 (P_MFREE).
        float4 mt[11];
        if (uc == 0) {
          aux_stage_matrix(cx.smem + OFF_MS + 4 * M_PLANE, Qg, t);
          aux_stage_matrix(cx.smem + OFF_MS, static_cast<const float*>(it.mat[0]) + (size_t)c * SP64 * SP64, t);
          prod_signal(cx.barrier(P_MFULL), t);
        }
        aux_load_matrix(static_cast<const float*>(it.mat[1]) + (size_t)c * SP64 * SP64, t, mt);
        if (uc > 0) mbar_wait(cx.barrier(P_MFREE), (uc - 1) & 1);
        aux_store_matrix(cx.smem + OFF_MS + 2 * M_PLANE, t, mt);
        prod_signal(cx.barrier(P_MFULL1), t);
        aux_load_matrix(reinterpret_cast<const float*>(static_cast<const char*>(it.mat[0]) + mat_t_delta) + (size_t)c * SP64 * SP64, t, mt);
        mbar_wait(cx.barrier(P_ADONE), uc & 1);
        aux_store_matrix(cx.smem + OFF_MS, t, mt);
        prod_signal(cx.barrier(P_MTFULL), t);
        aux_stage_matrix(cx.smem + OFF_MS + 2 * M_PLANE, reinterpret_cast<const float*>(static_cast<const char*>(it.mat[1]) + mat_t_delta) + (size_t)c * SP64 * SP64, t);
        prod_signal(cx.barrier(P_MTFULL1), t);
        {  // M_0 of the next round
          const DevPreItem* nt = nullptr;
          int nc = 0;
          if (c + 1 < C) {
            nt = &it;
            nc = c + 1;
          } else if (ui + 1 < cx.n_units) {
            nt = &items[(u + 1) / cx.n_tiles];
          }
          if (nt != nullptr) {
            aux_load_matrix(static_cast<const float*>(nt->mat[0]) + (size_t)nc * SP64 * SP64, t, mt);
            mbar_wait(cx.barrier(P_M0FREE), uc & 1);
            aux_store_matrix(cx.smem + OFF_MS, t, mt);
            prod_signal(cx.barrier(P_MFULL), t);
          }
        }
      }
    }
  } else if (warp == N_W - 1) {
    // ===== MMA issuer (whole warp converged; elect.sync inside the asm) =====
    const uint64_t dxhi = make_desc(xs), dxlo = make_desc(xs + X_PLANE);
    uint32_t uc = 0;
    for (uint32_t ui = 0; ui < cx.n_units; ++ui) {
      const DevPreItem& it = items[(cx.u0 + ui) / cx.n_tiles];
      const bool lo[2] = {it.kind[0] == KIND_PARTIALS || it.kind[0] == KIND_BCAST,
                          it.kind[1] == KIND_PARTIALS || it.kind[1] == KIND_BCAST};
      const bool need_q[2] = {it.q[0] != nullptr || it.slot[0] >= 0, it.q[1] != nullptr || it.slot[1] >= 0};
      for (int c = 0; c < C; ++c, ++uc) {
        // Qx_0 (first product of step A) may be overwritten once the previous round's q_0 epilogue has read it; a_0 / a_1
        // are free as soon as the previous step B has run (in-order pipe); Qx_1 waits for the q_1 epilogue further down
        if (uc > 0) mbar_wait(cx.barrier(P_TFREE0), (uc - 1) & 1);

#pragma unroll
        for (int k = 0; k < 2; ++k) {  // step A: a_k = X_k M_k^T, Qx_k = X_k Q^T
          mbar_wait(cx.barrier(k == 0 ? P_MFULL : P_MFULL1), uc & 1);
          mbar_wait(cx.barrier(P_XFULL), k);
          tc_fence_after();
#pragma unroll
          for (int ww = 0; ww < 2; ++ww) {  // w = 0: M_k, w = 1: Q.  Order Qx_0, a_0, a_1, Qx_1: the u-phase needs only the
            const int w = k == 0 ? 1 - ww : ww;  // a_k, so it is released before Qx_1 is on the pipe
            if (k == 1 && w == 1 && uc > 0) {
              mbar_wait(cx.barrier(P_TFREE), (uc - 1) & 1);
              tc_fence_after();
            }
            const uint32_t d = tmem_base + (w == 0 ? (k == 0 ? T_A0 : T_A1) : (k == 0 ? T_QX0 : T_QX1));
            const uint32_t mp = cx.smem + OFF_MS + (w == 0 ? 2 * k : 4) * M_PLANE;
            const uint64_t dmhi = make_desc(mp), dmlo = make_desc(mp + M_PLANE);
            uint32_t acc = 0;
            if (lo[k]) {
#pragma unroll
              for (int ks = 0; ks < 8; ++ks) {
                umma<IDESC>(d, dxlo + koff(ks, TP), dmhi + koff(ks, 64), acc);
                acc = 1;
              }
            }
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
              umma<IDESC>(d, dxhi + koff(ks, TP), dmlo + koff(ks, 64), acc);
              umma<IDESC>(d, dxhi + koff(ks, TP), dmhi + koff(ks, 64), 1);
              acc = 1;
            }
            if (k == 1 && w == 0) {  // a_0 and a_1 complete; M_0 / M_1 no longer read
              umma_commit(cx.barrier(P_AFULL));
              umma_commit(cx.barrier(P_ADONE));
            }
          }
          umma_commit(cx.barrier(P_XFREE));  // the producers' cue for X_1 / for X_0 of the next round
        }
        mbar_wait(cx.barrier(P_UFULL), uc & 1);
        tc_fence_after();
#pragma unroll
        for (int k = 0; k < 2; ++k) {  // step B: q_k = U_k M_k, A = U_k (hi, lo) in TMEM, B = M_k^T (K-major)
          mbar_wait(cx.barrier(k == 0 ? P_MTFULL : P_MTFULL1), uc & 1);
          tc_fence_after();
          if (need_q[k]) {
            const uint32_t d = tmem_base + (k == 0 ? T_Q0 : T_Q1);
            const uint32_t uhi = tmem_base + (k == 0 ? T_U0 : T_A0), ulo = tmem_base + (k == 0 ? T_U0 + 64 : T_A1);
            const uint32_t mp = cx.smem + OFF_MS + 2 * k * M_PLANE;
            const uint64_t bhi = make_desc(mp), blo = make_desc(mp + M_PLANE);  // M_k^T, K-major
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) umma_ta(d, ulo + 8 * ks, bhi + koff(ks, 64), (uint32_t)(ks > 0));
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
              umma_ta(d, uhi + 8 * ks, blo + koff(ks, 64), 1);
              umma_ta(d, uhi + 8 * ks, bhi + koff(ks, 64), 1);
            }
          }
          umma_commit(cx.barrier(k == 0 ? P_QFULL : P_QFULL1));
          if (k == 0) umma_commit(cx.barrier(P_M0FREE));
        }
        umma_commit(cx.barrier(P_MFREE));
      }
    }
  } else {
    // ===== epilogue: warp = 4 half + quarter; thread = pattern row 32 quarter + lane, states 32 half .. 32 half + 31 =====
    const int quarter = warp & 3, half = warp >> 2, row = 32 * quarter + lane;
    const uint32_t lane_tm = tmem_base + ((uint32_t)(32 * quarter) << 16) + 32 * half;  // + column base
    const uint32_t rowoff = (uint32_t)half * (TP * 128) + (uint32_t)row * 128;           // this row's 128-byte slice
    const uint32_t qm_row = cx.smem + OFF_QM + rowoff, xs_row = xs + rowoff;
    const uint32_t slice = cx.smem + OFF_QM + (uint32_t)half * (TP * 128) + (uint32_t)(32 * quarter) * 128;  // warp's 4 KB
    double* red = reinterpret_cast<double*>(tc5p_smem_raw + (cx.smem - smem_u32(tc5p_smem_raw)) + OFF_RED);
    float* smx = reinterpret_cast<float*>(tc5p_smem_raw + (cx.smem - smem_u32(tc5p_smem_raw)) + OFF_MX);
    uint32_t uc = 0;
    for (uint32_t ui = 0; ui < cx.n_units; ++ui) {
      const uint32_t u = cx.u0 + ui;
      const DevPreItem& it = items[u / cx.n_tiles];
      const int tile = (int)(u % cx.n_tiles), p0 = tile * TP, p = p0 + row;
      const bool want[2] = {it.slot[0] >= 0, it.slot[1] >= 0};
      const bool need_q[2] = {it.q[0] != nullptr || want[0], it.q[1] != nullptr || want[1]};
      const Pow2Pair<float> fq = pow2_pair(-pending_exp<float>(it.qm_scale, p, P, C), 0.f);
      const Pow2Pair<float> fx[2] = {pow2_pair(-pending_exp<float>(it.p_scale[0], p, P, C), 0.f),
                                     pow2_pair(-pending_exp<float>(it.p_scale[1], p, P, C), 0.f)};
      double den = 0.0, num[2] = {0.0, 0.0};
      const bool one_factor = __all_sync(0xffffffffu, fq.f2 == 1.f && fx[0].f2 == 1.f && fx[1].f2 == 1.f);
      for (int c = 0; c < C; ++c, ++uc) {
        const double cw = catw[c], cwr = catw[c] * catr[c];
        // the warp's own 32 x 32 slice of q_m, global -> shared (coalesced 128-byte row segments), under step A
        {
          const float* src = static_cast<const float*>(it.qm) + ((size_t)c * P + p0 + 32 * quarter) * SP64 + 32 * half;
          float4 v[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int idx = j * 32 + lane, r = idx >> 3, ch = idx & 7;
            v[j] = (p0 + 32 * quarter + r < P) ? ldg_nc(src + (size_t)r * SP64 + ch * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int idx = j * 32 + lane, r = idx >> 3, ch = idx & 7;
            sts128(slice + (uint32_t)r * 128 + (uint32_t)((ch ^ (r & 7)) << 4), v[j]);
          }
          __syncwarp();
        }
        mbar_wait(cx.barrier(P_AFULL), uc & 1);
        tc_fence_after();
        // ---- u_0 = q_m o a_1, u_1 = q_m o a_0 (split, straight into TMEM as the A operands of step B), den
        float dd = 0.f;
#pragma unroll
        for (int sub = 0; sub < 4; ++sub) {  // 8 states at a time keeps the split operands in registers
          uint32_t a0[8], a1[8];
          tmem_ld8(lane_tm + T_A0 + 8 * sub, a0);
          tmem_ld8(lane_tm + T_A1 + 8 * sub, a1);
          float qm[8];
#pragma unroll
          for (int q = 0; q < 2; ++q) {
            const float4 qv = lds128(qm_row + (uint32_t)(((2 * sub + q) ^ (row & 7)) << 4));
            qm[4 * q] = qv.x; qm[4 * q + 1] = qv.y; qm[4 * q + 2] = qv.z; qm[4 * q + 3] = qv.w;
          }
          tmem_ld_wait();
          float u0h[8], u0l[8], u1h[8], u1l[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            float s0, s1, qs;
            if (one_factor) {  // the usual case: every pending exponent fits one power-of-two factor
              s0 = __uint_as_float(a0[j]) * fx[0].f1;
              s1 = __uint_as_float(a1[j]) * fx[1].f1;
              qs = qm[j] * fq.f1;
            } else {
              s0 = scale2(a0[j], fx[0]);
              s1 = scale2(a1[j], fx[1]);
              qs = (qm[j] * fq.f1) * fq.f2;
            }
            const float u0 = qs * s1, u1 = qs * s0;
            dd = fmaf(u0, s0, dd);
            u0h[j] = tf32_hi(u0);
            u0l[j] = u0 - u0h[j];
            u1h[j] = tf32_hi(u1);
            u1l[j] = u1 - u1h[j];
          }
          tmem_st8(lane_tm + T_U0 + 8 * sub, u0h);
          tmem_st8(lane_tm + T_U0 + 64 + 8 * sub, u0l);
          tmem_st8(lane_tm + T_A0 + 8 * sub, u1h);
          tmem_st8(lane_tm + T_A1 + 8 * sub, u1l);
        }
        den = fma(cw, (double)dd, den);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(cx.barrier(P_UFULL));
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          mbar_wait(cx.barrier(k == 0 ? P_QFULL : P_QFULL1), uc & 1);
          tc_fence_after();
          float mx = 0.f;
          if (need_q[k]) {
            float nn = 0.f;
#pragma unroll
            for (int sub = 0; sub < 2; ++sub) {
              uint32_t qk[16], qx[16];
              tmem_ld16(lane_tm + (k == 0 ? T_Q0 : T_Q1) + 16 * sub, qk);
              tmem_ld16(lane_tm + (k == 0 ? T_QX0 : T_QX1) + 16 * sub, qx);
              tmem_ld_wait();
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                float v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  v[j] = __uint_as_float(qk[4 * q + j]);
                  mx = fmaxf(mx, v[j]);
                  nn = fmaf(v[j], scale2(qx[4 * q + j], fx[k]), nn);
                }
                if (it.q[k] != nullptr)  // stage for the coalesced store (the q_m slice is dead by now)
                  sts128(qm_row + (uint32_t)(((4 * sub + q) ^ (row & 7)) << 4), make_float4(v[0], v[1], v[2], v[3]));
              }
            }
            if (want[k]) num[k] = fma(cwr, (double)nn, num[k]);
          }
          tc_fence_before();
          __syncwarp();  // q_k and Qx_k of this round have been read: their columns may be overwritten
          if (lane == 0) mbar_arrive(cx.barrier(k == 0 ? P_TFREE0 : P_TFREE));
          if (it.q[k] != nullptr) {
            if (half == 1) smx[row] = mx;
            __syncwarp();
            float* dest = static_cast<float*>(it.q[k]) + ((size_t)c * P + p0 + 32 * quarter) * SP64 + 32 * half;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const int idx = j * 32 + lane, r = idx >> 3, ch = idx & 7;
              const float4 v = lds128(slice + (uint32_t)r * 128 + (uint32_t)((ch ^ (r & 7)) << 4));
              if (p0 + 32 * quarter + r < P) *reinterpret_cast<float4*>(dest + (size_t)r * SP64 + ch * 4) = v;
            }
            epi_bar();
            if (half == 0 && p < P) static_cast<float*>(it.q_scale[k])[(size_t)c * P + p] = fmaxf(mx, smx[row]);
            epi_bar();  // smx and the slices are free again
          }
        }
        __syncwarp();

      }
      // ---- per-pattern derivative and the tile's contribution to each gradient (fixed order)
      if (want[0] || want[1]) {
        if (half == 1) {
          red[row] = den;
          red[TP + row] = num[0];
          red[2 * TP + row] = num[1];
        }
        epi_bar();
        if (half == 0) {
          const double d = den + red[row];
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            double contrib = 0.0;
            if (want[k] && p < P) {
              const double ratio = (num[k] + red[(1 + k) * TP + row]) / d;
              if (site_out != nullptr) site_out[(size_t)it.slot[k] * P + p] = ratio;
              contrib = weights[p] * ratio;
            }
            red[(3 + k) * TP + row] = contrib;
          }
        }
        epi_bar();
        if (warp < 2 && want[warp]) {
          double v = 0.0;
          for (int i = lane; i < TP; i += 32) v += red[(3 + warp) * TP + i];
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
          if (lane == 0) grad_partial[(size_t)it.slot[warp] * n_part + tile] = v;
        }
        epi_bar();
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == N_W - 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

// returns the number of partial sums per gradient slot through *n_parts (row stride stays n_part)
inline int launch_pre(cudaStream_t stream, const DevPreItem* d_items, int n, int P, int S, int C, const float* Q,
                      long long mat_t_delta,
                      const double* catw, const double* catr, const double* weights, double* grad_partial, int n_part,
                      double* site, int sm_count, int* n_parts, int64_t* launches) {
  // per device and cheap: no process-wide "done" flag (instances may live on several GPUs)
  if (cudaFuncSetAttribute(k_pre_tc5, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES_PRE) != cudaSuccess)
    return PLK_ERR_CUDA;
  const int n_tiles = (P + TP - 1) / TP;
  *n_parts = n_tiles;
  const long long total = (long long)n * n_tiles;
  if (total <= 0) return PLK_SUCCESS;
  const int grid = total < sm_count ? (int)total : sm_count;
  k_pre_tc5<<<grid, THREADS_PRE, SMEM_BYTES_PRE, stream>>>(d_items, n, P, S, C, Q, mat_t_delta, catw, catr, weights, grad_partial, n_part,
                                                            site);
  if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
  ++*launches;
  return PLK_SUCCESS;
}

}  // namespace pre
}  // namespace tc5
}  // namespace plk
