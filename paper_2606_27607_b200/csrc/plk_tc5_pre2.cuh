// plk_tc5_pre2.cuh -- fp32 codon (SP = 64) fused pre-order + branch-derivative kernels, class-specialised and
// pipelined (sm_100a: tcgen05 / TMEM).  The general kernel of plk_tc5_pre.cuh stays for every other item shape.
//
// What is computed for a parent m with children 0, 1, per pattern p and
// category c, with x_k the post-order partials of child k, q_m the parent's pre-order partials, M_k the transition
// matrices and D_k = M_k Q the derivative matrices (k_prep_matrices64, once per pass):
//     a_k = M_k x_k,  b_k = D_k x_k                      (step A)
//     u_0 = q_m o a_1,  u_1 = q_m o a_0                   (elementwise)
//     den_c = sum_s u_0[s] a_0[s],   num_{k,c} = sum_s u_k[s] b_k[s]   (= q_k^T Q x_k, since q_k = M_k^T u_k)
//     q_k = M_k^T u_k    only for children whose pre-order partials are STORED (internal children) (step B)
// and, in k_grad64_finish,  d_k[p] = sum_c w_c r_c num_{k,c} / sum_c w_c den_c,  g_k = sum_p weight[p] d_k[p].
// Arithmetic: split TF32 (x = hi + lo, three products, fp32 accumulate; plk_tc5.cuh), deferred power-of-two
// rescaling, fp64 category / pattern sums.
//
// Item classes (the host sorts each dependency level, as for the 4-state kernels):
//   k_pre_tc5v<0>   both children internal (partials in, both q_k stored)
//   k_pre_tc5v<1>   child 0 internal, child 1 a compact tip: a_1 = M_1[:, z], b_1 = D_1[:, z] are row gathers from
//                   transposed tables in shared memory -- a tip edge costs no tensor work and no q_k
//   k_grad64_tips   both children compact tips: CUDA cores only, reads q_m and nothing else
//
// Why it is organised this way (measured on the first version, profiles/r01_codon_pre_tc5_fp32.txt: tensor pipe 24 %
// active, every phase of a (tile, category) round serial).  Shared memory cannot hold two rounds' operands, so:
//   * the X_k tiles never touch the tensor pipe's shared-memory port: producers transpose them through a small
//     buffer, split them and write hi / lo straight into TENSOR MEMORY (tcgen05.st); step A reads its A operand from
//     TMEM.  Shared memory then holds nothing but matrices: [M_0; D_0], [M_1; D_1] (step A, N = 128 stacked so a_k and
//     b_k come out of one product) and M_0^T, M_1^T (step B) as hi + lo planes = 192 KB, RESIDENT for a whole
//     (item, category) segment: rounds are ordered (item, category, tile) with the tile fastest, and the per-category
//     num / den go through a small fp32 scratch ([slot][C][P]) that k_grad64_finish reduces over categories.
//   * every product is issued in two N-halves (states 0..31, 32..63): the epilogue forms u for half 0 while the
//     tensor pipe computes half 1, and step B (K split the same way) of half 0 runs while u of half 1 is formed.
//     u is written IN PLACE over the a / b columns its thread has just read.
//   * the two X regions of TMEM play ping-pong: in round r the child f = r & 1 is issued first and BOTH q_k of the
//     round are accumulated in ITS (dead) X region, so the other region is free as soon as the second child's step A
//     has run -- the first tile of round r + 1 is stored there during this round's step B, and the second one during
//     the first child's step A of round r + 1.  No tile store sits on the critical path.
// TMEM (512 columns): region 0 = 0..127, region 1 = 128..255 (X_k hi | lo, later q_0 | q_1), [a_0|b_0] halves
// 256..383, [a_1|b_1] halves 384..511.
// Roles (14 warps): 0-7 epilogue (warp = quarter + 4 sub: TMEM lanes 32 quarter.., 16 of the 32 states of a half),
// 8-11 producers (warp w owns pattern rows 32 (w - 8)..; the next tile is always in registers and the ones after it
// are prefetched into L2), 12 MMA issue + TMEM allocation, 13 "meta": the per-row pending exponents (deferred
// rescaling) and tip states of the next two rounds, handed to the epilogue through shared memory.
// Round 2 measurements that shaped it (clock64 traces of one CTA, configs[3]): (i) the epilogue warps used to load
// those per-row scalars themselves -- twelve scattered DRAM loads per thread whose scoreboard every later wait of the
// warp inherited: 4.5 k of a round's 24 k cycles; (ii) the hi / lo split went through cvt.rna.tf32 twice per element
// in producers and epilogue, and the conversion unit was the bottleneck of both: hi is now the value with its 13 low
// mantissa bits masked off and lo one exact subtraction (tf32_hi, plk_tc5.cuh).  Together: 8.53 -> 6.50 ms per pass.
#pragma once
#include "plk_tc5_pre.cuh"

namespace plk {
namespace tc5 {
namespace pre2 {

using pre::tmem_ld8;
using pre::tmem_st8;
using pre::tmem_st_wait;
using pre::umma_ta;

constexpr int EPI_W = 8, PROD_W = 4, N_W = EPI_W + PROD_W + 1;
constexpr int META_W = N_W;                     // warp 13: per-row scalars of the next rounds (see the kernel)
constexpr int THREADS = (N_W + 1) * 32;         // 448
constexpr int STAGERS = (EPI_W + PROD_W) * 32;  // 384 threads stage the matrices of a segment
constexpr uint32_t PLANE_A = 128 * 64 * 4;   // one plane (hi or lo) of a stacked [M_k; D_k] operand: 128 rows
constexpr uint32_t OFF_MAT0 = 0, OFF_MAT1 = 2 * PLANE_A;        // [M_k; D_k] hi, lo  (class 1: raw tip tables at MAT1)
constexpr uint32_t OFF_MT0 = 4 * PLANE_A, OFF_MT1 = OFF_MT0 + 2 * M_PLANE;  // M_k^T hi, lo
constexpr uint32_t OFF_XT = OFF_MT1 + 2 * M_PLANE;              // producers' transposition buffers, 2 KB per warp
constexpr uint32_t OFF_QS = OFF_XT + PROD_W * 2048;             // epilogue staging (q_m in, q_k out), 2 KB per warp
constexpr uint32_t OFF_RED = OFF_QS + EPI_W * 2048;             // floats [2 parity][3][TP]: sub-1 partial sums
constexpr uint32_t OFF_SMX = OFF_RED + 2 * 3 * TP * 4;          // floats [2 parity][2 child][TP]: sub-1 row maxima
constexpr uint32_t OFF_EXP = OFF_SMX + 2 * 2 * TP * 4;           // ints [2 parity][3][TP]: pending exponents of q_m, x_0, x_1 (class 1: tip state)
constexpr uint32_t OFF_ITEM = OFF_EXP + 2 * 3 * TP * 4;          // the segment's item descriptor (one L2 round trip per segment)
constexpr uint32_t OFF_BAR2 = OFF_ITEM + 128;
constexpr uint32_t SMEM_USED2 = OFF_BAR2 + 256;
static_assert(sizeof(DevPreItem) <= 128, "item descriptor slot");
constexpr size_t SMEM_BYTES2 = SMEM_USED2 + 1024;
constexpr int TAB_LD = 68;                                      // class 1 tip tables: row stride (floats)
constexpr uint32_t TAB_BYTES = 65 * TAB_LD * 4;                 // 64 state rows + 1 "missing" row (sum of the others)
static_assert(2 * TAB_BYTES <= 2 * PLANE_A, "tip tables fit the [M_1; D_1] slot");
static_assert(SMEM_BYTES2 <= 232448, "shared memory budget");

// every barrier completes exactly once per round (MATFULL / MATFREE: once per segment)
enum { B_XFULL_A = 0,  // first tile of the round stored (producers); class 1: even rounds
       B_XFULL_B,      // second tile stored (class 0); class 1: the tile of odd rounds
       B_REGFREE,      // the second child's step A has run: its X region is free (commit)
       B_QREAD,        // the epilogue has read the round's q_k: the region they sat in is free
       B_QREAD1,       // class 1 only: rounds alternate between B_QREAD (even) and B_QREAD1 (odd), see the producers
       B_AFULL0, B_AFULL1, B_UFULL0, B_UFULL1, B_QFULL, B_MATFULL, B_MATFREE,
       B_EXPFULL, B_EXPFULL1,  // the round's pending exponents are in shared memory (meta warp): even / odd rounds, so that
                               // the writer may run two rounds ahead of the readers without wrapping a phase parity
       B_EXPFREE, B_EXPFREE1,  // the epilogue has read them (even / odd rounds)
       B_TMEM };
constexpr uint32_t T_REG = 128, T_AB0 = 256, T_AB1 = 384;  // X region r at T_REG * r: hi 0..63, lo 64..127

// byte deltas from a transition-matrix buffer to its derived copies (all inside the instance arena)
struct MatDeltas {
  long long d, t, dt;  // D = M Q;  M^T;  D^T
};

// ---- once per gradient pass: D = M Q, M^T, D^T for every matrix buffer and category (one block per 64 x 64 matrix) ----
__global__ void __launch_bounds__(256) k_prep_matrices64(const float* __restrict__ mats, const float* __restrict__ Q,
                                                         float* __restrict__ out_d, float* __restrict__ out_t,
                                                         float* __restrict__ out_dt) {
  // operands widened ONCE on the way into shared memory (the product loop used to convert both operands of every
  // FMA: half a million conversions per block on the slow conversion unit)
  __shared__ double sM[64][64];                             // broadcast reads only: no padding needed
  float(*sD)[65] = reinterpret_cast<float(*)[65]>(sM);     // D, written over M once every product is done
  const float* M = mats + (size_t)blockIdx.x * 4096;
  for (int i = threadIdx.x; i < 4096; i += 256) {
    const float v = M[i];
    sM[i >> 6][i & 63] = (double)v;
    out_t[(size_t)blockIdx.x * 4096 + (i & 63) * 64 + (i >> 6)] = v;
  }
  __syncthreads();
  // thread (col = tid & 63, g = tid >> 6) forms D[r][col] for its 16 rows r = g + 4 i at once: one element of Q
  // (converted once) serves 16 FMAs; the M operands are broadcast reads from shared memory; fp64 accumulation
  const int col = threadIdx.x & 63, g = threadIdx.x >> 6;
  double acc[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) acc[i] = 0.0;
#pragma unroll 4
  for (int k = 0; k < 64; ++k) {
    const double qk = (double)__ldg(Q + k * 64 + col);
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = fma(sM[g + 4 * i][k], qk, acc[i]);
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const float d = (float)acc[i];
    sD[g + 4 * i][col] = d;
    out_d[(size_t)blockIdx.x * 4096 + (g + 4 * i) * 64 + col] = d;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4096; i += 256) out_dt[(size_t)blockIdx.x * 4096 + i] = sD[i & 63][i >> 6];
}

// (item, category, tile) of a round, advanced incrementally (no division in the round loops)
struct Cur {
  int item, c, tile;
};
struct Ctx2 {
  const DevPreItem* items;
  int P, S, C, n_tiles;
  uint32_t n_rounds, r0;  // this CTA's rounds r0 .. r0 + n_rounds - 1; round = (item * C + c) * n_tiles + tile
  uint32_t smem, bar;
  __device__ __forceinline__ uint32_t barrier(int slot) const { return bar + 8u * slot; }
  __device__ __forceinline__ Cur first() const {
    Cur k;
    k.tile = (int)(r0 % (uint32_t)n_tiles);
    const uint32_t ic = r0 / (uint32_t)n_tiles;
    k.c = (int)(ic % (uint32_t)C);
    k.item = (int)(ic / (uint32_t)C);
    return k;
  }
  __device__ __forceinline__ void advance(Cur& k) const {
    if (++k.tile == n_tiles) {
      k.tile = 0;
      if (++k.c == C) {
        k.c = 0;
        ++k.item;
      }
    }
  }
  __device__ __forceinline__ Cur next(Cur k) const {
    advance(k);
    return k;
  }
};

__device__ __forceinline__ void stagers_bar() { asm volatile("bar.sync 2, %0;" ::"n"(STAGERS) : "memory"); }
__device__ __forceinline__ void epi_bar2() { asm volatile("bar.sync 1, %0;" ::"n"(EPI_W * 32) : "memory"); }

// 64-byte rows of a 2 KB transposition buffer, 16-byte chunk j of row r stored at chunk j ^ ((r >> 1) & 3): both the
// coalesced side (4 lanes per row) and the row side (lane = row) hit 8 distinct 16-byte bank groups per quarter warp
__device__ __forceinline__ uint32_t xt_off(int r, int j) { return (uint32_t)(r * 64 + ((j ^ ((r >> 1) & 3)) << 4)); }

// Stage the matrices of segment (item, c): called by the 384 stager threads (t = 0..383).
template <int CLS>
__device__ __forceinline__ void stage_segment(const Ctx2& cx, const DevPreItem& it, int c, const MatDeltas& md, int t) {
  const size_t co = (size_t)c * SP64 * SP64;
#pragma unroll 1
  for (int k = 0; k < (CLS == 0 ? 2 : 1); ++k) {
    const float* Mk = static_cast<const float*>(it.mat[k]) + co;
    const float* Dk = reinterpret_cast<const float*>(static_cast<const char*>(it.mat[k]) + md.d) + co;
    const float* Tk = reinterpret_cast<const float*>(static_cast<const char*>(it.mat[k]) + md.t) + co;
    const uint32_t mat = cx.smem + (k == 0 ? OFF_MAT0 : OFF_MAT1), mt = cx.smem + (k == 0 ? OFF_MT0 : OFF_MT1);
    // [M_k; D_k] stacked by N-halves: rows 64 h + j = M_k row 32 h + j, rows 64 h + 32 + j = D_k row 32 h + j
    for (int id = t; id < 2048; id += STAGERS) {
      const int R = id >> 4, ch = id & 15;
      const float* src = ((R & 32) ? Dk : Mk) + (((R >> 6) << 5) + (R & 31)) * SP64 + ch * 4;
      float4 h, l;
      split4(ldg_nc(src), h, l);
      const uint32_t o = mat + swz_off(R, ch, 128);
      sts128(o, h);
      sts128(o + PLANE_A, l);
    }
    for (int id = t; id < 1024; id += STAGERS) {  // M_k^T: the K-major B operand of step B
      const int R = id >> 4, ch = id & 15;
      float4 h, l;
      split4(ldg_nc(Tk + R * SP64 + ch * 4), h, l);
      const uint32_t o = mt + swz_off(R, ch, 64);
      sts128(o, h);
      sts128(o + M_PLANE, l);
    }
  }
  if (CLS == 1) {  // tip child 1: raw transposed tables, row z = column z of M_1 / D_1
    const float* T1 = reinterpret_cast<const float*>(static_cast<const char*>(it.mat[1]) + md.t) + co;
    const float* DT1 = reinterpret_cast<const float*>(static_cast<const char*>(it.mat[1]) + md.dt) + co;
    for (int id = t; id < 2048; id += STAGERS) {
      const int which = id >> 10, z = (id >> 4) & 63, ch = id & 15;
      const float4 v = ldg_nc((which ? DT1 : T1) + z * SP64 + ch * 4);
      sts128(cx.smem + OFF_MAT1 + which * TAB_BYTES + (uint32_t)(z * TAB_LD + ch * 4) * 4, v);
    }
  }
}
// class 1: row 64 of each table = sum of the state rows (a missing tip state contributes every state: SURVEY 8(c) row 15)
__device__ __forceinline__ void finish_tip_tables(const Ctx2& cx, int t) {
  if (t < 128) {
    const uint32_t tab = cx.smem + OFF_MAT1 + (t >> 6) * TAB_BYTES;
    const int col = t & 63;
    float s = 0.f;
    for (int z = 0; z < 64; ++z) s += lds32(tab + (uint32_t)(z * TAB_LD + col) * 4);
    sts32(tab + (uint32_t)(64 * TAB_LD + col) * 4, s);
  }
}

// ---------------------------------------------------------------------------------------------------------------
template <int CLS>
__global__ void __launch_bounds__(THREADS, 1)
    k_pre_tc5v(const DevPreItem* __restrict__ items, int n_items, int P, int S, int C, MatDeltas md,
               float* __restrict__ scratch /* [slot][num, den][C][P] */) {
  extern __shared__ unsigned char tc5v_smem_raw[];
  Ctx2 cx;
  cx.items = items; cx.P = P; cx.S = S; cx.C = C;
  cx.n_tiles = (P + TP - 1) / TP;
  {
    const uint32_t total = (uint32_t)n_items * (uint32_t)C * (uint32_t)cx.n_tiles;
    const uint32_t base = total / gridDim.x, rem = total % gridDim.x, b = blockIdx.x;
    cx.r0 = b * base + (b < rem ? b : rem);
    cx.n_rounds = base + (b < rem ? 1u : 0u);
  }
  if (cx.n_rounds == 0) return;
  cx.smem = (smem_u32(tc5v_smem_raw) + 1023u) & ~1023u;
  cx.bar = cx.smem + OFF_BAR2;
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(cx.barrier(B_XFULL_A), PROD_W);
    mbar_init(cx.barrier(B_XFULL_B), PROD_W);
    mbar_init(cx.barrier(B_REGFREE), 1);
    mbar_init(cx.barrier(B_QREAD), CLS == 0 ? 2 * EPI_W : EPI_W);  // class 0: one arrival per warp and q_k
    mbar_init(cx.barrier(B_QREAD1), EPI_W);
    mbar_init(cx.barrier(B_AFULL0), 1);
    mbar_init(cx.barrier(B_AFULL1), 1);
    mbar_init(cx.barrier(B_UFULL0), EPI_W);
    mbar_init(cx.barrier(B_UFULL1), EPI_W);
    mbar_init(cx.barrier(B_QFULL), 1);
    mbar_init(cx.barrier(B_MATFULL), 1);
    mbar_init(cx.barrier(B_MATFREE), 1);
    mbar_init(cx.barrier(B_EXPFULL), 1);
    mbar_init(cx.barrier(B_EXPFULL1), 1);
    mbar_init(cx.barrier(B_EXPFREE), EPI_W);
    mbar_init(cx.barrier(B_EXPFREE1), EPI_W);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == N_W - 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(cx.barrier(B_TMEM)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem) : "r"(cx.barrier(B_TMEM)) : "memory");
  // Round ui: class 0 issues child f = ui & 1 first, its X tile lives in region f, the other child's in region 1 - f;
  // class 1 has one tile per round (child 0), in region ui & 1.  The round's q_0 | q_1 accumulate in region ui & 1.

  if (warp == N_W - 1) {
    // ===== MMA issue (whole warp converged; elect.sync inside the asm) =====
    uint32_t seg = 0;
    // step A, child k (tile in region reg), N-half h: [a_kh | b_kh] = X_k . [M_k; D_k]_h^T   (A from TMEM, three split passes)
    auto step_a = [&](int k, uint32_t reg, int h) {
      const uint32_t d = tmem + (k ? T_AB1 : T_AB0) + 64 * h;
      const uint32_t xh = tmem + T_REG * reg, xl = xh + 64;
      const uint32_t mp = cx.smem + (k ? OFF_MAT1 : OFF_MAT0) + (uint32_t)h * (64 * 128);
      const uint64_t bhi = make_desc(mp), blo = make_desc(mp + PLANE_A);
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) umma_ta(d, xl + 8 * ks, bhi + koff(ks, 128), (uint32_t)(ks > 0));
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) {
        umma_ta(d, xh + 8 * ks, blo + koff(ks, 128), 1);
        umma_ta(d, xh + 8 * ks, bhi + koff(ks, 128), 1);
      }
    };
    // step B, child k, K-half h: q_k (+)= U_kh . (M_k^T)[:, 32 h ..]^T   (U hi | lo in place of a_kh | b_kh)
    auto step_b = [&](int k, uint32_t qreg, int h) {
      const uint32_t d = tmem + T_REG * qreg + 64 * k;
      const uint32_t uh = tmem + (k ? T_AB1 : T_AB0) + 64 * h, ul = uh + 32;
      const uint32_t mp = cx.smem + (k ? OFF_MT1 : OFF_MT0);
      const uint64_t bhi = make_desc(mp), blo = make_desc(mp + M_PLANE);
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) umma_ta(d, ul + 8 * ks, bhi + koff(4 * h + ks, 64), (uint32_t)(h > 0 || ks > 0));
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) {
        umma_ta(d, uh + 8 * ks, blo + koff(4 * h + ks, 64), 1);
        umma_ta(d, uh + 8 * ks, bhi + koff(4 * h + ks, 64), 1);
      }
    };
    int tile = cx.first().tile;  // the MMA warp needs the segment boundaries only
    for (uint32_t ui = 0; ui < cx.n_rounds; ++ui) {
      const uint32_t par = ui & 1;
      if (ui == 0 || tile == 0) {
        mbar_wait(cx.barrier(B_MATFULL), seg & 1);
        ++seg;
      }
      if (++tile == cx.n_tiles) tile = 0;
      // Class 1 has no wait that ties a producer warp to the CURRENT round (its next store only needs the q_0 of two
      // rounds ago to have been read), so a fast warp may be one round ahead of a slow one: with a single barrier its
      // arrival for round ui + 1 would complete the phase of round ui without the slow warp's rows (seen as rare
      // last-bits differences between repeated evaluations, a few rows of one quarter of a tile).  Even and odd rounds
      // therefore arrive on two barriers, as for QREAD / QREAD1.
      if (CLS == 0) mbar_wait(cx.barrier(B_XFULL_A), par);
      else mbar_wait(cx.barrier(par ? B_XFULL_B : B_XFULL_A), (ui >> 1) & 1);
      tc_fence_after();
      if (CLS == 0) {
        const int f = (int)par;  // first child = region index
        step_a(f, par, 0);
        step_a(f, par, 1);
        mbar_wait(cx.barrier(B_XFULL_B), par);
        tc_fence_after();
        step_a(1 - f, par ^ 1, 0);
        umma_commit(cx.barrier(B_AFULL0));
        step_a(1 - f, par ^ 1, 1);
        umma_commit(cx.barrier(B_AFULL1));
        umma_commit(cx.barrier(B_REGFREE));  // region 1 - f is dead: next round's first tile may be stored
      } else {
        step_a(0, par, 0);
        umma_commit(cx.barrier(B_AFULL0));
        step_a(0, par, 1);
        umma_commit(cx.barrier(B_AFULL1));
      }
      mbar_wait(cx.barrier(B_UFULL0), par);
      tc_fence_after();
      step_b(0, par, 0);
      if (CLS == 0) step_b(1, par, 0);
      mbar_wait(cx.barrier(B_UFULL1), par);
      tc_fence_after();
      step_b(0, par, 1);
      if (CLS == 0) step_b(1, par, 1);
      umma_commit(cx.barrier(B_QFULL));
      if (ui + 1 == cx.n_rounds || tile == 0) umma_commit(cx.barrier(B_MATFREE));  // last round of its segment
    }
  } else if (warp == META_W) {
    // ===== meta warp: pending per-pattern exponents (deferred rescaling) of q_m, child 0, child 1 -- class 1: the tip
    // state of child 1 -- of every row of a round, up to two rounds ahead, handed to the epilogue through shared memory.
    // (The epilogue warps used to load them themselves: twelve scattered DRAM loads per thread whose scoreboard every
    // later wait of the warp inherited -- 4.5 k of the 24 k cycles of a round; on the producer warps they delayed the
    // tile stores.  This warp has nothing else to wait for.)
    int* sexp = reinterpret_cast<int*>(tc5v_smem_raw + (cx.smem - smem_u32(tc5v_smem_raw)) + OFF_EXP);
    auto ldv = [](const float* m) {
      float v;
      asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(m));
      return v;
    };
    // the first four categories of src[.][pp] as independent loads (all of a round's loads are issued before the first
    // of them is used); further categories, if any, in a tail loop
    auto load4 = [&](const void* src, int pp) {
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (src != nullptr && pp < P) {
        const float* m = static_cast<const float*>(src) + pp;
        v.x = ldv(m);
        if (C > 1) v.y = ldv(m + (size_t)P);
        if (C > 2) v.z = ldv(m + 2 * (size_t)P);
        if (C > 3) v.w = ldv(m + 3 * (size_t)P);
      }
      return v;
    };
    auto finish4 = [&](const float4 r4, const void* src, int pp) {
      float v = fmaxf(fmaxf(r4.x, r4.y), fmaxf(r4.z, r4.w));
      if (C > 4 && src != nullptr && pp < P)
        for (int cc = 4; cc < C; ++cc) v = fmaxf(v, static_cast<const float*>(src)[(size_t)cc * P + pp]);
      return exp_of(v);
    };
    Cur k = cx.first();
    for (uint32_t ui = 0; ui < cx.n_rounds; ++ui, cx.advance(k)) {
      const uint32_t par = ui & 1;
      const DevPreItem& t = items[k.item];
      const void* src[3] = {t.qm_scale, t.p_scale[0], CLS == 0 ? t.p_scale[1] : nullptr};
      float4 raw[4][3];
      int z[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int pp = k.tile * TP + lane + 32 * j;
#pragma unroll
        for (int e = 0; e < (CLS == 0 ? 3 : 2); ++e) raw[j][e] = load4(src[e], pp);
        z[j] = 64;
        if (CLS == 1 && pp < P) asm volatile("ld.global.nc.u8 %0, [%1];" : "=r"(z[j]) : "l"(static_cast<const uint8_t*>(t.p[1]) + pp));
      }
      int ex[4][3];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int pp = k.tile * TP + lane + 32 * j;
        ex[j][0] = finish4(raw[j][0], src[0], pp);
        ex[j][1] = finish4(raw[j][1], src[1], pp);
        ex[j][2] = CLS == 0 ? finish4(raw[j][2], src[2], pp) : z[j];
      }
      if (ui > 1) mbar_wait(cx.barrier(par ? B_EXPFREE1 : B_EXPFREE), ((ui >> 1) + 1) & 1);  // round ui - 2 was read
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int e = 0; e < 3; ++e) sexp[(par * 3 + e) * TP + lane + 32 * j] = ex[j][e];
      __syncwarp();
      if (lane == 0) mbar_arrive(cx.barrier(par ? B_EXPFULL1 : B_EXPFULL));
    }
  } else {
    const int st = (int)threadIdx.x;  // stager index 0..383 (warps 0..11)
    uint32_t seg = 0;
    // segment boundary, executed by all 12 stager warps in program order with their rounds
    const DevPreItem* sit = reinterpret_cast<const DevPreItem*>(tc5v_smem_raw + (cx.smem - smem_u32(tc5v_smem_raw)) + OFF_ITEM);
    int staged_item = -1;
    // the descriptor of item i: the shared-memory copy while i is the staged segment's item, else global memory (only a
    // look-ahead across a segment boundary takes that path)
    auto item_of = [&](int i) -> const DevPreItem& { return i == staged_item ? *sit : items[i]; };
    auto segment_start = [&](const Cur& k) {
      stagers_bar();  // nobody still reads the previous segment's tip tables or item descriptor
      if (st < (int)(sizeof(DevPreItem) / 4))
        reinterpret_cast<uint32_t*>(tc5v_smem_raw + (cx.smem - smem_u32(tc5v_smem_raw)) + OFF_ITEM)[st] =
            reinterpret_cast<const uint32_t*>(items + k.item)[st];
      if (seg > 0) mbar_wait(cx.barrier(B_MATFREE), (seg - 1) & 1);  // nor does the tensor pipe read its planes
      stage_segment<CLS>(cx, items[k.item], k.c, md, st);
      staged_item = k.item;
      if (CLS == 1) {
        stagers_bar();
        finish_tip_tables(cx, st);
      }
      fence_async_smem();
      stagers_bar();
      if (st == 0) mbar_arrive(cx.barrier(B_MATFULL));
      ++seg;
    };

    if (warp >= EPI_W) {
      // ===== producers: tile -> transposition buffer -> split -> TMEM (hi | lo); the next tile is in registers =====
      // Tile sequence: class 0: (round, first child), (round, second child), ...; class 1: (round, child 0), ...
      const int w = warp - EPI_W;  // pattern rows 32 w .. 32 w + 31 = TMEM lanes of this warp
      const uint32_t xt = cx.smem + OFF_XT + (uint32_t)w * 2048;
      const uint32_t lane_tm = tmem + ((uint32_t)(32 * w) << 16);
      constexpr uint32_t TPR = CLS == 0 ? 2 : 1;  // tiles per round
      const uint32_t n_seq = cx.n_rounds * TPR;
      // a position in the tile sequence: round cursor + index of the tile inside its round
      struct TileCur {
        Cur k;
        uint32_t ui, j;
      };
      auto tile_next = [&](TileCur& t) {
        if (++t.j == TPR) {
          t.j = 0;
          ++t.ui;
          cx.advance(t.k);
        }
      };
      auto tile_ptr = [&](const TileCur& t) -> const float* {  // this warp's 32 rows of the tile
        const int k = CLS == 0 ? (int)((t.ui & 1) ^ t.j) : 0;  // the first child of round ui is ui & 1
        return static_cast<const float*>(item_of(t.k.item).p[k]) + ((size_t)t.k.c * P + t.k.tile * TP + 32 * w) * SP64;
      };
      float4 r[16];
      auto load_tile = [&](const TileCur& t) {
        const float* src = tile_ptr(t);
        const int row0 = t.k.tile * TP + 32 * w;
#pragma unroll
        for (int i = 0; i < 16; ++i) {  // pass i >> 2 (16 columns), chunk id = lane + 32 (i & 3): row id >> 2, chunk id & 3
          const int id = lane + 32 * (i & 3), rr = id >> 2, j = id & 3;
          r[i] = (row0 + rr < P) ? ldg_nc(src + (size_t)rr * SP64 + 16 * (i >> 2) + 4 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      };
      auto prefetch_tile = [&](const TileCur& t) {  // HBM -> L2, this warp's 32 rows (8 KB contiguous)
        if (t.ui < cx.n_rounds && lane == 0) {
          const int n = min(32, P - (t.k.tile * TP + 32 * w));
          if (n > 0) l2_prefetch_bulk(tile_ptr(t), (uint32_t)n * 256u);
        }
      };
      auto store_tile = [&](uint32_t col_hi) {
#pragma unroll
        for (int cp = 0; cp < 4; ++cp) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int id = lane + 32 * i;
            sts128(xt + xt_off(id >> 2, id & 3), r[4 * cp + i]);
          }
          __syncwarp();
          float hi[16], lo[16];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            float4 h, l;
            split4(lds128(xt + xt_off(lane, j)), h, l);
            hi[4 * j] = h.x; hi[4 * j + 1] = h.y; hi[4 * j + 2] = h.z; hi[4 * j + 3] = h.w;
            lo[4 * j] = l.x; lo[4 * j + 1] = l.y; lo[4 * j + 2] = l.z; lo[4 * j + 3] = l.w;
          }
          pre::tmem_st16(lane_tm + col_hi + 16 * cp, hi);
          pre::tmem_st16(lane_tm + col_hi + 64 + 16 * cp, lo);
          __syncwarp();
        }
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
      };
      Cur cur = cx.first();
      TileCur ld{cur, 0u, 0u}, pf{cur, 0u, 0u};  // next tile to load into registers / to prefetch into L2
      segment_start(cur);  // (the first round always opens a segment)
      load_tile(ld);
      tile_next(ld);
      tile_next(pf);
      prefetch_tile(pf);
      tile_next(pf);
      prefetch_tile(pf);
      tile_next(pf);
      for (uint32_t ui = 0; ui < cx.n_rounds; ++ui) {
        const uint32_t par = ui & 1, prev = par ^ 1;
        if (ui > 0 && cur.tile == 0) segment_start(cur);
        // first tile -> region par.  Class 0: that region was the SECOND child's in round ui - 1 (free since its step A
        // ran: REGFREE).  Class 1: it held X_0 and then q_0 of round ui - 2; the epilogue signals the reads of even and
        // odd rounds on two barriers, so that waiting for round ui - 2 does not have to wait for round ui - 1.
        if (CLS == 0) {
          if (ui > 0) mbar_wait(cx.barrier(B_REGFREE), prev);
        } else if (ui > 1) {
          mbar_wait(cx.barrier(par ? B_QREAD1 : B_QREAD), ((ui >> 1) + 1) & 1);
        }
        tc_fence_after();
        store_tile(T_REG * par);
        if (lane == 0) mbar_arrive(cx.barrier((CLS == 1 && par) ? B_XFULL_B : B_XFULL_A));  // class 1: see the MMA warp
        if (ld.ui < cx.n_rounds) load_tile(ld);
        tile_next(ld);
        prefetch_tile(pf);
        tile_next(pf);
        if (CLS == 0) {
          // second tile -> region 1 - par, which holds the q_k of round ui - 1 until the epilogue has read them
          if (ui > 0) mbar_wait(cx.barrier(B_QREAD), prev);
          tc_fence_after();
          store_tile(T_REG * (par ^ 1));
          if (lane == 0) mbar_arrive(cx.barrier(B_XFULL_B));
          if (ld.ui < cx.n_rounds) load_tile(ld);
          tile_next(ld);
          prefetch_tile(pf);
          tile_next(pf);
        }
        cx.advance(cur);
      }
    } else {
      // ===== epilogue: warp = quarter + 4 sub; thread = pattern row 32 quarter + lane; 16 states of each half =====
      const int quarter = warp & 3, sub = warp >> 2, row = 32 * quarter + lane;
      const uint32_t lane_tm = tmem + ((uint32_t)(32 * quarter) << 16);
      const uint32_t qs = cx.smem + OFF_QS + (uint32_t)warp * 2048;
      float* red = reinterpret_cast<float*>(tc5v_smem_raw + (cx.smem - smem_u32(tc5v_smem_raw)) + OFF_RED);
      float* smx = reinterpret_cast<float*>(tc5v_smem_raw + (cx.smem - smem_u32(tc5v_smem_raw)) + OFF_SMX);
      const size_t CP = (size_t)C * P;
      float4 qv[4];  // q_m slice of the next half-round, in flight: 32 rows x 16 states, chunk id = lane + 32 i
      auto load_qm = [&](const DevPreItem& it, int c, int p0, int h) {
        const float* src = static_cast<const float*>(it.qm) + ((size_t)c * P + p0 + 32 * quarter) * SP64 + 32 * h + 16 * sub;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int id = lane + 32 * i, rr = id >> 2, j = id & 3;
          qv[i] = (p0 + 32 * quarter + rr < P) ? ldg_nc(src + (size_t)rr * SP64 + 4 * j) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      };
      const int* sexp = reinterpret_cast<const int*>(tc5v_smem_raw + (cx.smem - smem_u32(tc5v_smem_raw)) + OFF_EXP);
      Cur cur = cx.first();
      segment_start(cur);  // (the first round always opens a segment)
      load_qm(*sit, cur.c, cur.tile * TP, 0);
      for (uint32_t ui = 0; ui < cx.n_rounds; ++ui) {
        const uint32_t par = ui & 1;
        if (ui > 0 && cur.tile == 0) segment_start(cur);
        const DevPreItem& it = *sit;
        const int c = cur.c, p0 = cur.tile * TP, p = p0 + row;
        const Cur nxt = cx.next(cur);
        mbar_wait(cx.barrier(par ? B_EXPFULL1 : B_EXPFULL), (ui >> 1) & 1);  // this round's pending exponents (long since there)
        const int e_q = sexp[(par * 3 + 0) * TP + row], e_x0 = sexp[(par * 3 + 1) * TP + row], e_2 = sexp[(par * 3 + 2) * TP + row];
        const Pow2Pair<float> fq = pow2_pair(-e_q, 0.f);
        const Pow2Pair<float> fx0 = pow2_pair(-e_x0, 0.f);
        const Pow2Pair<float> fx1 = pow2_pair(-(CLS == 0 ? e_2 : 0), 0.f);
        const int z1 = (CLS == 1 && e_2 < S) ? e_2 : 64;  // class 1: compact state of the tip child (missing -> the summed row 64)
        __syncwarp();
        if (lane == 0) mbar_arrive(cx.barrier(par ? B_EXPFREE1 : B_EXPFREE));
        // the usual case: every pending exponent fits ONE power-of-two factor (warp-uniform test)
        const bool one_factor = __all_sync(0xffffffffu, fq.f2 == 1.f && fx0.f2 == 1.f && fx1.f2 == 1.f);
        float dd = 0.f, n0 = 0.f, n1 = 0.f;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          // q_m slice: registers -> staging -> this thread's row (16 states)
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int id = lane + 32 * i;
            sts128(qs + xt_off(id >> 2, id & 3), qv[i]);
          }
          __syncwarp();
          float qm[16];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 v = lds128(qs + xt_off(lane, j));
            qm[4 * j] = v.x; qm[4 * j + 1] = v.y; qm[4 * j + 2] = v.z; qm[4 * j + 3] = v.w;
          }
          __syncwarp();
          if (h == 0) {
            load_qm(it, c, p0, 1);
          } else if (ui + 1 < cx.n_rounds) {
            load_qm(item_of(nxt.item), nxt.c, nxt.tile * TP, 0);
          }
          mbar_wait(cx.barrier(h == 0 ? B_AFULL0 : B_AFULL1), par);
          tc_fence_after();
          const uint32_t c0 = lane_tm + T_AB0 + 64 * h + 16 * sub, c1 = lane_tm + T_AB1 + 64 * h + 16 * sub;
#pragma unroll
          for (int e = 0; e < 2; ++e) {  // 8 states at a time keeps the split operands in registers
            uint32_t a0[8], b0[8], a1[8], b1[8];
            tmem_ld8(c0 + 8 * e, a0);
            tmem_ld8(c0 + 32 + 8 * e, b0);
            if (CLS == 0) {
              tmem_ld8(c1 + 8 * e, a1);
              tmem_ld8(c1 + 32 + 8 * e, b1);
            } else {
              const uint32_t ta = cx.smem + OFF_MAT1 + (uint32_t)(z1 * TAB_LD + 32 * h + 16 * sub + 8 * e) * 4;
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                const float4 va = lds128(ta + 16 * j), vb = lds128(ta + TAB_BYTES + 16 * j);
                a1[4 * j] = __float_as_uint(va.x); a1[4 * j + 1] = __float_as_uint(va.y);
                a1[4 * j + 2] = __float_as_uint(va.z); a1[4 * j + 3] = __float_as_uint(va.w);
                b1[4 * j] = __float_as_uint(vb.x); b1[4 * j + 1] = __float_as_uint(vb.y);
                b1[4 * j + 2] = __float_as_uint(vb.z); b1[4 * j + 3] = __float_as_uint(vb.w);
              }
            }
            tmem_ld_wait();
            float u0h[8], u0l[8], u1h[8], u1l[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              float s0, t0, s1, t1, qsj;
              if (one_factor) {
                s0 = __uint_as_float(a0[j]) * fx0.f1;
                t0 = __uint_as_float(b0[j]) * fx0.f1;
                s1 = CLS == 0 ? __uint_as_float(a1[j]) * fx1.f1 : __uint_as_float(a1[j]);
                t1 = CLS == 0 ? __uint_as_float(b1[j]) * fx1.f1 : __uint_as_float(b1[j]);
                qsj = qm[8 * e + j] * fq.f1;
              } else {
                s0 = pre::scale2(a0[j], fx0);
                t0 = pre::scale2(b0[j], fx0);
                s1 = CLS == 0 ? pre::scale2(a1[j], fx1) : __uint_as_float(a1[j]);
                t1 = CLS == 0 ? pre::scale2(b1[j], fx1) : __uint_as_float(b1[j]);
                qsj = (qm[8 * e + j] * fq.f1) * fq.f2;
              }
              const float u0 = qsj * s1, u1 = qsj * s0;
              dd = fmaf(u0, s0, dd);
              n0 = fmaf(u0, t0, n0);
              n1 = fmaf(u1, t1, n1);
              u0h[j] = tf32_hi(u0);
              u0l[j] = u0 - u0h[j];
              if (CLS == 0) {
                u1h[j] = tf32_hi(u1);
                u1l[j] = u1 - u1h[j];
              }
            }
            tmem_st8(c0 + 8 * e, u0h);       // U_0 hi over a_0, lo over b_0
            tmem_st8(c0 + 32 + 8 * e, u0l);
            if (CLS == 0) {
              tmem_st8(c1 + 8 * e, u1h);     // U_1 hi over a_1, lo over b_1
              tmem_st8(c1 + 32 + 8 * e, u1l);
            }
          }
          tmem_st_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(cx.barrier(h == 0 ? B_UFULL0 : B_UFULL1));
        }
        // ---- q_k: TMEM (region par: q_0 | q_1) -> registers (columns 32 sub ..), row maximum, coalesced store
        float mx[2] = {0.f, 0.f};
        mbar_wait(cx.barrier(B_QFULL), par);
        tc_fence_after();
#pragma unroll
        for (int k = 0; k < (CLS == 0 ? 2 : 1); ++k) {
          uint32_t qk[32];
          tmem_ld32(lane_tm + T_REG * par + 64 * k + 32 * sub, qk);
          tmem_ld_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(cx.barrier((CLS == 1 && par) ? B_QREAD1 : B_QREAD));
          float m4[4] = {0.f, 0.f, 0.f, 0.f};  // four independent chains
#pragma unroll
          for (int j = 0; j < 32; ++j) m4[j & 3] = fmaxf(m4[j & 3], __uint_as_float(qk[j]));
          mx[k] = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
          float* dest = static_cast<float*>(it.q[k]) + ((size_t)c * P + p0 + 32 * quarter) * SP64 + 32 * sub;
#pragma unroll
          for (int ps = 0; ps < 2; ++ps) {
#pragma unroll
            for (int j = 0; j < 4; ++j)
              sts128(qs + xt_off(lane, j), make_float4(__uint_as_float(qk[16 * ps + 4 * j]), __uint_as_float(qk[16 * ps + 4 * j + 1]),
                                                        __uint_as_float(qk[16 * ps + 4 * j + 2]), __uint_as_float(qk[16 * ps + 4 * j + 3])));
            __syncwarp();
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int id = lane + 32 * i, rr = id >> 2, j = id & 3;
              const float4 v = lds128(qs + xt_off(rr, j));
              if (p0 + 32 * quarter + rr < P) *reinterpret_cast<float4*>(dest + (size_t)rr * SP64 + 16 * ps + 4 * j) = v;
            }
            __syncwarp();
          }
        }
        // ---- combine the two sub warps of a row (fixed order), write the category's num / den and the q_k maxima
        if (sub == 1) {
          red[(par * 3 + 0) * TP + row] = dd;
          red[(par * 3 + 1) * TP + row] = n0;
          red[(par * 3 + 2) * TP + row] = n1;
          smx[(par * 2 + 0) * TP + row] = mx[0];
          smx[(par * 2 + 1) * TP + row] = mx[1];
        }
        epi_bar2();  // one barrier per round: the small arrays are double-buffered by round parity
        if (sub == 0 && p < P) {
          const float den = dd + red[(par * 3 + 0) * TP + row];
          const size_t at = (size_t)c * P + p;
          float* s0 = scratch + (size_t)it.slot[0] * 2 * CP;
          float* s1 = scratch + (size_t)it.slot[1] * 2 * CP;
          s0[at] = n0 + red[(par * 3 + 1) * TP + row];
          s0[CP + at] = den;
          s1[at] = n1 + red[(par * 3 + 2) * TP + row];
          s1[CP + at] = den;
          static_cast<float*>(it.q_scale[0])[at] = fmaxf(mx[0], smx[(par * 2 + 0) * TP + row]);
          if (CLS == 0) static_cast<float*>(it.q_scale[1])[at] = fmaxf(mx[1], smx[(par * 2 + 1) * TP + row]);
        }
        cur = nxt;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == N_W - 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------------------
// both children compact tips: den_c = sum_s q_m[s] M_0[s][z0] M_1[s][z1], num_0 = sum_s q_m[s] M_1[s][z1] D_0[s][z0],
// num_1 likewise.  HALF A WARP per pattern: lane l of the half holds states 4 l .. 4 l + 3, so a pattern's q_m row is one
// coalesced 256-byte request and the four table rows of its tip states are read as whole contiguous rows (128-bit
// loads, no bank conflicts), followed by a 4-step shuffle reduction of the three sums.  (The first version gave a lane
// a whole pattern: its 4 x 64 table values were gathered with scalar loads from rows that differ from lane to lane --
// 4-way bank conflicts on top of 1 KB of shared-memory traffic per 256 B of q_m: 1.9 TB/s.)
// blockIdx.x = chunk of G_TP patterns, blockIdx.y = item, blockIdx.z = category.
// ---------------------------------------------------------------------------------------------------------------
constexpr int G_THREADS = 256;  // patterns per block: chosen by the launcher (tables are re-staged per block)
constexpr int G_LD = 64;  // table row stride (floats): rows are read whole
constexpr size_t G_SMEM = (size_t)4 * 65 * G_LD * 4;  // M_0^T, D_0^T, M_1^T, D_1^T with the summed row 64

__global__ void __launch_bounds__(G_THREADS) k_grad64_tips(const DevPreItem* __restrict__ items, int P, int S, int C,
                                                           MatDeltas md, float* __restrict__ scratch, int G_TP) {
  extern __shared__ __align__(16) float g_tab[];  // [4][65][G_LD]
  const DevPreItem& it = items[blockIdx.y];
  const int c = blockIdx.z;
  const int p_begin = blockIdx.x * G_TP, p_end = min(P, p_begin + G_TP);
  const size_t CP = (size_t)C * P;
  for (int i = threadIdx.x; i < 4 * 1024; i += G_THREADS) {
    const int tb = i >> 10, e = i & 1023;  // e = 16 z + chunk: row z, four states
    const char* base = static_cast<const char*>(it.mat[tb >> 1]) + ((tb & 1) ? md.dt : md.t);
    const float4 v = ldg_nc(reinterpret_cast<const float*>(base) + (size_t)c * 4096 + 4 * e);
    *reinterpret_cast<float4*>(g_tab + tb * 65 * G_LD + 4 * e) = v;
  }
  __syncthreads();
  {
    const int tb = threadIdx.x >> 6, col = threadIdx.x & 63;
    float s = 0.f;
    for (int z = 0; z < 64; ++z) s += g_tab[(tb * 65 + z) * G_LD + col];
    g_tab[(tb * 65 + 64) * G_LD + col] = s;
  }
  __syncthreads();
  const float* qm = static_cast<const float*>(it.qm) + (size_t)c * P * SP64;
  float* s0 = scratch + (size_t)it.slot[0] * 2 * CP + (size_t)c * P;
  float* s1 = scratch + (size_t)it.slot[1] * 2 * CP + (size_t)c * P;
  const uint8_t* z0p = static_cast<const uint8_t*>(it.p[0]);
  const uint8_t* z1p = static_cast<const uint8_t*>(it.p[1]);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, half = lane >> 4, l = lane & 15;
  // a warp takes batches of 32 consecutive patterns: in step i its halves take patterns 2 i and 2 i + 1 of the batch;
  // lane (half, l) keeps the sums of step l, so that after 16 steps the batch is stored with coalesced requests
  for (int base = p_begin + 32 * warp; base < p_end; base += 32 * (G_THREADS / 32)) {
    const int pz = base + lane;  // this lane's pattern for the coalesced state loads / result stores
    int z0 = 64, z1 = 64;
    if (pz < p_end) {
      z0 = z0p[pz];
      z1 = z1p[pz];
      z0 = z0 >= S ? 64 : z0;
      z1 = z1 >= S ? 64 : z1;
    }
    const int zz = z0 | (z1 << 8);
    float vd[16], v0[16], v1[16];  // the three partial sums of the 16 steps (registers: the loops are unrolled)
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      const int src = 2 * i + half, p = base + src;
      const int y = __shfl_sync(0xffffffffu, zz, src), y0 = y & 255, y1 = y >> 8;
      float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
      if (p < p_end) q = ldg_nc(qm + (size_t)p * SP64 + 4 * l);
      const float4 a0 = *reinterpret_cast<const float4*>(g_tab + (0 * 65 + y0) * G_LD + 4 * l);
      const float4 b0 = *reinterpret_cast<const float4*>(g_tab + (1 * 65 + y0) * G_LD + 4 * l);
      const float4 a1 = *reinterpret_cast<const float4*>(g_tab + (2 * 65 + y1) * G_LD + 4 * l);
      const float4 b1 = *reinterpret_cast<const float4*>(g_tab + (3 * 65 + y1) * G_LD + 4 * l);
      const float u0x = q.x * a1.x, u0y = q.y * a1.y, u0z = q.z * a1.z, u0w = q.w * a1.w;
      const float u1x = q.x * a0.x, u1y = q.y * a0.y, u1z = q.z * a0.z, u1w = q.w * a0.w;
      vd[i] = fmaf(u0x, a0.x, fmaf(u0y, a0.y, fmaf(u0z, a0.z, u0w * a0.w)));
      v0[i] = fmaf(u0x, b0.x, fmaf(u0y, b0.y, fmaf(u0z, b0.z, u0w * b0.w)));
      v1[i] = fmaf(u1x, b1.x, fmaf(u1y, b1.y, fmaf(u1z, b1.z, u1w * b1.w)));
    }
    // sums over the 16 lanes of a half for all 16 steps at once: a reduce-scatter (8 + 4 + 2 + 1 exchanges per
    // quantity instead of 16 x 4), after which lane l holds the complete sums of step l in element 0
#pragma unroll
    for (int w = 8; w >= 1; w >>= 1) {
      const bool up = (l & w) != 0;
#pragma unroll
      for (int i = 0; i < w; ++i) {
        const float gd = __shfl_xor_sync(0xffffffffu, up ? vd[i] : vd[i + w], w);
        const float g0 = __shfl_xor_sync(0xffffffffu, up ? v0[i] : v0[i + w], w);
        const float g1 = __shfl_xor_sync(0xffffffffu, up ? v1[i] : v1[i + w], w);
        vd[i] = (up ? vd[i + w] : vd[i]) + gd;
        v0[i] = (up ? v0[i + w] : v0[i]) + g0;
        v1[i] = (up ? v1[i + w] : v1[i]) + g1;
      }
    }
    const float kd = vd[0], k0 = v0[0], k1 = v1[0];
    // lane (half, l) holds pattern base + 2 l + half
    const int po = base + 2 * l + half;
    if (po < p_end) {
      s0[po] = k0;
      s0[CP + po] = kd;
      s1[po] = k1;
      s1[CP + po] = kd;
    }
  }
}

// d_k[p] = sum_c w_c r_c num[c][p] / sum_c w_c den[c][p]; block partial sums of weight[p] d_k[p] in a fixed order.
// blockIdx.y indexes `slots` (the gradient slots served by the kernels above), blockIdx.x a chunk of 256 patterns.
__global__ void __launch_bounds__(256) k_grad64_finish(const float* __restrict__ scratch, const int* __restrict__ slots,
                                                       int P, int C, const double* __restrict__ catw,
                                                       const double* __restrict__ catr, const double* __restrict__ weights,
                                                       double* __restrict__ grad_partial, int n_part,
                                                       double* __restrict__ site_out) {
  __shared__ double redd[8];
  const int slot = slots[blockIdx.y];
  const size_t CP = (size_t)C * P;
  const float* num = scratch + (size_t)slot * 2 * CP;
  const float* den = num + CP;
  const int p = blockIdx.x * 256 + threadIdx.x;
  double contrib = 0.0;
  if (p < P) {
    double n = 0.0, d = 0.0;
    for (int c = 0; c < C; ++c) {
      n = fma(catw[c] * catr[c], (double)num[(size_t)c * P + p], n);
      d = fma(catw[c], (double)den[(size_t)c * P + p], d);
    }
    const double ratio = n / d;
    if (site_out != nullptr) site_out[(size_t)slot * P + p] = ratio;
    contrib = weights[p] * ratio;
  }
  const double s = block_sum(contrib, redd);
  if (threadIdx.x == 0) grad_partial[(size_t)slot * n_part + blockIdx.x] = s;
}

// ---- host-side launchers -------------------------------------------------------------------------------------------
inline int launch_prep(cudaStream_t stream, const float* mats, const float* Q, float* out_d, float* out_t, float* out_dt,
                       int n_matrices, int64_t* launches) {
  k_prep_matrices64<<<n_matrices, 256, 0, stream>>>(mats, Q, out_d, out_t, out_dt);
  if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
  ++*launches;
  return PLK_SUCCESS;
}

template <int CLS>
inline int launch_class(cudaStream_t stream, const DevPreItem* d_items, int n, int P, int S, int C, MatDeltas md,
                        float* scratch, int sm_count, int64_t* launches) {
  if (cudaFuncSetAttribute(k_pre_tc5v<CLS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES2) != cudaSuccess)
    return PLK_ERR_CUDA;
  const long long total = (long long)n * C * ((P + TP - 1) / TP);
  if (total <= 0) return PLK_SUCCESS;
  const int grid = total < sm_count ? (int)total : sm_count;
  k_pre_tc5v<CLS><<<grid, THREADS, SMEM_BYTES2, stream>>>(d_items, n, P, S, C, md, scratch);
  if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
  ++*launches;
  return PLK_SUCCESS;
}

inline int launch_tips(cudaStream_t stream, const DevPreItem* d_items, int n, int P, int S, int C, MatDeltas md,
                       float* scratch, int sm_count, int64_t* launches) {
  if (cudaFuncSetAttribute(k_grad64_tips, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G_SMEM) != cudaSuccess)
    return PLK_ERR_CUDA;
  // patterns per block: as many as still give every SM a few blocks (a block stages 66 KB of tables first)
  int tp = 4096;
  while (tp > 512 && (long long)((P + tp - 1) / tp) * n * C < 4LL * sm_count) tp >>= 1;
  for (int first = 0; first < n; first += 32768) {
    const int m = n - first < 32768 ? n - first : 32768;
    dim3 grid((P + tp - 1) / tp, m, C);
    k_grad64_tips<<<grid, G_THREADS, G_SMEM, stream>>>(d_items + first, P, S, C, md, scratch, tp);
    if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
    ++*launches;
  }
  return PLK_SUCCESS;
}

inline int launch_finish(cudaStream_t stream, const float* scratch, const int* d_slots, int n_slots, int P, int C,
                         const double* catw, const double* catr, const double* weights, double* grad_partial, int n_part,
                         double* site, int* n_parts, int64_t* launches) {
  *n_parts = (P + 255) / 256;
  for (int first = 0; first < n_slots; first += 32768) {
    const int m = n_slots - first < 32768 ? n_slots - first : 32768;
    dim3 grid(*n_parts, m);
    k_grad64_finish<<<grid, 256, 0, stream>>>(scratch, d_slots + first, P, C, catw, catr, weights, grad_partial, n_part, site);
    if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
    ++*launches;
  }
  return PLK_SUCCESS;
}

}  // namespace pre2
}  // namespace tc5
}  // namespace plk
