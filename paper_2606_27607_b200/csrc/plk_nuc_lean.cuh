// plk_nuc_lean.cuh -- 4-state fused pre-order + gradient kernel, specialised.
//
// Why.  The general TMA-staged kernel (plk_nuc_tma.cuh) spends ~600 warp instructions per (8 patterns x 4
// categories) cell group, of which 165 are fp64 arithmetic: the rest is operand-kind / slot / store-flag branching,
// index arithmetic and reductions done once per child (profiles/r01_nuc_pre4_tma.md: issue slots 42 % busy, "wait"
// the top stall, 2 CTAs per SM at 140 registers).  The hot case has no such variety: C = 4 categories, both
// derivatives wanted, a child is either an internal node (full partials in, q_k out) or a compact tip (states in,
// nothing out).  This file compiles exactly those three item classes -- the host sorts the items of a level by
// class and launches one grid per class -- so that the consumer body is straight-line code:
//   CLS 0  both children internal          CLS 1  child 0 internal, child 1 compact tip          CLS 2  both tips
// (a tip / internal pair is stored with the internal child first; the update is symmetric in the two children).
// Everything else (other category counts, tips given as partials, single-child items, the walk order) stays on
// the general kernels.
//
// Pipeline, stage layout and producer are those of plk_nuc_tma.cuh (cp.async.bulk into an NS-deep ring of stages,
// mbarrier full / empty pairs, level order: tiles of 32 patterns dealt round-robin to the CTAs).  Lane mapping:
// lane = 8 g + pl, g = category, pl = pattern within the warp's 8 patterns.  The category sums finish on the lanes
// of g = 0 (child 0) and g = 1 (child 1), which therefore hold ONE gradient accumulator each: a single 3-step
// xor reduction per tile serves both children.
#pragma once
#include "plk_nuc_tma.cuh"

namespace plk {

constexpr int NL_C = 4;

// tiles of CTA b in level order, without 64-bit division: tile j is (item, t) with item * n_tp + t = b + j * G
struct NlWalk {
  uint32_t item, t, step_item, step_t, n_tp;
  __device__ __forceinline__ void init(uint32_t b, uint32_t G, uint32_t n_tp_) {
    n_tp = n_tp_;
    item = b / n_tp;
    t = b - item * n_tp;
    step_item = G / n_tp;
    step_t = G - step_item * n_tp;
  }
  __device__ __forceinline__ void next() {
    item += step_item;
    t += step_t;
    if (t >= n_tp) {
      t -= n_tp;
      ++item;
    }
  }
};

// D[m] = M[m] Q for every 4 x 4 matrix m (16 threads each): the derivative matrices of the compact-tip children.
// With x_k = e_z:  num_k = q_k . (Q e_z) = u_k^T M_k Q e_z = sum_x u_k[x] D_k[x][z]  -- a 4-term gather-dot instead of
// the transposed product q_k = M_k^T u_k (which a tip never stores) followed by a dot with column z of Q.
template <typename T>
__global__ void __launch_bounds__(256) k_deriv_matrices4(const T* __restrict__ M, const T* __restrict__ Q, T* __restrict__ D,
                                                         int n_buffers, int C, size_t buffer_stride /* elements */) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_buffers * C * 16) return;
  const int m = i >> 4, x = (i >> 2) & 3, z = i & 3;
  const size_t base = (size_t)(m / C) * buffer_stride + (size_t)(m % C) * 16;
  const T* Mm = M + base;
  D[base + x * 4 + z] = Mm[x * 4] * Q[z] + Mm[x * 4 + 1] * Q[4 + z] + Mm[x * 4 + 2] * Q[8 + z] + Mm[x * 4 + 3] * Q[12 + z];
}

// rows per consumer lane: the 4-byte instantiation takes two patterns per lane (tile = 64 patterns), so that a matrix
// row read from shared memory serves both and twice the operand bytes are in flight per instruction -- the fp32
// kernels are bound by instructions per byte (same instruction count per cell as fp64 for half the bytes)
template <typename T>
struct NlRows {
  static constexpr int R = sizeof(T) == 4 ? 2 : 1;
};

// one cell of a staged operand tile.  fp64: a cell is 32 bytes and a 128-bit shared-memory load serves 8 lanes per
// phase, so 8 consecutive cells read half by half hit every bank group twice (2-way conflict: a third of all the
// kernel's shared-memory wavefronts, profiles/r01_nuc_pre4_lean_fp64.txt).  Lanes 4..7 of each group of 8 therefore
// read the upper half first: each phase then covers 8 distinct 16-byte bank groups.
__device__ __forceinline__ void ld4_cell(const double* p, double v[4], bool swap) {
  const double2* q = reinterpret_cast<const double2*>(p);
  const double2 a = q[swap ? 1 : 0], b = q[swap ? 0 : 1];
  v[0] = swap ? b.x : a.x;
  v[1] = swap ? b.y : a.y;
  v[2] = swap ? a.x : b.x;
  v[3] = swap ? a.y : b.y;
}
__device__ __forceinline__ void ld4_cell(const float* p, float v[4], bool) { ld4(p, v); }

// a[u][s] = sum_x M[s][x] v[u][x] / sum_x M[x][s] v[u][x] for R vectors at once
template <typename T, int R>
__device__ __forceinline__ void mv4r(const T* __restrict__ M, const T (&v)[R][4], T (&a)[R][4]) {
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    T r[4];
    ld4(M + 4 * s, r);
#pragma unroll
    for (int u = 0; u < R; ++u) a[u][s] = r[0] * v[u][0] + r[1] * v[u][1] + r[2] * v[u][2] + r[3] * v[u][3];
  }
}
// the rate matrix Q of the pass by value: a kernel parameter sits in the constant bank, so the products with Q take
// their matrix operand straight from there (no shared-memory reads: the l1tex pipe is the busiest unit of this
// kernel, profiles/r01_nuc_pre4_lean_fp64.txt)
template <typename T>
struct NlQ {
  T v[16];
};
template <typename T, int R>
__device__ __forceinline__ void mvq4r(const NlQ<T>& Q, const T (&v)[R][4], T (&a)[R][4]) {
#pragma unroll
  for (int s = 0; s < 4; ++s)
#pragma unroll
    for (int u = 0; u < R; ++u)
      a[u][s] = Q.v[4 * s] * v[u][0] + Q.v[4 * s + 1] * v[u][1] + Q.v[4 * s + 2] * v[u][2] + Q.v[4 * s + 3] * v[u][3];
}
template <typename T, int R>
__device__ __forceinline__ void mvt4r(const T* __restrict__ M, const T (&v)[R][4], T (&a)[R][4]) {
  T r[4];
  ld4(M, r);
#pragma unroll
  for (int u = 0; u < R; ++u)
#pragma unroll
    for (int s = 0; s < 4; ++s) a[u][s] = r[s] * v[u][0];
#pragma unroll
  for (int x = 1; x < 4; ++x) {
    ld4(M + 4 * x, r);
#pragma unroll
    for (int u = 0; u < R; ++u)
#pragma unroll
      for (int s = 0; s < 4; ++s) a[u][s] = fma(r[s], v[u][x], a[u][s]);
  }
}

template <typename T, int CLS>
__global__ void __launch_bounds__(NT_THREADS, 4) k_pre4_lean(const DevPreItem* __restrict__ items, int n_items, int P,
                                                             const NlQ<T> Qc, long long dmat_delta, NucModel md,
                                                             double* __restrict__ grad_partial, int n_part,
                                                             int wait_first) {
  constexpr int C = NL_C;
  constexpr int R = NlRows<T>::R;
  constexpr bool TIP0 = CLS == 2, TIP1 = CLS >= 1;
  using St = NtStage<T, C, 3, true, R>;
  constexpr int MS = St::MS, TP = St::TP;
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
  // Launch chain of one level (plk_api.cu): the first kernel of a level waits for the previous level and only then
  // lets the next launch in; the other classes of the level are independent of it, start as its CTAs drain and
  // wait at their END, so that a grid never completes before the one it overlaps.
  if (wait_first) pdl_wait();
  pdl_trigger();
  __syncthreads();
  const uint32_t n_tp = (uint32_t)((P + TP - 1) / TP);
  const uint32_t total = (uint32_t)n_items * n_tp;
  const uint32_t G = gridDim.x, b = blockIdx.x;
  const int J = total > b ? (int)((total - b + G - 1) / G) : 0;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == NT_CW) {  // ---- producer (one lane)
    if (lane == 0) {
      NlWalk w;
      w.init(b, G, n_tp);
      for (int j = 0; j < J; ++j, w.next()) {
        if (j >= NT_NS) mbar_wait(&empty[j % NT_NS], (uint32_t)((j / NT_NS - 1) & 1));
        const DevPreItem* it = items + w.item;
        const int p0 = (int)w.t * TP;
        const int n = P - p0 < TP ? P - p0 : TP;
        const void* ptr[3] = {it->qm, it->p[0], it->p[1]};
        const int kind[3] = {KIND_PARTIALS, TIP0 ? KIND_STATES : KIND_PARTIALS, TIP1 ? KIND_STATES : KIND_PARTIALS};
        const void* mat[2] = {it->mat[0], it->mat[1]};
        nt_fill<T, C, 3, true, R>(nt_smem + (size_t)(j % NT_NS) * St::BYTES, &full[j % NT_NS], it, sizeof(DevPreItem),
                                  ptr, kind, mat, md.weights, P, p0, n, dmat_delta);
      }
    }
    if (!wait_first) pdl_wait();
    return;
  }
  // ---- consumers: lane = 8 g + pl takes category g of patterns warp * 8 + pl + 32 u, u < R
  const int g = lane >> 3, pl = lane & 7;
  // category sums and num / den in the working precision (fp32 instances: the double versions of the three products,
  // five shuffles and the division were a tenth of the instructions of an issue-bound kernel; 1e-7 per pattern is far
  // inside the fp32 tolerance); the weighted pattern sum stays fp64
  const T cw = (T)md.catw[g], cwr = (T)(md.catw[g] * md.catr[g]);
  for (int j = 0; j < J; ++j) {
    const int s = j % NT_NS;
    unsigned char* stage = nt_smem + (size_t)s * St::BYTES;
    mbar_wait(&full[s], (uint32_t)((j / NT_NS) & 1));
    const NtHdr h = *reinterpret_cast<const NtHdr*>(stage + St::OFF_HDR);
    const DevPreItem& it = *reinterpret_cast<const DevPreItem*>(stage + St::OFF_DESC);
    const T* sM0 = reinterpret_cast<const T*>(stage + St::OFF_MATS) + g * MS;
    const T* sM1 = sM0 + C * MS;
    const T* sOp = reinterpret_cast<const T*>(stage + St::OFF_OPS);
    int r[R], p[R];
    bool live[R];
#pragma unroll
    for (int u = 0; u < R; ++u) {
      r[u] = warp * 8 + pl + 32 * u;
      live[u] = r[u] < h.n;
      p[u] = h.p0 + r[u];
    }

    // compact-tip child k: a_k = column z of M_k; qx_k holds column z of D_k = M_k Q (0 for a missing state), so that
    // num_k = u_k . qx_k and no q_k is formed (k_deriv_matrices4)
    T a0[R][4], a1[R][4], qx0[R][4], qx1[R][4];
    if (TIP0) {
      const T* D0 = sOp + (size_t)C * TP * 4 + g * 16;  // staged in the child's unused operand segment (nt_fill)
#pragma unroll
      for (int u = 0; u < R; ++u) {
        const int z = stage[St::OFF_ST + h.soff0 + r[u]];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          a0[u][x] = z < 4 ? sM0[x * 4 + z] : T(1);
          qx0[u][x] = z < 4 ? D0[x * 4 + z] : T(0);
        }
      }
    } else {
      T x0[R][4];
#pragma unroll
      for (int u = 0; u < R; ++u) ld4_cell(sOp + ((C + g) * TP + r[u]) * 4, x0[u], (pl & 4) != 0);
      mv4r<T, R>(sM0, x0, a0);
      mvq4r<T, R>(Qc, x0, qx0);
    }
    if (TIP1) {
      const T* D1 = sOp + (size_t)2 * C * TP * 4 + g * 16;
#pragma unroll
      for (int u = 0; u < R; ++u) {
        const int z = stage[St::OFF_ST + (TP + 16) + h.soff1 + r[u]];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          a1[u][x] = z < 4 ? sM1[x * 4 + z] : T(1);
          qx1[u][x] = z < 4 ? D1[x * 4 + z] : T(0);
        }
      }
    } else {
      T x1[R][4];
#pragma unroll
      for (int u = 0; u < R; ++u) ld4_cell(sOp + ((2 * C + g) * TP + r[u]) * 4, x1[u], (pl & 4) != 0);
      mv4r<T, R>(sM1, x1, a1);
      mvq4r<T, R>(Qc, x1, qx1);
    }
    T u0[R][4], u1[R][4], dd[R];
#pragma unroll
    for (int u = 0; u < R; ++u) {
      T qm[4];
      ld4_cell(sOp + (g * TP + r[u]) * 4, qm, (pl & 4) != 0);
      dd[u] = T(0);
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        u0[u][x] = qm[x] * a1[u][x];
        u1[u][x] = qm[x] * a0[u][x];
        dd[u] = fma(u0[u][x], a0[u][x], dd[u]);
      }
    }
    T q0[R][4], q1[R][4];
    if (TIP0) {
#pragma unroll
      for (int u = 0; u < R; ++u)
#pragma unroll
        for (int x = 0; x < 4; ++x) q0[u][x] = u0[u][x];  // num_0 = u_0 . D_0[:, z]
    } else {
      mvt4r<T, R>(sM0, u0, q0);
    }
    if (TIP1) {
#pragma unroll
      for (int u = 0; u < R; ++u)
#pragma unroll
        for (int x = 0; x < 4; ++x) q1[u][x] = u1[u][x];
    } else {
      mvt4r<T, R>(sM1, u1, q1);
    }
    double contrib = 0.0;
#pragma unroll
    for (int u = 0; u < R; ++u) {
      T n0 = q0[u][0] * qx0[u][0], n1 = q1[u][0] * qx1[u][0];
#pragma unroll
      for (int x = 1; x < 4; ++x) {
        n0 = fma(q0[u][x], qx0[u][x], n0);
        n1 = fma(q1[u][x], qx1[u][x], n1);
      }
      // ---- rescaled q_k of the internal children (power-of-two factor, discarded: it cancels in num / den)
      if (!TIP0) {
        int key = max(max(max_key(q0[u][0]), max_key(q0[u][1])), max(max_key(q0[u][2]), max_key(q0[u][3])));
        key = max(key, 0);
        key = max(key, __shfl_xor_sync(0xffffffffu, key, 8));
        key = max(key, __shfl_xor_sync(0xffffffffu, key, 16));
        const T f = pow2_neg(exp_of_key(key, T(0)), T(0));
        if (live[u]) {
          T v[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) v[x] = q0[u][x] * f;
          stg4c(static_cast<T*>(it.q[0]) + ((size_t)g * P + p[u]) * 4, v);
        }
      }
      if (!TIP1) {
        int key = max(max(max_key(q1[u][0]), max_key(q1[u][1])), max(max_key(q1[u][2]), max_key(q1[u][3])));
        key = max(key, 0);
        key = max(key, __shfl_xor_sync(0xffffffffu, key, 8));
        key = max(key, __shfl_xor_sync(0xffffffffu, key, 16));
        const T f = pow2_neg(exp_of_key(key, T(0)), T(0));
        if (live[u]) {
          T v[4];
#pragma unroll
          for (int x = 0; x < 4; ++x) v[x] = q1[u][x] * f;
          stg4c(static_cast<T*>(it.q[1]) + ((size_t)g * P + p[u]) * 4, v);
        }
      }
      // ---- category sums: den on every lane, num_0 on the lanes of g = 0, num_1 on those of g = 1
      T den = cw * dd[u], m0 = cwr * n0, m1 = cwr * n1;
      den += __shfl_xor_sync(0xffffffffu, den, 16);
      m0 += __shfl_xor_sync(0xffffffffu, m0, 16);
      m1 += __shfl_xor_sync(0xffffffffu, m1, 16);
      den += __shfl_xor_sync(0xffffffffu, den, 8);
      const bool odd = g & 1;
      const T got = __shfl_xor_sync(0xffffffffu, odd ? m0 : m1, 8);
      const T num = (odd ? m1 : m0) + got;
      if (live[u] && g < 2) {
        const double ratio = (double)(num / den);
        if (md.site_out != nullptr) md.site_out[(size_t)it.slot[g] * P + p[u]] = ratio;
        contrib += reinterpret_cast<const double*>(stage + St::OFF_WTS)[r[u]] * ratio;
      }
    }
    const int slot = it.slot[g & 1];
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);  // stage no longer needed (slot and weights are in registers)
    contrib += __shfl_xor_sync(0xffffffffu, contrib, 1);
    contrib += __shfl_xor_sync(0xffffffffu, contrib, 2);
    contrib += __shfl_xor_sync(0xffffffffu, contrib, 4);
    if (pl == 0 && g < 2) grad_partial[(size_t)slot * n_part + (h.p0 / TP) * NT_CW + warp] = contrib;
  }
  if (!wait_first) pdl_wait();
}

// ---------------------------------------------------------------------------------------------------------------
// Class 2 (both children compact tips) without the staging ring: the item reads only q_m (one cell per pattern and
// category) and writes nothing, so it is instruction-bound in the lane-per-cell mapping above.  Here a lane owns a
// whole PATTERN (R of them: p and p + 32, like the tiles of k_pre4_lean) and loops over the categories: the category
// sums stay in registers (no shuffles), a_k and the derivative column D_k[:, z] come as one vector each from small
// transposed tables in shared memory, and there is one division per pattern and child.
//   den = sum_c w_c sum_x q_m[x] a_1[x] a_0[x],  num_k = sum_c w_c r_c sum_x (q_m[x] a_{1-k}[x]) D_k[x][z_k]
// Gradient partial sums land exactly where k_pre4_lean puts them (entry = tile * NT_CW + lane / 8, tile = 32 R patterns).
// ---------------------------------------------------------------------------------------------------------------
// tiles of 32 R patterns a warp takes per launch: a CTA lives long enough to amortise its table set-up (item
// descriptor -> matrix pointers -> table entries: dependent global loads), and the loads of tile t + 1 are in flight
// while tile t is computed
// (all both-tips items of a pass run as ONE launch, plk_api.cu, so long CTAs leave no tail: fp64 141 us at 4 tiles per
// warp against 175 at one; the fp32 body took two rows per lane at first and ran out of registers at 4 tiles per warp
// (140 registers, 3 CTAs / SM); with ONE row per lane it needs 72 and takes 4 as well: configs[1] fp32 pre-order +
// gradient 0.561 -> 0.542 ms; 8 tiles per warp: no further change)
template <typename T>
struct NlTipsTpw {
  static constexpr int V = 4;
};
template <typename T>
struct NlTipsRows {  // pattern rows per lane of the both-tips kernel
  static constexpr int R = 1;
};

template <typename T>
struct NlTipsTile {  // what a lane reads for its R patterns of one tile
  static constexpr int C = NL_C, R = NlTipsRows<T>::R;
  int p[R], z0[R], z1[R];
  T qm[R][C][4];
  __device__ __forceinline__ void load(int tile, int lane, int P, const T* __restrict__ qmp,
                                       const uint8_t* __restrict__ st0, const uint8_t* __restrict__ st1) {
#pragma unroll
    for (int u = 0; u < R; ++u) {  // every load of the lane is issued before any arithmetic
      p[u] = tile * 32 * R + lane + 32 * u;
      const bool live = p[u] < P;
      z0[u] = live ? min((int)st0[p[u]], 4) : 4;
      z1[u] = live ? min((int)st1[p[u]], 4) : 4;
#pragma unroll
      for (int c = 0; c < C; ++c) {
        if (live) {
          ldg4(qmp + ((size_t)c * P + p[u]) * 4, qm[u][c]);
        } else {
#pragma unroll
          for (int x = 0; x < 4; ++x) qm[u][c][x] = T(0);
        }
      }
    }
  }
};

template <typename T>
__global__ void __launch_bounds__(NT_CW * 32) k_grad4_tips(const DevPreItem* __restrict__ items, int P, long long dmat_delta,
                                                           NucModel md, double* __restrict__ grad_partial, int n_part,
                                                           int wait_first) {
  constexpr int C = NL_C, R = NlTipsRows<T>::R, TPW = NlTipsTpw<T>::V;
  __shared__ __align__(16) T tabA[2][C][5][4];  // [child][category][state z (4 = missing)][x]: M_k[x][z]; missing: 1
  __shared__ __align__(16) T tabD[2][C][5][4];  // D_k[x][z]; missing: 0 (Q . 1 = 0)
  T scw[C], scwr[C];
#pragma unroll
  for (int c = 0; c < C; ++c) {
    scw[c] = (T)md.catw[c];
    scwr[c] = (T)(md.catw[c] * md.catr[c]);
  }
  if (wait_first) pdl_wait();  // launch chain: see k_pre4_lean
  pdl_trigger();
  const DevPreItem& it = items[blockIdx.y];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_tp = (P + 32 * R - 1) / (32 * R);
  const int tile0 = blockIdx.x * (NT_CW * TPW) + warp;  // the warp's tiles: tile0 + t NT_CW, t < TPW
  const uint8_t* st0 = static_cast<const uint8_t*>(it.p[0]);
  const uint8_t* st1 = static_cast<const uint8_t*>(it.p[1]);
  const T* qmp = static_cast<const T*>(it.qm);
  NlTipsTile<T> buf[2];
  buf[0].load(tile0, lane, P, qmp, st0, st1);  // in flight under the table set-up (a tile past the end loads nothing)
  for (int i = threadIdx.x; i < 2 * C * 16; i += blockDim.x) {
    const int k = i / (C * 16), c = (i / 16) % C, x = (i >> 2) & 3, z = i & 3;
    const T* M = static_cast<const T*>(it.mat[k]) + c * 16;
    const T* D = reinterpret_cast<const T*>(static_cast<const char*>(it.mat[k]) + dmat_delta) + c * 16;
    tabA[k][c][z][x] = M[x * 4 + z];
    tabD[k][c][z][x] = D[x * 4 + z];
  }
  for (int i = threadIdx.x; i < 2 * C * 4; i += blockDim.x) {
    const int k = i / (C * 4), c = (i >> 2) % C, x = i & 3;
    tabA[k][c][4][x] = T(1);
    tabD[k][c][4][x] = T(0);
  }
  __syncthreads();
  const int slot0 = it.slot[0], slot1 = it.slot[1];
#pragma unroll
  for (int t = 0; t < TPW; ++t) {
    const int tile = tile0 + t * NT_CW;
    if (tile >= n_tp) break;
    if (t + 1 < TPW) buf[(t + 1) & 1].load(tile + NT_CW, lane, P, qmp, st0, st1);
    const NlTipsTile<T>& b = buf[t & 1];
    double contrib[2] = {0.0, 0.0};
#pragma unroll
    for (int u = 0; u < R; ++u) {
      T den = T(0), num0 = T(0), num1 = T(0);  // working precision, as in k_pre4_lean
#pragma unroll
      for (int c = 0; c < C; ++c) {
        T a0[4], a1[4], d0[4], d1[4];
        ld4(&tabA[0][c][b.z0[u]][0], a0);
        ld4(&tabA[1][c][b.z1[u]][0], a1);
        ld4(&tabD[0][c][b.z0[u]][0], d0);
        ld4(&tabD[1][c][b.z1[u]][0], d1);
        T dd = T(0), n0 = T(0), n1 = T(0);
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          const T u0 = b.qm[u][c][x] * a1[x], u1 = b.qm[u][c][x] * a0[x];
          dd = fma(u0, a0[x], dd);
          n0 = fma(u0, d0[x], n0);
          n1 = fma(u1, d1[x], n1);
        }
        den = fma(scw[c], dd, den);
        num0 = fma(scwr[c], n0, num0);
        num1 = fma(scwr[c], n1, num1);
      }
      if (b.p[u] < P) {
        const double w = md.weights[b.p[u]], r0 = (double)(num0 / den), r1 = (double)(num1 / den);
        if (md.site_out != nullptr) {
          md.site_out[(size_t)slot0 * P + b.p[u]] = r0;
          md.site_out[(size_t)slot1 * P + b.p[u]] = r1;
        }
        contrib[0] += w * r0;
        contrib[1] += w * r1;
      }
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      double v = contrib[k];
      v += __shfl_xor_sync(0xffffffffu, v, 1);
      v += __shfl_xor_sync(0xffffffffu, v, 2);
      v += __shfl_xor_sync(0xffffffffu, v, 4);
      if ((lane & 7) == 0) grad_partial[(size_t)(k ? slot1 : slot0) * n_part + tile * NT_CW + (lane >> 3)] = v;
    }
  }
  if (!wait_first) pdl_wait();
}

}  // namespace plk
