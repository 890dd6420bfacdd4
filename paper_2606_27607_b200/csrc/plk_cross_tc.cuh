// plk_cross_tc.cuh -- rate-matrix gradient at 61 states (padded to 64) on the tensor cores (PAPER.md:29,
// :45-47, reading 14).  Same sum as k_cross64 (plk_cross.cuh):
//     G[i][j] = sum_b t_b sum_p omega_p ( sum_c w_c r_c q_b[c,p,i] p_b[c,p,j] ) / ( sum_c w_c q_b[c,p]^T p_b[c,p] )
// For one branch and category this is the contraction  G_c = (diag(s_c) Q_c)^T X_c  over the PATTERN axis: 64 x 64 x P.
// The partials sit in HBM as [pattern][state], i.e. both operands have the contraction index as their slow index; the
// mma.sync fragments take that directly from a shared-memory tile (a fragment's k index is the tile row), so nothing is
// transposed.  fp64: DMMA m8n8k4, the accumulators ARE the fp64 sums.  fp32: split-TF32 m16n8k8 (three products,
// plk_tc.cuh), fp32 accumulators over one branch (C x 32 patterns), widened into fp64 sums per branch.  In fp32 a
// compact tip (the other half of the branches) is never staged: its indicator rows are formed from the state in
// registers, exact in TF32, so its low-part product is skipped.
//   work unit = (tile of TP patterns, range of branches); units are dealt round-robin to a fixed grid, a CTA keeps its
//   64 x 64 sums in registers over all its units and writes ONE partial (fixed order: bitwise repeatable).
//   per (unit, branch): all C categories of q and p staged with cp.async (the quotient's denominator needs every
//   category before the first product), den and the per-(category, pattern) factors s, then the products.
//   4 warps, each a 32 x 32 block of G.  The m / n labels of a fragment are free, so a lane's rows / columns are chosen
//   adjacent in memory: one 128-bit shared-memory load per operand row gives the values of all of the lane's fragments
//   (fp32: rows i0 + 4g .. 4g+3 for both m-tiles; fp64: two loads of rows i0 + 2g, +1 and i0 + 16 + 2g, +1), and the
//   row strides (72 floats / 68 doubles) make those loads conflict-free.
#pragma once
#include "plk_common.cuh"
#include "plk_cross.cuh"
#include "plk_tc.cuh"

namespace plk {

template <typename T>
struct CrossTc;
template <>
struct CrossTc<float> {
  static constexpr int TP = 32, LD = 72, KSTEP = 8;
};
template <>
struct CrossTc<double> {
  static constexpr int TP = 16, LD = 68, KSTEP = 4;
};
constexpr int CROSS_TC_THREADS = 128, CROSS_TC_MAX_GRID = 512;

__device__ __forceinline__ void cross_tc_dmma(double& d0, double& d1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <typename T>
inline size_t cross_tc_smem(int C) {
  return (size_t)2 * C * CrossTc<T>::TP * CrossTc<T>::LD * sizeof(T) + (size_t)2 * C * sizeof(T) + (size_t)C * CrossTc<T>::TP * sizeof(T) +
         (size_t)CrossTc<T>::TP * 4;
}

// rows p0 .. p0+TP-1 of one category of full partials (`base` = that category's [P][64] plane) -> tile[row][0..63]
// (row stride LD); rows beyond P are zero.  A thread keeps its 16-byte column and takes every RPP-th row.
template <typename T>
__device__ __forceinline__ void cross_tc_stage_partials(T* __restrict__ tile, const T* __restrict__ base, int p0, int P) {
  constexpr int TP = CrossTc<T>::TP, LD = CrossTc<T>::LD, VEC = 16 / (int)sizeof(T), CPR = SP64 / VEC;
  constexpr int RPP = CROSS_TC_THREADS / CPR, PASSES = TP / RPP;
  const int ch = threadIdx.x % CPR, r0 = threadIdx.x / CPR;
  const T* src = base + (size_t)(p0 + r0) * SP64 + ch * VEC;
  T* dst = tile + r0 * LD + ch * VEC;
  if (p0 + TP <= P) {
#pragma unroll
    for (int k = 0; k < PASSES; ++k) tc_cp_async16(dst + k * RPP * LD, src + (size_t)k * RPP * SP64);
  } else {
#pragma unroll
    for (int k = 0; k < PASSES; ++k) {
      if (p0 + r0 + k * RPP < P) {
        tc_cp_async16(dst + k * RPP * LD, src + (size_t)k * RPP * SP64);
      } else {
#pragma unroll
        for (int j = 0; j < VEC; ++j) dst[k * RPP * LD + j] = T(0);
      }
    }
  }
}
// compact tip states (st == nullptr: an absent operand, zeros): indicator rows, the same for every category
template <typename T>
__device__ __forceinline__ void cross_tc_stage_states(T* __restrict__ tile, const uint8_t* __restrict__ st, int p0, int P, int S) {
  constexpr int TP = CrossTc<T>::TP, LD = CrossTc<T>::LD, VEC = 16 / (int)sizeof(T), CPR = SP64 / VEC;
  constexpr int RPP = CROSS_TC_THREADS / CPR, PASSES = TP / RPP;
  const int ch = threadIdx.x % CPR, r0 = threadIdx.x / CPR;
#pragma unroll
  for (int k = 0; k < PASSES; ++k) {
    const int row = r0 + k * RPP;
    const int z = (st != nullptr && p0 + row < P) ? (int)st[p0 + row] : -1;
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
      const int x = ch * VEC + j;
      tile[row * LD + x] = z < 0 ? T(0) : (z >= S ? (x < S ? T(1) : T(0)) : (x == z ? T(1) : T(0)));
    }
  }
}

// indicator of a compact tip state z at state x (z < 0: a row beyond P, zeros; z >= S: missing, 1 for every real state)
template <typename T>
__device__ __forceinline__ T cross_tc_ind(int z, int x, int S) {
  return z < 0 ? T(0) : (z >= S ? (x < S ? T(1) : T(0)) : (x == z ? T(1) : T(0)));
}

// partial[blockIdx.x][i * 64 + j]; padded rows / columns stay 0 (their operands are 0).  CC = the category count as a
// compile-time constant (loops unrolled), 0 = the runtime value C.
template <typename T, int CC>
__global__ void __launch_bounds__(CROSS_TC_THREADS, 3) k_cross_tc(const DevCrossBranch* __restrict__ br, int n_br, int n_split,
                                                                  int n_units, int P, int S, int C,
                                                                  const double* __restrict__ catw,
                                                                  const double* __restrict__ catr,
                                                                  const double* __restrict__ weights,
                                                                  double* __restrict__ partial) {
  using K = CrossTc<T>;
  constexpr int TP = K::TP, LD = K::LD, VEC = 16 / (int)sizeof(T), CPR = SP64 / VEC, NR = TP / 16;
  // fp32: a compact tip is never staged, its indicator rows are formed in registers (exact in TF32: no low-part
  // product); fp64: staged once for all categories (forming 64-bit indicators per k-step was slower than reading them)
  constexpr bool REG_TIPS = sizeof(T) == 4;
  using V = typename VecOf<T>::type;
  const int Cn = CC ? CC : C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sQ = reinterpret_cast<T*>(smem_raw);  // [C][TP][LD]
  T* sX = sQ + (size_t)Cn * TP * LD;       // [C][TP][LD]
  T* sW = sX + (size_t)Cn * TP * LD;       // w_c [C], then w_c r_c [C]
  T* sScale = sW + 2 * Cn;                 // [C][TP]
  int* sZ = reinterpret_cast<int*>(sScale + Cn * TP);  // [TP] compact tip states of the item (-1 beyond P)
  if (threadIdx.x < Cn) {
    sW[threadIdx.x] = (T)catw[threadIdx.x];
    sW[Cn + threadIdx.x] = (T)(catw[threadIdx.x] * catr[threadIdx.x]);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int i0 = (warp >> 1) * 32, j0 = (warp & 1) * 32;
  const int pp = threadIdx.x >> 3, l8 = threadIdx.x & 7;  // den pass: 8 lanes per pattern, rows pp (+ 16)

  double G[32];
#pragma unroll
  for (int e = 0; e < 32; ++e) G[e] = 0.0;

  for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
    const int chunk = u / n_split, sp = u % n_split;
    const int p0 = chunk * TP;
    const int b_lo = (int)((long long)sp * n_br / n_split), b_hi = (int)((long long)(sp + 1) * n_br / n_split);
    for (int b = b_lo; b < b_hi; ++b) {
      const DevCrossBranch Br = br[b];
      __syncthreads();  // the products of the previous branch have read the tiles
      // a tip's operand is the same for every category: staged once, or (REG_TIPS) not at all
      const bool per_cat = Br.kind == KIND_PARTIALS;
      const bool tip_states = Br.kind == KIND_STATES || Br.kind == KIND_NONE;
      const bool states = REG_TIPS && tip_states;
      const size_t xstep = per_cat ? (size_t)TP * LD : 0;
      if (states && threadIdx.x < TP)
        sZ[threadIdx.x] = (Br.kind == KIND_STATES && p0 + threadIdx.x < P) ? (int)static_cast<const uint8_t*>(Br.p)[p0 + threadIdx.x] : -1;
#pragma unroll
      for (int c = 0; c < Cn; ++c) {
        cross_tc_stage_partials<T>(sQ + (size_t)c * TP * LD, static_cast<const T*>(Br.q) + (size_t)c * P * SP64, p0, P);
        if (per_cat) cross_tc_stage_partials<T>(sX + (size_t)c * TP * LD, static_cast<const T*>(Br.p) + (size_t)c * P * SP64, p0, P);
      }
      if (Br.kind == KIND_BCAST) cross_tc_stage_partials<T>(sX, static_cast<const T*>(Br.p), p0, P);
      if (!REG_TIPS && tip_states)
        cross_tc_stage_states<T>(sX, Br.kind == KIND_STATES ? static_cast<const uint8_t*>(Br.p) : nullptr, p0, P, S);
      tc_cp_commit();
      T wt_row[NR];  // omega_p t_b of this thread's den rows, in flight while the tiles arrive
#pragma unroll
      for (int rr = 0; rr < NR; ++rr) {
        const int p = p0 + rr * 16 + pp;
        wt_row[rr] = p < P ? (T)(weights[p] * Br.t) : T(0);
      }
      tc_cp_wait<0>();
      __syncthreads();

      // den_p = sum_c w_c q^T p, then s[c][p] = omega_p w_c r_c t_b / den_p   (working precision: the quotient's
      // error is that of the products it scales)
      {
        T dsum[NR];
#pragma unroll
        for (int rr = 0; rr < NR; ++rr) {
          const int row = rr * 16 + pp;
          const int z = states ? sZ[row] : 0;
          T ds = T(0);
#pragma unroll
          for (int c = 0; c < Cn; ++c) {
            const T* q = sQ + ((size_t)c * TP + row) * LD;
            const T* x = sX + c * xstep + (size_t)row * LD;
            T d[2] = {T(0), T(0)};
#pragma unroll
            for (int k = 0; k < CPR / 8; ++k) {
              T qa[VEC], xa[VEC];
              unpack(*reinterpret_cast<const V*>(q + (l8 + 8 * k) * VEC), qa);
              if (states) {
#pragma unroll
                for (int j = 0; j < VEC; ++j) xa[j] = cross_tc_ind<T>(z, (l8 + 8 * k) * VEC + j, S);
              } else {
                unpack(*reinterpret_cast<const V*>(x + (l8 + 8 * k) * VEC), xa);
              }
#pragma unroll
              for (int j = 0; j < VEC; ++j) d[k & 1] = fma(qa[j], xa[j], d[k & 1]);
            }
            ds = fma(sW[c], d[0] + d[1], ds);
          }
          dsum[rr] = ds;
        }
#pragma unroll
        for (int rr = 0; rr < NR; ++rr) dsum[rr] = lane8_sum(dsum[rr]);
#pragma unroll
        for (int rr = 0; rr < NR; ++rr) {
          const T f = wt_row[rr] != T(0) ? wt_row[rr] / dsum[rr] : T(0);  // rows beyond P (den = 0), weight 0: factor 0
          for (int c = l8; c < Cn; c += 8) sScale[c * TP + rr * 16 + pp] = sW[Cn + c] * f;
        }
      }
      __syncthreads();

      if constexpr (sizeof(T) == 4) {
        float acc[2][4][4];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = acc[mt][nt][2] = acc[mt][nt][3] = 0.0f;
#pragma unroll 1
        for (int c = 0; c < Cn; ++c) {
          const float* q = sQ + (size_t)c * TP * LD + i0 + 4 * g;
          const float* x = sX + c * xstep + j0 + 4 * g;
          const float* sc = sScale + c * TP;
#pragma unroll
          for (int ks = 0; ks < TP / 8; ++ks) {
            const int r0 = ks * 8 + t, r1 = r0 + 4;
            const float s0 = sc[r0], s1 = sc[r1];
            const float4 qa = *reinterpret_cast<const float4*>(q + r0 * LD);
            const float4 qb = *reinterpret_cast<const float4*>(q + r1 * LD);
            // fragment row g <-> state i0 + 4g + 2 mt, row g + 8 <-> i0 + 4g + 2 mt + 1; column n = g of n-tile nt <->
            // state j0 + 4g + nt
            uint32_t ah[2][4], al[2][4], bh[4][2], bl[4][2];
            tc_split(qa.x * s0, ah[0][0], al[0][0]);
            tc_split(qa.y * s0, ah[0][1], al[0][1]);
            tc_split(qb.x * s1, ah[0][2], al[0][2]);
            tc_split(qb.y * s1, ah[0][3], al[0][3]);
            tc_split(qa.z * s0, ah[1][0], al[1][0]);
            tc_split(qa.w * s0, ah[1][1], al[1][1]);
            tc_split(qb.z * s1, ah[1][2], al[1][2]);
            tc_split(qb.w * s1, ah[1][3], al[1][3]);
            if (states) {  // indicator rows: exact in TF32, no low part
              const int z0 = sZ[r0], z1 = sZ[r1];
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) {
                bh[nt][0] = __float_as_uint(cross_tc_ind<float>(z0, j0 + 4 * g + nt, S));
                bh[nt][1] = __float_as_uint(cross_tc_ind<float>(z1, j0 + 4 * g + nt, S));
              }
            } else {
              const float4 xa = *reinterpret_cast<const float4*>(x + r0 * LD);
              const float4 xb = *reinterpret_cast<const float4*>(x + r1 * LD);
              tc_split(xa.x, bh[0][0], bl[0][0]);
              tc_split(xb.x, bh[0][1], bl[0][1]);
              tc_split(xa.y, bh[1][0], bl[1][0]);
              tc_split(xb.y, bh[1][1], bl[1][1]);
              tc_split(xa.z, bh[2][0], bl[2][0]);
              tc_split(xb.z, bh[2][1], bl[2][1]);
              tc_split(xa.w, bh[3][0], bl[3][0]);
              tc_split(xb.w, bh[3][1], bl[3][1]);
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) tc_mma(acc[mt][nt], al[mt], bh[nt]);
            if (!states) {
#pragma unroll
              for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) tc_mma(acc[mt][nt], ah[mt], bl[nt]);
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) tc_mma(acc[mt][nt], ah[mt], bh[nt]);
          }
        }
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt)
#pragma unroll
            for (int e = 0; e < 4; ++e) G[(mt * 4 + nt) * 4 + e] += (double)acc[mt][nt][e];
      } else {
        for (int c = 0; c < Cn; ++c) {
          const double* q = sQ + (size_t)c * TP * LD + i0 + 2 * g;
          const double* x = sX + c * xstep + j0 + 2 * g;
          const double* sc = sScale + c * TP;
#pragma unroll
          for (int ks = 0; ks < TP / 4; ++ks) {
            const int r = ks * 4 + t;
            const double s = sc[r];
            const double2 qa = *reinterpret_cast<const double2*>(q + r * LD);
            const double2 qb = *reinterpret_cast<const double2*>(q + r * LD + 16);
            // fragment row g of m-tile mt <-> state i0 + 16 (mt >> 1) + 2g + (mt & 1); the same for columns
            const double a[4] = {qa.x * s, qa.y * s, qb.x * s, qb.y * s};
            double bb[4];
            if (states) {
              const int z = sZ[r];
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) bb[nt] = cross_tc_ind<double>(z, j0 + 16 * (nt >> 1) + 2 * g + (nt & 1), S);
            } else {
              const double2 xa = *reinterpret_cast<const double2*>(x + r * LD);
              const double2 xb = *reinterpret_cast<const double2*>(x + r * LD + 16);
              bb[0] = xa.x; bb[1] = xa.y; bb[2] = xb.x; bb[3] = xb.y;
            }
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) cross_tc_dmma(G[(mt * 4 + nt) * 2], G[(mt * 4 + nt) * 2 + 1], a[mt], bb[nt]);
          }
        }
      }
    }
  }

  double* out = partial + (size_t)blockIdx.x * SP64 * SP64;
  if constexpr (sizeof(T) == 4) {
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 4; ++nt)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          // accumulator e: fragment row g (+8 for e >= 2), fragment column 2t + (e & 1)
          const int i = i0 + 4 * g + 2 * mt + (e >> 1);
          const int j = j0 + 4 * (2 * t + (e & 1)) + nt;
          out[i * SP64 + j] = G[(mt * 4 + nt) * 4 + e];
        }
  } else {
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
      for (int nt = 0; nt < 4; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int i = i0 + 16 * (mt >> 1) + 2 * g + (mt & 1);
          const int j = j0 + 16 * (nt >> 1) + 2 * (2 * t + e) + (nt & 1);
          out[i * SP64 + j] = G[(mt * 4 + nt) * 2 + e];
        }
  }
}

}  // namespace plk
