// plk_tc.cuh -- tensor-pipe kernels for state counts padded to SP = 64 (61-state codon models): the path taken when
// the instance carries PLK_FLAG_TENSOR_CORES (BASELINE.json configs[2] "CUDA-core vs tensor-core partials update",
// configs[3] "fp32 tensor-core path"; "tensor cores ... for amino acid and codon models").
//
// The contraction.  For one (operation, category) the post-order update is, per child k,
//     A_k[p][s] = sum_x X_k[p][x] * M_k[s][x]
// i.e. D = X . M^T with X the child's partials, row-major [pattern][state] exactly as they sit in HBM ([c][p][s]
// layout), and M the row-major transition matrix = the column-major B operand of an `mma ... row.col`.  No operand
// is transposed or repacked on its way from HBM to the tensor pipe.  The pre-order update needs M_k^T u instead:
// same instruction, B fragment read with the two indices swapped.
//
// Instructions (the two the ISA offers for these precisions):
//   fp64  mma.sync.aligned.m8n8k4.f64        (DMMA)   -- tcgen05 has no fp64 kind
//   fp32  mma.sync.aligned.m16n8k8.tf32 x 3  (split TF32): x = hi + lo with hi = tf32(x), lo = tf32(x - hi);
//         x.m ~= lo.hi + hi.lo + hi.hi, fp32 accumulate: the dropped lo.lo term is 2^-22 relative, so the result
//         keeps fp32 accuracy (plain TF32 would give 1e-3, outside the 1e-4 parity bar of BASELINE.json).
//
// Tiling.  A CTA of 8 warps owns a tile of TP patterns (fp64: 64, fp32: 128); warp w owns rows w*MT .. w*MT+MT-1
// (MT = 8 / 16) and all 64 output states = 8 n-tiles, so every per-pattern reduction (maximum for the deferred
// rescaling, gradient numerator / denominator) stays inside groups of 4 lanes.  Both precisions therefore use the
// same shared-memory budget: one tile = one matrix = 64 x 68 fp64 = 34 816 B (fp32: 128 x 68 for a tile, hi + lo
// planes for a matrix).  Row stride 68 makes the fragment reads (8 rows x 4 consecutive elements per warp)
// bank-conflict-free.
//
// Staging.  Operand tiles are copied global -> shared with cp.async (16-byte chunks into the padded rows), double
// buffered in the post-order kernel: the copy of work item i+1 is in flight while item i is on the tensor pipe.
// Work items (operation, category, tile) are dealt to a persistent grid in contiguous ranges with the tile index
// fastest, so a CTA reloads its two matrices only when (operation, category) changes.
//
// Rescaling is deferred exactly as in plk_gen.cuh (unscaled partials + per-(c,p) maxima, power-of-two factors
// applied by the reader), so both 64-state paths are interchangeable buffer by buffer.
#pragma once
#include "plk_common.cuh"
#include "plk_gen.cuh"

namespace plk {

constexpr int TC_THREADS = 256;
constexpr int TC_WARPS = TC_THREADS / 32;

template <typename T>
struct Tc;
template <>
struct Tc<double> {
  static constexpr int MT = 8, KT = 4, CN = 2;  // m-tile rows, k per instruction, accumulator registers per n-tile
  static constexpr int TP = MT * TC_WARPS, RPT = CN / 2;  // patterns per tile (64), rows per thread (1)
  static constexpr int LD = 68;                            // padded row stride (elements) of tiles and matrices
  static constexpr int TILE_BYTES = TP * LD * 8, MAT_BYTES = 64 * LD * 8;  // 34 816 each
};
template <>
struct Tc<float> {
  static constexpr int MT = 16, KT = 8, CN = 4;
  static constexpr int TP = MT * TC_WARPS, RPT = CN / 2;  // 128, 2
  static constexpr int LD = 72;
  static constexpr int TILE_BYTES = TP * LD * 4, MAT_BYTES = 2 * 64 * LD * 4;  // 36 864; hi plane + lo plane
};

// ---- PTX ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t tc_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void tc_cp_async16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(tc_smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void tc_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void tc_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void tc_mma(double (&d)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void tc_mma(float (&d)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
  asm(
      "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}
// x = hi + lo with hi = x, low 13 mantissa bits cleared, lo = x - hi exactly: two ALU operations instead of two
// conversions and a subtraction (see tf32_hi in plk_tc5.cuh: the conversion unit is slow and was the bottleneck)
__device__ __forceinline__ void tc_split(float x, uint32_t& hi, uint32_t& lo) {
  hi = __float_as_uint(x) & 0xffffe000u;
  lo = __float_as_uint(x - __uint_as_float(hi));
}

// ---- staging ---------------------------------------------------------------------------------------------------
// rows 0..n-1 of `src` ([.][64] row-major in global memory) -> tile rows (stride Tc<T>::LD); rows n..TP-1 <- 0
template <typename T>
__device__ __forceinline__ void tc_load_tile(T* __restrict__ tile, const T* __restrict__ src, int n) {
  constexpr int VEC = 16 / (int)sizeof(T), CPR = SP64 / VEC, TP = Tc<T>::TP;
  for (int idx = threadIdx.x; idx < TP * CPR; idx += TC_THREADS) {
    const int row = idx / CPR, ch = idx % CPR;
    T* dst = tile + row * Tc<T>::LD + ch * VEC;
    if (row < n) {
      tc_cp_async16(dst, src + (size_t)row * SP64 + ch * VEC);
    } else {
#pragma unroll
      for (int j = 0; j < VEC; ++j) dst[j] = T(0);
    }
  }
}
// the calling warp's MT rows (first row m0) of the same tile, copied by the warp's own lanes: rows are warp-private
// (only the owning warp reads them as A fragments), so a cp.async wait + __syncwarp is all the consumer needs
template <typename T>
__device__ __forceinline__ void tc_load_rows(T* __restrict__ tile, const T* __restrict__ src, int n, int m0, int lane) {
  constexpr int VEC = 16 / (int)sizeof(T), CPR = SP64 / VEC, MT = Tc<T>::MT;
#pragma unroll
  for (int idx = lane; idx < MT * CPR; idx += 32) {
    const int row = m0 + idx / CPR, ch = idx % CPR;
    T* dst = tile + row * Tc<T>::LD + ch * VEC;
    if (row < n) {
      tc_cp_async16(dst, src + (size_t)row * SP64 + ch * VEC);
    } else {
#pragma unroll
      for (int j = 0; j < VEC; ++j) dst[j] = T(0);
    }
  }
}
template <typename T>
__device__ __forceinline__ void tc_load_operand_rows(T* tile, int kind, const void* ptr, int c, int p0, int n, int P,
                                                     int m0, int lane) {
  if (kind == KIND_PARTIALS)
    tc_load_rows<T>(tile, static_cast<const T*>(ptr) + ((size_t)c * P + p0) * SP64, n, m0, lane);
  else if (kind == KIND_BCAST)
    tc_load_rows<T>(tile, static_cast<const T*>(ptr) + (size_t)p0 * SP64, n, m0, lane);
}
// operand tile of a child / of the parent's pre-order partials; compact tips and absent operands load nothing
template <typename T>
__device__ __forceinline__ void tc_load_operand(T* tile, int kind, const void* ptr, int c, int p0, int n, int P) {
  if (kind == KIND_PARTIALS) tc_load_tile<T>(tile, static_cast<const T*>(ptr) + ((size_t)c * P + p0) * SP64, n);
  else if (kind == KIND_BCAST) tc_load_tile<T>(tile, static_cast<const T*>(ptr) + (size_t)p0 * SP64, n);
}

// matrix [64][64] row-major in global memory -> shared (padded rows), asynchronously (cp.async, 16-byte chunks)
template <typename T>
__device__ __forceinline__ void tc_load_matrix(T* __restrict__ sM, const T* __restrict__ M) {
  constexpr int VEC = 16 / (int)sizeof(T), CPR = SP64 / VEC;
  for (int idx = threadIdx.x; idx < SP64 * CPR; idx += TC_THREADS) {
    const int r = idx / CPR, ch = idx % CPR;
    tc_cp_async16(sM + r * Tc<T>::LD + ch * VEC, M + r * SP64 + ch * VEC);
  }
}
// element M[s][x] of a staged matrix (tip gathers)
__device__ __forceinline__ double tc_mat_at(const double* sM, int s, int x) { return sM[s * Tc<double>::LD + x]; }
__device__ __forceinline__ float tc_mat_at(const float* sM, int s, int x) {
  return sM[s * Tc<float>::LD + x] + sM[SP64 * Tc<float>::LD + s * Tc<float>::LD + x];  // hi + lo: exact
}
// fp32: split a landed matrix in place into its TF32 hi plane and the exact remainder (lo plane), once per staging,
// so that the inner loop of tc_gemm converts nothing on the B side.  Callers put a barrier on both sides.
__device__ __forceinline__ void tc_split_matrix(double*) {}
__device__ __forceinline__ void tc_split_matrix(float* sM) {
  constexpr int LD = Tc<float>::LD;
  for (int idx = threadIdx.x; idx < SP64 * SP64 / 4; idx += TC_THREADS) {
    const int r = idx >> 4, c4 = (idx & 15) * 4;
    float4 v = *reinterpret_cast<float4*>(sM + r * LD + c4);
    float4 h, l;
    h.x = __uint_as_float(__float_as_uint(v.x) & 0xffffe000u); l.x = v.x - h.x;
    h.y = __uint_as_float(__float_as_uint(v.y) & 0xffffe000u); l.y = v.y - h.y;
    h.z = __uint_as_float(__float_as_uint(v.z) & 0xffffe000u); l.z = v.z - h.z;
    h.w = __uint_as_float(__float_as_uint(v.w) & 0xffffe000u); l.w = v.w - h.w;
    *reinterpret_cast<float4*>(sM + r * LD + c4) = h;
    *reinterpret_cast<float4*>(sM + SP64 * LD + r * LD + c4) = l;
  }
}

// ---- warp-level product: acc[nt][.] = sum_x A[row][x] * B(x, 8 nt + n)  for the warp's MT rows ----------------------
//   TRANS = false: B(x, s) = M[s][x]  (M . x);   TRANS = true: B(x, s) = M[x][s]  (M^T . x)
// Fragment ownership (PTX ISA, mma.m8n8k4 / m16n8k8): with r = lane / 4, c = lane % 4 a lane holds
//   accumulator (row r [+8], columns 8 nt + 2c, 2c + 1),  A (row r [+8], k0 + c [+4]),  B (k0 + c [+4], column 8 nt + r).
template <bool TRANS>
__device__ __forceinline__ void tc_gemm(const double* __restrict__ sA, const double* __restrict__ sM, double (&acc)[8][2],
                                        int r, int c) {
#pragma unroll
  for (int nt = 0; nt < 8; ++nt) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll 4
  for (int k0 = 0; k0 < SP64; k0 += 4) {
    const double a = sA[r * Tc<double>::LD + k0 + c];
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      const double b = TRANS ? sM[(k0 + c) * Tc<double>::LD + nt * 8 + r] : sM[(nt * 8 + r) * Tc<double>::LD + k0 + c];
      tc_mma(acc[nt], a, b);
    }
  }
}
// fp32: the k index of an mma is only a summation index, so the non-transposed product assigns lane c the
// physical columns k0 + 2c, 2c + 1 (instead of k0 + c, c + 4) for BOTH operands: one 64-bit shared-memory load per
// fragment pair.  The A side is split into hi / lo in registers, the B side comes pre-split (tc_split_matrix); the three products of one k-step are issued term by term
// over the 8 independent accumulators so that no mma waits on the one before it.
template <bool TRANS>
__device__ __forceinline__ void tc_gemm(const float* __restrict__ sA, const float* __restrict__ sM, float (&acc)[8][4],
                                        int r, int c) {
  constexpr int LD = Tc<float>::LD;
#pragma unroll
  for (int nt = 0; nt < 8; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.0f;
#pragma unroll 2
  for (int k0 = 0; k0 < SP64; k0 += 8) {
    float av[4];
    if (!TRANS) {
      const float2 t0 = *reinterpret_cast<const float2*>(sA + r * LD + k0 + 2 * c);
      const float2 t1 = *reinterpret_cast<const float2*>(sA + (r + 8) * LD + k0 + 2 * c);
      av[0] = t0.x; av[1] = t1.x; av[2] = t0.y; av[3] = t1.y;
    } else {
      av[0] = sA[r * LD + k0 + c];
      av[1] = sA[(r + 8) * LD + k0 + c];
      av[2] = sA[r * LD + k0 + c + 4];
      av[3] = sA[(r + 8) * LD + k0 + c + 4];
    }
    uint32_t ah[4], al[4], bh[8][2], bl[8][2];
#pragma unroll
    for (int j = 0; j < 4; ++j) tc_split(av[j], ah[j], al[j]);
    const uint32_t* sH = reinterpret_cast<const uint32_t*>(sM);
    const uint32_t* sL = sH + SP64 * LD;
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      if (!TRANS) {
        const uint2 th = *reinterpret_cast<const uint2*>(sH + (nt * 8 + r) * LD + k0 + 2 * c);
        const uint2 tl = *reinterpret_cast<const uint2*>(sL + (nt * 8 + r) * LD + k0 + 2 * c);
        bh[nt][0] = th.x; bh[nt][1] = th.y;
        bl[nt][0] = tl.x; bl[nt][1] = tl.y;
      } else {
        bh[nt][0] = sH[(k0 + c) * LD + nt * 8 + r];
        bh[nt][1] = sH[(k0 + c + 4) * LD + nt * 8 + r];
        bl[nt][0] = sL[(k0 + c) * LD + nt * 8 + r];
        bl[nt][1] = sL[(k0 + c + 4) * LD + nt * 8 + r];
      }
    }
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) tc_mma(acc[nt], al, bh[nt]);
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) tc_mma(acc[nt], ah, bl[nt]);
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) tc_mma(acc[nt], ah, bh[nt]);
  }
}

template <typename T>
struct Vec2Of;
template <>
struct Vec2Of<double> {
  using type = double2;
};
template <>
struct Vec2Of<float> {
  using type = float2;
};

// acc <- column z of M (a compact tip: SURVEY 8(c) row 15), `missing` for a missing state, 0 in the padding
template <typename T>
__device__ __forceinline__ void tc_gather(const T* __restrict__ sM, int z, int S, T missing, int h, int c,
                                          T (&acc)[8][Tc<T>::CN]) {
#pragma unroll
  for (int nt = 0; nt < 8; ++nt)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int s = nt * 8 + 2 * c + j;
      acc[nt][h * 2 + j] = z < S ? tc_mat_at(sM, s, z) : (s < S ? missing : T(0));
    }
}

// ---------------------------------------------------------------------------------------------------------------
// post-order update (maxima for the deferred step 3)
// persistent grid over work items (operation, category, tile), tile fastest
// ---------------------------------------------------------------------------------------------------------------
template <typename T>
constexpr size_t tc_post_smem() { return 2 * (size_t)Tc<T>::MAT_BYTES + 4 * (size_t)Tc<T>::TILE_BYTES; }  // 2 stages

template <typename T>
__global__ void __launch_bounds__(TC_THREADS, 1) k_post_tc(const DevOp* __restrict__ ops, int n_ops, int P, int S, int C) {
  using K = Tc<T>;
  using V2 = typename Vec2Of<T>::type;
  constexpr int TP = Tc<T>::TP, RPT = Tc<T>::RPT;
  extern __shared__ __align__(16) unsigned char tc_smem[];
  constexpr int LD = K::LD;
  T* sM[2] = {reinterpret_cast<T*>(tc_smem), reinterpret_cast<T*>(tc_smem + K::MAT_BYTES)};
  T* sX[2][2];
#pragma unroll
  for (int st = 0; st < 2; ++st)
#pragma unroll
    for (int k = 0; k < 2; ++k) sX[st][k] = reinterpret_cast<T*>(tc_smem + 2 * (size_t)K::MAT_BYTES + (size_t)(2 * st + k) * K::TILE_BYTES);

  const int n_tiles = (P + TP - 1) / TP;
  const long long total = (long long)n_ops * C * n_tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // This CTA's contiguous run of work items i = (operation, category, tile), tile fastest.  Items differ in cost by an
  // order of magnitude -- a child given as compact states is a column gather, a child with partials a 64^3 contraction
  // -- so the runs are cut by COST (2 + 3 per contracted child; measured at configs[2] fp64: 3.7 / 8.8 / 14 us per item
  // with 0 / 1 / 2 contracted children), not by count: with equal counts the SMs of a level were active 65 % of the
  // launch (profiles/r02_codon_post_tc_fp64.txt).
  __shared__ long long s_run[2];
  if (warp == 0) {
    const long long unit = (long long)C * n_tiles;
    auto weight = [&](int o) -> long long {
      if (o >= n_ops) return 0;
      int n = 0;
#pragma unroll
      for (int k = 0; k < 2; ++k) n += (ops[o].kind[k] == KIND_PARTIALS || ops[o].kind[k] == KIND_BCAST) ? 1 : 0;
      return 2 + 3 * n;
    };
    long long tot = 0;
    for (int base = 0; base < n_ops; base += 32) {
      long long w = weight(base + lane);
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) w += __shfl_xor_sync(0xffffffffu, w, d);
      tot += w;
    }
    tot *= unit;
    const long long pos[2] = {tot / gridDim.x * blockIdx.x + tot % gridDim.x * blockIdx.x / gridDim.x,
                              blockIdx.x + 1 == gridDim.x ? tot
                                                          : tot / gridDim.x * (blockIdx.x + 1) + tot % gridDim.x * (blockIdx.x + 1) / gridDim.x};
    if (lane < 2 && pos[lane] >= tot) s_run[lane] = total;
    long long prefix = 0;
    for (int base = 0; base < n_ops; base += 32) {
      const long long w = weight(base + lane), mine = w * unit;
      long long incl = mine;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const long long v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
      }
      const long long lo = prefix + incl - mine, hi = prefix + incl;
#pragma unroll
      for (int e = 0; e < 2; ++e)
        if (w > 0 && lo <= pos[e] && pos[e] < hi) s_run[e] = (long long)(base + lane) * unit + (pos[e] - lo) / w;
      prefix += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  const long long i0 = s_run[0], i1 = s_run[1];
  if (i0 >= i1) return;

  const int r = lane >> 2, c4 = lane & 3, m0 = warp * K::MT;

  auto issue = [&](long long i, int st) {
    const int tile = (int)(i % n_tiles);
    const long long oc = i / n_tiles;
    const int c = (int)(oc % C);
    const DevOp& o = ops[oc / C];
    const int p0 = tile * TP, n = P - p0 < TP ? P - p0 : TP;
    tc_load_operand_rows<T>(sX[st][0], o.kind[0], o.child[0], c, p0, n, P, m0, lane);
    tc_load_operand_rows<T>(sX[st][1], o.kind[1], o.child[1], c, p0, n, P, m0, lane);
  };
  // per-row scalars of an item, fetched one item ahead into registers: compact states and pending exponents
  struct RowMeta {
    int z[2][RPT], e[2][RPT];
  };
  auto fetch = [&](long long i, RowMeta& m) {
    const int tile = (int)(i % n_tiles);
    const DevOp& o = ops[i / n_tiles / C];
#pragma unroll
    for (int h = 0; h < RPT; ++h) {
      const int p = tile * TP + m0 + r + 8 * h;
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        m.z[k][h] = (o.kind[k] == KIND_STATES && p < P) ? static_cast<const uint8_t*>(o.child[k])[p] : 0;
        m.e[k][h] = pending_exp<T>(o.cscale[k], p, P, C);
      }
    }
  };
  issue(i0, 0);
  tc_cp_commit();
  RowMeta cur, nxt;
  fetch(i0, cur);
  long long cur_oc = -1;
  for (long long i = i0; i < i1; ++i) {
    const int st = (int)((i - i0) & 1);
    const int tile = (int)(i % n_tiles);
    const long long oc = i / n_tiles;
    const int c = (int)(oc % C);
    const DevOp o = ops[oc / C];
    const bool mma0 = o.kind[0] == KIND_PARTIALS || o.kind[0] == KIND_BCAST;
    const bool mma1 = o.kind[1] == KIND_PARTIALS || o.kind[1] == KIND_BCAST;
    const bool new_oc = oc != cur_oc;
    // Tile rows are warp-private (each warp stages and reads its own MT rows), so between items a warp only waits
    // for its own copies: the warps of a CTA drift apart and one warp's epilogue overlaps another's contraction.
    // The CTA meets at a barrier only when the (operation, category) run ends and the matrices are replaced.
    tc_cp_wait<0>();
    __syncwarp();
    if (new_oc) __syncthreads();
    if (new_oc) {
      tc_load_matrix<T>(sM[0], static_cast<const T*>(o.mat[0]) + (size_t)c * SP64 * SP64);
      tc_load_matrix<T>(sM[1], static_cast<const T*>(o.mat[1]) + (size_t)c * SP64 * SP64);
      tc_cp_commit();
    }
    if (i + 1 < i1) {
      issue(i + 1, st ^ 1);
      fetch(i + 1, nxt);
    }
    tc_cp_commit();
    if (new_oc) {
      tc_cp_wait<1>();  // the matrices (the older group); the next item's tiles stay in flight
      __syncthreads();
      if (sizeof(T) == 4) {
        tc_split_matrix(sM[0]);
        tc_split_matrix(sM[1]);
        __syncthreads();
      }
      cur_oc = oc;
    }
    const int p0 = tile * TP;
    T acc[2][8][K::CN];
    if (mma0) tc_gemm<false>(sX[st][0] + m0 * LD, sM[0], acc[0], r, c4);
    if (mma1) tc_gemm<false>(sX[st][1] + m0 * LD, sM[1], acc[1], r, c4);
#pragma unroll
    for (int h = 0; h < RPT; ++h) {
      const int p = p0 + m0 + r + 8 * h;
      const bool live = p < P;
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (o.kind[k] == KIND_STATES) {
          tc_gather<T>(sM[k], cur.z[k][h], S, T(1), h, c4, acc[k]);
        } else if (o.kind[k] == KIND_NONE) {
#pragma unroll
          for (int nt = 0; nt < 8; ++nt) acc[k][nt][h * 2] = acc[k][nt][h * 2 + 1] = T(0);
        }
      }
      const Pow2Pair<T> f0 = pow2_pair(-cur.e[0][h], T(0));
      const Pow2Pair<T> f1 = pow2_pair(-cur.e[1][h], T(0));
      T mx = T(0);
#pragma unroll
      for (int nt = 0; nt < 8; ++nt)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const T v = ((acc[0][nt][h * 2 + j] * f0.f1) * f0.f2) * ((acc[1][nt][h * 2 + j] * f1.f1) * f1.f2);
          acc[0][nt][h * 2 + j] = v;
          mx = fmax(mx, v);
        }
      mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
      mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
      if (live) {
        T* drow = static_cast<T*>(o.dest) + ((size_t)c * P + p) * SP64 + 2 * c4;
#pragma unroll
        for (int nt = 0; nt < 8; ++nt) {
          V2 v;
          v.x = acc[0][nt][h * 2];
          v.y = acc[0][nt][h * 2 + 1];
          *reinterpret_cast<V2*>(drow + nt * 8) = v;
        }
        if (c4 == 0 && o.scale != nullptr) static_cast<T*>(o.scale)[(size_t)c * P + p] = mx;
      }
    }
    cur = nxt;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// pre-order update of both children of one parent fused with both branch derivatives (
// PAPER.md:43, :101).  One CTA per (tile, item); the category loop runs inside so that num_p and den_p are complete
// when the CTA forms num_p / den_p.  Per category, with a_k = M_k x_k and x_k the child's post-order partials:
//   u_k = q_m o a_{1-k},  q_k = M_k^T u_k,  den = sum_s u_0[s] a_0[s],  num_k = sum_s q_k[s] (Q x_k)[s].
// u_k goes through shared memory (accumulator layout -> A-fragment layout) in the rows of the x_k tile, which only
// the owning warp touches, so a __syncwarp is the only barrier between the two products.
// ---------------------------------------------------------------------------------------------------------------
template <typename T>
constexpr size_t tc_pre_smem() {
  return 3 * (size_t)Tc<T>::MAT_BYTES + 3 * (size_t)Tc<T>::TILE_BYTES + 2 * Tc<T>::TP * sizeof(double);
}

template <typename T>
__global__ void __launch_bounds__(TC_THREADS, 1) k_pre_tc(const DevPreItem* __restrict__ items, int P, int S, int C,
                                                          const T* __restrict__ Qg, const double* __restrict__ catw,
                                                          const double* __restrict__ catr,
                                                          const double* __restrict__ weights,
                                                          double* __restrict__ grad_partial, int n_part,
                                                          double* __restrict__ site_out) {
  using K = Tc<T>;
  using V2 = typename Vec2Of<T>::type;
  constexpr int TP = Tc<T>::TP, RPT = Tc<T>::RPT;
  extern __shared__ __align__(16) unsigned char tc_smem[];
  T* sQ = reinterpret_cast<T*>(tc_smem);
  constexpr int LD = K::LD;
  constexpr size_t MB = K::MAT_BYTES, TB = K::TILE_BYTES;
  T* sM[2] = {reinterpret_cast<T*>(tc_smem + MB), reinterpret_cast<T*>(tc_smem + 2 * MB)};
  T* tQM = reinterpret_cast<T*>(tc_smem + 3 * MB);
  T* tX[2] = {reinterpret_cast<T*>(tc_smem + 3 * MB + TB), reinterpret_cast<T*>(tc_smem + 3 * MB + 2 * TB)};
  double* sRed = reinterpret_cast<double*>(tc_smem + 3 * MB + 3 * TB);  // [2][TP]

  const DevPreItem it = items[blockIdx.y];
  const int p0 = blockIdx.x * TP, n = P - p0 < TP ? P - p0 : TP;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r = lane >> 2, c4 = lane & 3, m0 = warp * K::MT;
  const bool want[2] = {it.slot[0] >= 0, it.slot[1] >= 0};
  const bool need_q[2] = {it.q[0] != nullptr || want[0], it.q[1] != nullptr || want[1]};
  const bool mma_x[2] = {it.kind[0] == KIND_PARTIALS || it.kind[0] == KIND_BCAST,
                         it.kind[1] == KIND_PARTIALS || it.kind[1] == KIND_BCAST};

  if (want[0] || want[1]) tc_load_matrix<T>(sQ, Qg);  // joins the first category's cp.async group

  int z[2][RPT];
  Pow2Pair<T> fx[2][RPT], fq[RPT];
  double num[2][RPT], den[RPT];
#pragma unroll
  for (int h = 0; h < RPT; ++h) {
    const int p = p0 + m0 + r + 8 * h;
    fq[h] = pow2_pair(-pending_exp<T>(it.qm_scale, p, P, C), T(0));
    den[h] = 0.0;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      z[k][h] = (it.kind[k] == KIND_STATES && p < P) ? static_cast<const uint8_t*>(it.p[k])[p] : 0;
      fx[k][h] = pow2_pair(-pending_exp<T>(it.p_scale[k], p, P, C), T(0));
      num[k][h] = 0.0;
    }
  }

  // Staging of category c+1 is spread over category c: each buffer is refilled (cp.async) as soon as a barrier
  // says every warp is done with it -- q_m after the u_k have been formed, M_k and the x_k tile after q_k.
  auto stage_child = [&](int k, int c) {
    tc_load_operand<T>(tX[k], it.kind[k], it.p[k], c, p0, n, P);
    tc_load_matrix<T>(sM[k], static_cast<const T*>(it.mat[k]) + (size_t)c * SP64 * SP64);
  };
  tc_load_operand<T>(tQM, KIND_PARTIALS, it.qm, 0, p0, n, P);
  stage_child(0, 0);
  stage_child(1, 0);
  tc_cp_commit();
  for (int c = 0; c < C; ++c) {
    const bool more = c + 1 < C;
    tc_cp_wait<0>();
    __syncthreads();
    if (sizeof(T) == 4) {
      if (c == 0 && (want[0] || want[1])) tc_split_matrix(sQ);
      tc_split_matrix(sM[0]);
      tc_split_matrix(sM[1]);
      __syncthreads();
    }

    T a[2][8][K::CN], qx[2][8][K::CN];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      if (mma_x[k]) {
        if (want[k]) tc_gemm<false>(tX[k] + m0 * LD, sQ, qx[k], r, c4);
        tc_gemm<false>(tX[k] + m0 * LD, sM[k], a[k], r, c4);
      } else {
#pragma unroll
        for (int h = 0; h < RPT; ++h) {
          if (it.kind[k] == KIND_STATES) {
            tc_gather<T>(sM[k], z[k][h], S, T(1), h, c4, a[k]);
            if (want[k]) tc_gather<T>(sQ, z[k][h], S, T(0), h, c4, qx[k]);
          } else {
#pragma unroll
            for (int nt = 0; nt < 8; ++nt)
              a[k][nt][h * 2] = a[k][nt][h * 2 + 1] = qx[k][nt][h * 2] = qx[k][nt][h * 2 + 1] = T(0);
          }
        }
      }
    }
    __syncwarp();  // the warp's rows of tX[0], tX[1] have been read; they now receive u_0, u_1
    const double cw = catw[c], cwr = catw[c] * catr[c];
#pragma unroll
    for (int h = 0; h < RPT; ++h) {
      const int row = m0 + r + 8 * h;
      T dd = T(0);
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        const int col = nt * 8 + 2 * c4;
        const V2 qv = *reinterpret_cast<const V2*>(tQM + row * LD + col);
        const T qm[2] = {(qv.x * fq[h].f1) * fq[h].f2, (qv.y * fq[h].f1) * fq[h].f2};
        V2 u0, u1;
        T t0[2], t1[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const T a0 = (a[0][nt][h * 2 + j] * fx[0][h].f1) * fx[0][h].f2;
          const T a1 = (a[1][nt][h * 2 + j] * fx[1][h].f1) * fx[1][h].f2;
          t0[j] = qm[j] * a1;
          t1[j] = qm[j] * a0;
          dd = fma(t0[j], a0, dd);
        }
        u0.x = t0[0]; u0.y = t0[1];
        u1.x = t1[0]; u1.y = t1[1];
        *reinterpret_cast<V2*>(tX[0] + row * LD + col) = u0;
        *reinterpret_cast<V2*>(tX[1] + row * LD + col) = u1;
      }
      den[h] = fma(cw, (double)dd, den[h]);
    }
    __syncwarp();
    if (more) {
      __syncthreads();
      tc_load_operand<T>(tQM, KIND_PARTIALS, it.qm, c + 1, p0, n, P);
      tc_cp_commit();
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      if (need_q[k]) {
      tc_gemm<true>(tX[k] + m0 * LD, sM[k], a[k], r, c4);  // a[k] <- q_k
#pragma unroll
      for (int h = 0; h < RPT; ++h) {
        const int p = p0 + m0 + r + 8 * h;
        T mx = T(0), nn = T(0);
#pragma unroll
        for (int nt = 0; nt < 8; ++nt)
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            mx = fmax(mx, a[k][nt][h * 2 + j]);
            if (want[k]) nn = fma(a[k][nt][h * 2 + j], (qx[k][nt][h * 2 + j] * fx[k][h].f1) * fx[k][h].f2, nn);
          }
        if (want[k]) num[k][h] = fma(cwr, (double)nn, num[k][h]);
        if (it.q[k] != nullptr) {
          mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
          mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
          if (p < P) {
            T* drow = static_cast<T*>(it.q[k]) + ((size_t)c * P + p) * SP64 + 2 * c4;
#pragma unroll
            for (int nt = 0; nt < 8; ++nt) {
              V2 v;
              v.x = a[k][nt][h * 2];
              v.y = a[k][nt][h * 2 + 1];
              *reinterpret_cast<V2*>(drow + nt * 8) = v;
            }
            if (c4 == 0) static_cast<T*>(it.q_scale[k])[(size_t)c * P + p] = mx;
          }
        }
      }
      }
      if (more) {
        __syncthreads();
        stage_child(k, c + 1);
        tc_cp_commit();
      }
    }
  }

  if (!(want[0] || want[1])) return;
#pragma unroll
  for (int h = 0; h < RPT; ++h) {
    const int row = m0 + r + 8 * h, p = p0 + row;
    double d = den[h];
    d += __shfl_xor_sync(0xffffffffu, d, 1);
    d += __shfl_xor_sync(0xffffffffu, d, 2);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      double v = num[k][h];
      v += __shfl_xor_sync(0xffffffffu, v, 1);
      v += __shfl_xor_sync(0xffffffffu, v, 2);
      if (c4 == 0) {
        double contrib = 0.0;
        if (want[k] && p < P) {
          const double ratio = v / d;
          if (site_out != nullptr) site_out[(size_t)it.slot[k] * P + p] = ratio;
          contrib = weights[p] * ratio;
        }
        sRed[k * TP + row] = contrib;
      }
    }
  }
  __syncthreads();
  if (warp < 2 && want[warp]) {  // warp k sums child k's TP contributions in a fixed order
    double v = 0.0;
    for (int i = lane; i < TP; i += 32) v += sRed[warp * TP + i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) grad_partial[(size_t)it.slot[warp] * n_part + blockIdx.x] = v;
  }
}

// ---- host-side launchers (called from plk_api.cu) ---------------------------------------------------------------
template <typename T>
int tc_launch_post(cudaStream_t stream, const DevOp* d_ops, int n_ops, int P, int S, int C, int sm_count,
                   int64_t* launches) {
  // per device and cheap: no process-wide "done" flag (instances may live on several GPUs)
  if (cudaFuncSetAttribute(k_post_tc<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_post_smem<T>()) != cudaSuccess)
    return PLK_ERR_CUDA;
  const int n_tiles = (P + Tc<T>::TP - 1) / Tc<T>::TP;
  const long long total = (long long)n_ops * C * n_tiles;
  if (total <= 0) return PLK_SUCCESS;
  const int grid = total < sm_count ? (int)total : sm_count;
  k_post_tc<T><<<grid, TC_THREADS, tc_post_smem<T>(), stream>>>(d_ops, n_ops, P, S, C);
  if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
  ++*launches;
  return PLK_SUCCESS;
}

// returns the number of partial sums per gradient slot through *n_parts (row stride stays n_part)
template <typename T>
int tc_launch_pre(cudaStream_t stream, const DevPreItem* d_items, int n, int P, int S, int C, const T* Q,
                  const double* catw, const double* catr, const double* weights, double* grad_partial, int n_part,
                  double* site, int* n_parts, int64_t* launches) {
  // per device and cheap: no process-wide "done" flag (instances may live on several GPUs)
  if (cudaFuncSetAttribute(k_pre_tc<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tc_pre_smem<T>()) !=
      cudaSuccess)
    return PLK_ERR_CUDA;
  const int n_tiles = (P + Tc<T>::TP - 1) / Tc<T>::TP;
  *n_parts = n_tiles;
  if (n <= 0) return PLK_SUCCESS;
  dim3 grid(n_tiles, n);
  k_pre_tc<T><<<grid, TC_THREADS, tc_pre_smem<T>(), stream>>>(d_items, P, S, C, Q, catw, catr, weights, grad_partial,
                                                             n_part, site);
  if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
  ++*launches;
  return PLK_SUCCESS;
}

}  // namespace plk
