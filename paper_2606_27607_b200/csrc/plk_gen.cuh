// plk_gen.cuh -- CUDA-core kernels for state counts padded to SP = 64 (61-state codon models): the comparison arm
// BASELINE.json configs[2] asks for ("CUDA-core vs tensor-core partials update") and the path used when the
// instance was created without PLK_FLAG_TENSOR_CORES -- and, instantiated with SP = 32, the kernels of the 20-state
// amino-acid models (5..32 states): a quarter of the flops and half of the bytes of
// padding them to 64.  Everything below is templated on the padded state count SP (a multiple of 32), default 64.
//
// A block of 256 threads handles one (operation, category, tile of 32 patterns).  Thread (pp = tid / 8, sb = tid % 8)
// owns 8 output states of pattern pp: chunks of VEC = 16 / sizeof(T) consecutive states, interleaved over sb so that
// the 8 lanes of one pattern read 128 contiguous bytes of a matrix row from shared memory (conflict-free 128-bit
// loads) while the operand value is a broadcast.  Matrices are staged in shared memory as A[x][s] (i.e. transposed
// on load for M.x, natural for M^T.x).
//
// Rescaling is DEFERRED: a node stores its partials unscaled together with
// mx[c][p] = max_s p[c][p][s]; whoever reads the node multiplies M.x by 2^-e, e = exponent of max_c mx[c][p].
// This keeps the (operation, category, tile) work items independent of one another.
#pragma once
#include "plk_common.cuh"

namespace plk {

constexpr int SP64 = 64;
constexpr int GEN_TP = 32;        // patterns per tile
constexpr int GEN_THREADS = 256;  // 32 patterns x 8 state-lanes

template <typename T, int SP = SP64>
struct Gen {
  static constexpr int VEC = 16 / sizeof(T);  // 4 (fp32) or 2 (fp64)
  static constexpr int NPT = SP / 8;          // states per thread (8 lanes share a pattern)
  static constexpr int NCH = NPT / VEC;       // chunks per thread
  static constexpr int TS = SP + VEC;         // padded tile row stride
  static_assert(SP % 32 == 0 && NCH >= 1, "padded state count");
};
template <typename T>
struct VecOf;
template <>
struct VecOf<float> {
  using type = float4;
};
template <>
struct VecOf<double> {
  using type = double2;
};

__device__ __forceinline__ void unpack(const float4& v, float* o) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
__device__ __forceinline__ void unpack(const double2& v, double* o) { o[0] = v.x; o[1] = v.y; }
__device__ __forceinline__ float4 pack(const float* o, float4) { return make_float4(o[0], o[1], o[2], o[3]); }
__device__ __forceinline__ double2 pack(const double* o, double2) { return make_double2(o[0], o[1]); }

// state owned by (sb, chunk i, element j)
template <typename T>
__device__ __forceinline__ int state_of(int sb, int i, int j) {
  return (Gen<T>::VEC * 8) * i + Gen<T>::VEC * sb + j;
}

// A[x][s] <- transpose ? M[s][x] : M[x][s]    (M row-major [64][64] in global memory)
template <typename T, int SP = SP64>
__device__ __forceinline__ void fill_matrix(T* __restrict__ A, const T* __restrict__ M, bool transpose) {
  for (int idx = threadIdx.x; idx < SP * SP; idx += GEN_THREADS) {
    const T v = M[idx];
    const int r = idx / SP, col = idx % SP;
    if (transpose) A[col * SP + r] = v; else A[idx] = v;
  }
}

// tile[pp][x] for patterns p0..p0+31 of one operand; rows beyond P are zero
template <typename T, int SP = SP64>
__device__ __forceinline__ void load_tile(T* __restrict__ tile, int kind, const void* ptr, int c, int p0, int P, int S) {
  constexpr int VEC = Gen<T, SP>::VEC, TS = Gen<T, SP>::TS, CPR = SP / VEC;  // chunks per row
  using V = typename VecOf<T>::type;
  if (kind == KIND_NONE) {
    for (int idx = threadIdx.x; idx < GEN_TP * TS; idx += GEN_THREADS) tile[idx] = T(0);
  } else if (kind == KIND_STATES) {
    const uint8_t* st = static_cast<const uint8_t*>(ptr);
    for (int idx = threadIdx.x; idx < GEN_TP * SP; idx += GEN_THREADS) {
      const int row = idx / SP, x = idx % SP;
      T v = T(0);
      if (p0 + row < P) {
        const int z = st[p0 + row];
        v = (z >= S) ? (x < S ? T(1) : T(0)) : (x == z ? T(1) : T(0));
      }
      tile[row * TS + x] = v;
    }
  } else {
    const T* base = static_cast<const T*>(ptr) + (kind == KIND_BCAST ? (size_t)0 : (size_t)c * P * SP);
    for (int idx = threadIdx.x; idx < GEN_TP * CPR; idx += GEN_THREADS) {
      const int row = idx / CPR, ch = idx % CPR;
      T tmp[VEC];
      if (p0 + row < P) {
        unpack(*reinterpret_cast<const V*>(base + (size_t)(p0 + row) * SP + ch * VEC), tmp);
      } else {
#pragma unroll
        for (int j = 0; j < VEC; ++j) tmp[j] = T(0);
      }
#pragma unroll
      for (int j = 0; j < VEC; ++j) tile[row * TS + ch * VEC + j] = tmp[j];
    }
  }
}

// pending per-pattern exponent of an operand (deferred rescaling); 0 when it carries none
template <typename T>
__device__ __forceinline__ int pending_exp(const void* mx, int p, int P, int C) {
  if (mx == nullptr || p >= P) return 0;
  const T* m = static_cast<const T*>(mx);
  T v = T(0);
  for (int c = 0; c < C; ++c) v = fmax(v, m[(size_t)c * P + p]);
  return exp_of(v);
}

// acc[i*VEC+j] = sum_x A[x][state_of(sb,i,j)] * vrow[x]
template <typename T, int SP = SP64>
__device__ __forceinline__ void mv64(const T* __restrict__ A, const T* __restrict__ vrow, int sb, T (&acc)[Gen<T, SP>::NPT]) {
  constexpr int VEC = Gen<T, SP>::VEC, NCH = Gen<T, SP>::NCH;
  using V = typename VecOf<T>::type;
#pragma unroll
  for (int k = 0; k < Gen<T, SP>::NPT; ++k) acc[k] = T(0);
#pragma unroll 4
  for (int x = 0; x < SP; ++x) {
    const T v = vrow[x];
#pragma unroll
    for (int i = 0; i < NCH; ++i) {
      T a[VEC];
      unpack(*reinterpret_cast<const V*>(A + x * SP + (VEC * 8) * i + VEC * sb), a);
#pragma unroll
      for (int j = 0; j < VEC; ++j) acc[i * VEC + j] = fma(a[j], v, acc[i * VEC + j]);
    }
  }
}

// acc = column z of the matrix (row z of A[x][s]); a missing state gives `missing` for real states, 0 for padding
template <typename T, int SP = SP64>
__device__ __forceinline__ void gather64(const T* __restrict__ A, int z, int S, T missing, int sb, T (&acc)[Gen<T, SP>::NPT]) {
  constexpr int VEC = Gen<T, SP>::VEC, NCH = Gen<T, SP>::NCH;
#pragma unroll
  for (int i = 0; i < NCH; ++i)
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
      const int s = state_of<T>(sb, i, j);
      acc[i * VEC + j] = z < S ? A[z * SP + s] : (s < S ? missing : T(0));
    }
}

// store the owned states of pattern p to dst[p][.] (row stride SP)
template <typename T, int SP = SP64>
__device__ __forceinline__ void store_states(T* __restrict__ dst_row, int sb, const T (&acc)[Gen<T, SP>::NPT]) {
  constexpr int VEC = Gen<T, SP>::VEC, NCH = Gen<T, SP>::NCH;
  using V = typename VecOf<T>::type;
#pragma unroll
  for (int i = 0; i < NCH; ++i)
    *reinterpret_cast<V*>(dst_row + (VEC * 8) * i + VEC * sb) = pack(acc + i * VEC, V());
}

template <typename T>
__device__ __forceinline__ T lane8_max(T v) {
  v = fmax(v, __shfl_xor_sync(0xffffffffu, v, 1));
  v = fmax(v, __shfl_xor_sync(0xffffffffu, v, 2));
  v = fmax(v, __shfl_xor_sync(0xffffffffu, v, 4));
  return v;
}
template <typename T>
__device__ __forceinline__ T lane8_sum(T v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  return v;
}

template <typename T, int SP = SP64>
constexpr size_t pre64_smem() {
  return (3 * SP * SP + 5 * GEN_TP * Gen<T, SP>::TS) * sizeof(T) + 3 * GEN_TP * sizeof(int) +
         4 * GEN_TP * sizeof(double);
}
template <typename T, int SP = SP64>
constexpr size_t deriv64_smem() {
  return (SP * SP + 2 * GEN_TP * Gen<T, SP>::TS) * sizeof(T) + 2 * GEN_TP * sizeof(double);
}

// ---------------------------------------------------------------------------------------------------------------
// post-order update, register-tiled (round 2).  The first version (k_post64, removed) gave a thread 8 states
// of ONE pattern, so every FMA needs its own shared-memory operand: 17 shared-memory wavefronts per 8 warp-FMAs, i.e.
// the kernel is bound by shared memory at ~7 % of the fp64 FMA rate.  Here a thread owns 4 patterns x 8 states of a
// tile of PT patterns (PT / 4 x SP / 8 = 128 threads): per contraction index x it reads 8 matrix values and 4 operand
// values for 32 FMAs.  Layouts chosen so that no load conflicts: the matrix row A[x][.] (A[x][s] = M[s][x]) is stored in
// 16-byte chunks interleaved as (chunk i of state group sg) -> position i * NSG + sg, so the lanes of a quarter warp
// (distinct sg) read consecutive chunks; the operand tile is transposed to Vt[x][p] with an odd row stride, read as
// broadcasts.  The two children go through the same buffers one after the other; a compact-tip child is a row gather.
// Same arithmetic per output as before (sum over x in increasing order, deferred rescaling).
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int SP>
struct GenT {
  static constexpr int VEC = 16 / sizeof(T);       // elements per 16-byte chunk
  static constexpr int NSG = SP / 8;               // state groups (8 states each)
  static constexpr int PT = 128 * 4 / NSG;         // patterns per tile: 64 (SP = 64), 128 (SP = 32)
  static constexpr int NCH = 8 / VEC;              // chunks per thread and matrix row
  static constexpr int LDV = PT + 1;               // operand tile row stride (odd: conflict-free transposing stores)
  static constexpr size_t SMEM = ((size_t)SP * SP + (size_t)SP * LDV) * sizeof(T) + 2 * PT * sizeof(int);
};

template <typename T, int SP = SP64>
__global__ void __launch_bounds__(128) k_post64t(const DevOp* __restrict__ ops, int P, int S, int C) {
  using G = GenT<T, SP>;
  using V = typename VecOf<T>::type;
  constexpr int VEC = G::VEC, NSG = G::NSG, PT = G::PT, NCH = G::NCH, LDV = G::LDV;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* A = reinterpret_cast<T*>(smem_raw);  // [SP][SP], chunk-interleaved rows
  T* Vt = A + SP * SP;                    // [SP][LDV]
  int* sE = reinterpret_cast<int*>(Vt + SP * LDV);  // [2][PT] pending exponents of the children

  const DevOp op = ops[blockIdx.z];
  const int c = blockIdx.y, p0 = blockIdx.x * PT;
  const int sg = threadIdx.x % NSG, pg = threadIdx.x / NSG;  // states 8 sg .., patterns p0 + 4 pg ..
  for (int i = threadIdx.x; i < 2 * PT; i += 128) sE[i] = pending_exp<T>(op.cscale[i / PT], p0 + i % PT, P, C);

  T acc[2][4][8];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    __syncthreads();  // the previous child's buffers are no longer read
    // matrix of child k: A[x][s] = M[s][x]; element (x, s) at A[x * SP + ((s % 8) / VEC * NSG + s / 8) * VEC + s % VEC]
    // (filled in VEC x VEC blocks: 16-byte loads of VEC rows of M, 16-byte stores of VEC rows of A to consecutive
    // chunk positions -- a scalar transposing copy would store at a stride of a whole row: 32-way bank conflicts)
    const T* M = static_cast<const T*>(op.mat[k]) + (size_t)c * SP * SP;
    constexpr int CPR = SP / VEC;
    for (int idx = threadIdx.x; idx < CPR * CPR; idx += 128) {
      const int pos = idx % CPR, xc = idx / CPR;     // chunk position inside the rows of A; chunk of x
      const int cs = (pos % NSG) * NCH + pos / NSG;  // the chunk of states stored at that position
      T blk[VEC][VEC];
#pragma unroll
      for (int j = 0; j < VEC; ++j) unpack(*reinterpret_cast<const V*>(M + (size_t)(cs * VEC + j) * SP + xc * VEC), blk[j]);
#pragma unroll
      for (int i = 0; i < VEC; ++i) {
        T o[VEC];
#pragma unroll
        for (int j = 0; j < VEC; ++j) o[j] = blk[j][i];
        *reinterpret_cast<V*>(A + (xc * VEC + i) * SP + pos * VEC) = pack(o, V());
      }
    }
    const int kind = op.kind[k];
    if (kind == KIND_PARTIALS || kind == KIND_BCAST) {  // operand tile, transposed: lane = pattern, loop over chunks
      const T* base = static_cast<const T*>(op.child[k]) + (kind == KIND_BCAST ? (size_t)0 : (size_t)c * P * SP);
      for (int idx = threadIdx.x; idx < PT * (SP / VEC); idx += 128) {
        const int pp = idx % PT, ch = idx / PT;
        T tmp[VEC];
        if (p0 + pp < P) {
          unpack(*reinterpret_cast<const V*>(base + (size_t)(p0 + pp) * SP + ch * VEC), tmp);
        } else {
#pragma unroll
          for (int j = 0; j < VEC; ++j) tmp[j] = T(0);
        }
#pragma unroll
        for (int j = 0; j < VEC; ++j) Vt[(ch * VEC + j) * LDV + pp] = tmp[j];
      }
    }
    __syncthreads();
    if (kind == KIND_STATES) {  // column z of M = row z of A; a missing state: 1 for real states
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int p = p0 + 4 * pg + i;
        const int z = p < P ? static_cast<const uint8_t*>(op.child[k])[p] : S;
#pragma unroll
        for (int q = 0; q < NCH; ++q) {
          T a[VEC];
          unpack(*reinterpret_cast<const V*>(A + (z < S ? z : 0) * SP + (q * NSG + sg) * VEC), a);
#pragma unroll
          for (int j = 0; j < VEC; ++j) {
            const int s = 8 * sg + q * VEC + j;
            acc[k][i][q * VEC + j] = z < S ? a[j] : (s < S ? T(1) : T(0));
          }
        }
      }
    } else if (kind == KIND_NONE) {
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[k][i][j] = T(0);
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[k][i][j] = T(0);
      const T* vrow = Vt + 4 * pg;
      const T* arow = A + sg * VEC;
#pragma unroll 2
      for (int x = 0; x < SP; ++x) {
        T a[8], v[4];
#pragma unroll
        for (int q = 0; q < NCH; ++q) unpack(*reinterpret_cast<const V*>(arow + x * SP + q * NSG * VEC), a + q * VEC);
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = vrow[x * LDV + i];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 8; ++j) acc[k][i][j] = fma(a[j], v[i], acc[k][i][j]);
      }
    }
  }
  // product of the two children with their pending factors, per-pattern maximum, store
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int pl = 4 * pg + i, p = p0 + pl;
    const Pow2Pair<T> f0 = pow2_pair(-sE[pl], T(0)), f1 = pow2_pair(-sE[PT + pl], T(0));
    T mx = T(0);
    T out[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      out[j] = ((acc[0][i][j] * f0.f1) * f0.f2) * ((acc[1][i][j] * f1.f1) * f1.f2);
      mx = fmax(mx, out[j]);
    }
#pragma unroll
    for (int o = 1; o < NSG; o <<= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (p < P) {
      T* drow = static_cast<T*>(op.dest) + ((size_t)c * P + p) * SP + 8 * sg;
#pragma unroll
      for (int q = 0; q < NCH; ++q) *reinterpret_cast<V*>(drow + q * VEC) = pack(out + q * VEC, V());
      if (sg == 0 && op.scale != nullptr) static_cast<T*>(op.scale)[(size_t)c * P + p] = mx;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// pre-order update of both children of one parent + both branch derivatives
// one (tile, item) per block, categories looped inside so that num_p and den_p are summed over c in the block
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int SP = SP64>
__global__ void __launch_bounds__(GEN_THREADS) k_pre64(const DevPreItem* __restrict__ items, int P, int S, int C,
                                                       const T* __restrict__ Qg, const double* __restrict__ catw,
                                                       const double* __restrict__ catr,
                                                       const double* __restrict__ weights,
                                                       double* __restrict__ grad_partial, int n_tiles,
                                                       double* __restrict__ site_out) {
  constexpr int TS = Gen<T, SP>::TS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* B0 = reinterpret_cast<T*>(smem_raw);
  T* B1 = B0 + SP * SP;
  T* BQ = B1 + SP * SP;
  T* tQM = BQ + SP * SP;
  T* tX[2] = {tQM + GEN_TP * TS, tQM + 2 * GEN_TP * TS};
  T* tU[2] = {tQM + 3 * GEN_TP * TS, tQM + 4 * GEN_TP * TS};
  int* sE = reinterpret_cast<int*>(tQM + 5 * GEN_TP * TS);              // [3][32]: child0, child1, parent q
  double* sNum = reinterpret_cast<double*>(sE + 3 * GEN_TP + (GEN_TP & 1));  // [2][32]
  double* sDen = sNum + 2 * GEN_TP;

  const DevPreItem it = items[blockIdx.y];
  const int p0 = blockIdx.x * GEN_TP;
  const int pp = threadIdx.x >> 3, sb = threadIdx.x & 7, p = p0 + pp;
  const bool want_grad = it.slot[0] >= 0 || it.slot[1] >= 0;
  T* B[2] = {B0, B1};

  if (want_grad) fill_matrix<T, SP>(BQ, Qg, true);
  if (threadIdx.x < 3 * GEN_TP) {
    const int k = threadIdx.x / GEN_TP, r = threadIdx.x % GEN_TP;
    sE[threadIdx.x] = pending_exp<T>(k == 2 ? it.qm_scale : it.p_scale[k], p0 + r, P, C);
  }
  if (threadIdx.x < 4 * GEN_TP) sNum[threadIdx.x] = 0.0;  // sNum and sDen are contiguous

  int z[2] = {0, 0};
#pragma unroll
  for (int k = 0; k < 2; ++k)
    if (it.kind[k] == KIND_STATES && p < P) z[k] = static_cast<const uint8_t*>(it.p[k])[p];

  for (int c = 0; c < C; ++c) {
    __syncthreads();
    fill_matrix<T, SP>(B0, static_cast<const T*>(it.mat[0]) + (size_t)c * SP * SP, true);
    fill_matrix<T, SP>(B1, static_cast<const T*>(it.mat[1]) + (size_t)c * SP * SP, true);
    load_tile<T, SP>(tQM, KIND_PARTIALS, it.qm, c, p0, P, S);
    load_tile<T, SP>(tX[0], it.kind[0], it.p[0], c, p0, P, S);
    load_tile<T, SP>(tX[1], it.kind[1], it.p[1], c, p0, P, S);
    __syncthreads();

    T a[2][Gen<T, SP>::NPT], qx[2][Gen<T, SP>::NPT];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      if (it.kind[k] == KIND_STATES) {
        gather64<T, SP>(B[k], z[k], S, T(1), sb, a[k]);
        if (want_grad) gather64<T, SP>(BQ, z[k], S, T(0), sb, qx[k]);
      } else {
        mv64<T, SP>(B[k], tX[k] + pp * TS, sb, a[k]);
        if (want_grad) mv64<T, SP>(BQ, tX[k] + pp * TS, sb, qx[k]);
      }
      const Pow2Pair<T> f = pow2_pair(-sE[k * GEN_TP + pp], T(0));
#pragma unroll
      for (int i = 0; i < Gen<T, SP>::NPT; ++i) a[k][i] = (a[k][i] * f.f1) * f.f2;
    }
    {
      const Pow2Pair<T> f = pow2_pair(-sE[2 * GEN_TP + pp], T(0));
#pragma unroll
      for (int i = 0; i < Gen<T, SP>::NCH; ++i)
#pragma unroll
        for (int j = 0; j < Gen<T, SP>::VEC; ++j) {
          const int s = state_of<T>(sb, i, j);
          const T qm = (tQM[pp * TS + s] * f.f1) * f.f2;
          tU[0][pp * TS + s] = qm * a[1][i * Gen<T, SP>::VEC + j];
          tU[1][pp * TS + s] = qm * a[0][i * Gen<T, SP>::VEC + j];
        }
    }
    __syncthreads();
    fill_matrix<T, SP>(B0, static_cast<const T*>(it.mat[0]) + (size_t)c * SP * SP, false);
    fill_matrix<T, SP>(B1, static_cast<const T*>(it.mat[1]) + (size_t)c * SP * SP, false);
    __syncthreads();

#pragma unroll
    for (int k = 0; k < 2; ++k) {
      T q[Gen<T, SP>::NPT];
      mv64<T, SP>(B[k], tU[k] + pp * TS, sb, q);
      T mx = T(0);
#pragma unroll
      for (int i = 0; i < Gen<T, SP>::NPT; ++i) mx = fmax(mx, q[i]);
      mx = lane8_max(mx);
      if (it.q[k] != nullptr && p < P) {
        store_states<T, SP>(static_cast<T*>(it.q[k]) + ((size_t)c * P + p) * SP, sb, q);
        if (sb == 0) static_cast<T*>(it.q_scale[k])[(size_t)c * P + p] = mx;
      }
      if (it.slot[k] >= 0) {
        T n = T(0), d = T(0);
#pragma unroll
        for (int i = 0; i < Gen<T, SP>::NCH; ++i)
#pragma unroll
          for (int j = 0; j < Gen<T, SP>::VEC; ++j) {
            const int s = state_of<T>(sb, i, j);
            n = fma(q[i * Gen<T, SP>::VEC + j], qx[k][i * Gen<T, SP>::VEC + j], n);
            d = fma(q[i * Gen<T, SP>::VEC + j], tX[k][pp * TS + s], d);
          }
        n = lane8_sum(n);
        d = lane8_sum(d);
        if (sb == 0) {  // one writer per (k, pp): no race
          sNum[k * GEN_TP + pp] += catw[c] * catr[c] * (double)n;
          sDen[k * GEN_TP + pp] += catw[c] * (double)d;
        }
      }
    }
  }
  __syncthreads();
  if (want_grad && threadIdx.x < 2 * GEN_TP) {  // warp 0 -> child 0, warp 1 -> child 1
    const int k = threadIdx.x / GEN_TP, r = threadIdx.x % GEN_TP;
    double v = 0.0;
    if (it.slot[k] >= 0 && p0 + r < P) {
      const double ratio = sNum[k * GEN_TP + r] / sDen[k * GEN_TP + r];
      if (site_out != nullptr) site_out[(size_t)it.slot[k] * P + p0 + r] = ratio;
      v = weights[p0 + r] * ratio;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (r == 0 && it.slot[k] >= 0) grad_partial[(size_t)it.slot[k] * n_tiles + blockIdx.x] = v;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// unfused branch derivatives from stored pre- and post-order partials
// ---------------------------------------------------------------------------------------------------------------
template <typename T, int SP = SP64>
__global__ void __launch_bounds__(GEN_THREADS) k_deriv64(const DevBranch* __restrict__ br, int P, int S, int C,
                                                         const T* __restrict__ Qg, const double* __restrict__ catw,
                                                         const double* __restrict__ catr,
                                                         const double* __restrict__ weights,
                                                         double* __restrict__ grad_partial, int n_tiles,
                                                         double* __restrict__ site_out) {
  constexpr int TS = Gen<T, SP>::TS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* BQ = reinterpret_cast<T*>(smem_raw);
  T* tQ = BQ + SP * SP;
  T* tX = tQ + GEN_TP * TS;
  double* sNum = reinterpret_cast<double*>(tX + GEN_TP * TS);
  double* sDen = sNum + GEN_TP;

  const DevBranch b = br[blockIdx.y];
  const int p0 = blockIdx.x * GEN_TP;
  const int pp = threadIdx.x >> 3, sb = threadIdx.x & 7;
  fill_matrix<T, SP>(BQ, Qg, true);
  if (threadIdx.x < 2 * GEN_TP) sNum[threadIdx.x] = 0.0;
  for (int c = 0; c < C; ++c) {
    __syncthreads();
    load_tile<T, SP>(tQ, KIND_PARTIALS, b.q, c, p0, P, S);
    load_tile<T, SP>(tX, b.kind, b.p, c, p0, P, S);
    __syncthreads();
    T qx[Gen<T, SP>::NPT];
    mv64<T, SP>(BQ, tX + pp * TS, sb, qx);
    T n = T(0), d = T(0);
#pragma unroll
    for (int i = 0; i < Gen<T, SP>::NCH; ++i)
#pragma unroll
      for (int j = 0; j < Gen<T, SP>::VEC; ++j) {
        const int s = state_of<T>(sb, i, j);
        n = fma(tQ[pp * TS + s], qx[i * Gen<T, SP>::VEC + j], n);
        d = fma(tQ[pp * TS + s], tX[pp * TS + s], d);
      }
    n = lane8_sum(n);
    d = lane8_sum(d);
    if (sb == 0) {
      sNum[pp] += catw[c] * catr[c] * (double)n;
      sDen[pp] += catw[c] * (double)d;
    }
  }
  __syncthreads();
  if (threadIdx.x < GEN_TP) {
    const int r = threadIdx.x;
    double v = 0.0;
    if (p0 + r < P) {
      const double ratio = sNum[r] / sDen[r];
      if (site_out != nullptr) site_out[(size_t)b.slot * P + p0 + r] = ratio;
      v = weights[p0 + r] * ratio;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (r == 0) grad_partial[(size_t)b.slot * n_tiles + blockIdx.x] = v;
  }
}

}  // namespace plk
