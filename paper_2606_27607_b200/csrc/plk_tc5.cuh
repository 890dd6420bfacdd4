// plk_tc5.cuh -- fp32 codon (61 states padded to SP = 64) post-order kernel on the 5th-generation tensor cores:
// tcgen05.mma.kind::tf32 with accumulators in tensor memory (TMEM), sm_100a only.
//
// What it computes (SURVEY 8(a) steps 2-3; PAPER.md:27 pruning, :59/:71 tensor cores for codon models): for one work
// item (operation, category c, tile of 128 patterns) and each child k
//     D_k[p][s] = sum_x X_k[p][x] * M_k[s][x]                      (X_k: child partials, M_k: transition matrix)
//     dest[p][s] = (D_0[p][s] 2^-e0[p]) * (D_1[p][s] 2^-e1[p]),    mx[c][p] = max_s dest[p][s]   (deferred rescaling)
// exactly the arithmetic of k_post_tc<float> (plk_tc.cuh): split TF32, x = hi + lo with hi = tf32(x),
// lo = tf32(x - hi), x.m ~= lo.hi + hi.lo + hi.hi accumulated in fp32 (dropped term 2^-22 relative).
//
// Mapping onto tcgen05.  A = X_k tile, 128 x 64, K-major (a pattern row of the [c][p][s] HBM layout IS a K-major
// operand row); B = M_k, 64 x 64, K-major (row-major M[s][x]); D = 128 x 64 fp32 in TMEM, lane = pattern,
// column = state.  K = 64 is eight k-steps of 8 (32 bytes); the three split products of both children are
// 48 tcgen05.mma per item, issued by one thread.  Operands sit in shared memory in the canonical 128-byte-swizzled
// K-major layout (8-row groups of 1024 B, 16-byte chunk j of row r stored at chunk j ^ (r & 7)); since K = 64 fp32 is
// 256 B per row, a tile is two such 128 x 32 blocks.
//
// Compact tips (uint8 states) take the same route: the producer writes the one-hot (missing: all-ones) rows straight
// into shared memory, so a tip costs no HBM read and its "gather" M[s][z] = hi + lo is exact on the tensor pipe
// (its lo.hi product is skipped: lo = 0).
//
// Roles (warp-specialised, one persistent CTA per SM, 17 warps):
//   warps 0-7   epilogue: warp 4h + q takes patterns 32q..32q+31 x states 32h..32h+31: tcgen05.ld (32 lanes x 32
//               columns), factors, product, row maximum, transposition through a small swizzled shared-memory stage
//               so that global stores are full 128-byte segments; pending maxima fetched one item ahead
//   warps 8-15  producers (group g = warps 8+4g .. 11+4g owns child g): ld.global (16-byte chunks, register-staged) -> hi/lo split -> st.shared in the swizzled
//               layout -> fence.proxy.async -> mbarrier arrive; HBM -> L2 streaming runs ahead of them through
//               cp.async.bulk.prefetch.L2 of the (contiguous, 32 KB) tiles two items ahead
//   warp 16     TMEM allocation; one lane issues the MMAs and the tcgen05.commit that free the shared-memory stage,
//               publish the accumulators and release the matrices
// Pipelines: shared-memory stage per child (full/empty), two TMEM accumulator sets (full/empty), matrices
// (full/empty; reloaded only when (operation, category) changes: items are dealt tile-fastest in contiguous ranges).
#pragma once
#include "plk_common.cuh"
#include "plk_gen.cuh"

namespace plk {
namespace tc5 {

constexpr int TP = 128;                    // patterns per tile = MMA M
constexpr int EPI_WARPS = 8, PROD_WARPS = 8, N_WARPS = EPI_WARPS + PROD_WARPS + 1;
constexpr int META_WARP = N_WARPS;         // warp 17: pending exponents of the next items' rows (see the kernel)
constexpr int THREADS = (N_WARPS + 1) * 32;  // 576
constexpr int PROD_THREADS = PROD_WARPS * 32;
constexpr int GROUP_THREADS = PROD_THREADS / 2;  // one producer group per child
constexpr int XCHUNKS = 16, MCHUNKS = 8;   // 16-byte chunks per producer thread: operand tile / matrix
constexpr uint32_t X_PLANE = TP * 64 * 4;  // 32 768: one plane (hi or lo) of a tile
constexpr uint32_t M_PLANE = 64 * 64 * 4;  // 16 384
constexpr uint32_t OFF_X = 0;              // [child][hi, lo]
constexpr uint32_t OFF_M = 4 * X_PLANE;    // [child][hi, lo]
constexpr uint32_t OFF_STAGE = OFF_M + 4 * M_PLANE;
constexpr uint32_t STAGE_WARP = 32 * 128;  // per epilogue warp: 32 rows x 32 columns, 16-byte chunks XOR-swizzled by row
constexpr uint32_t OFF_MAX = OFF_STAGE + EPI_WARPS * STAGE_WARP;  // [2][TP] row maxima of the upper column half
constexpr uint32_t OFF_EXP = OFF_MAX + 2 * TP * 4;              // int16 [2 children][TP]: pending exponents of the next item
constexpr uint32_t OFF_BAR = OFF_EXP + 2 * TP * 2;
constexpr uint32_t SMEM_USED = OFF_BAR + 128;
constexpr size_t SMEM_BYTES = SMEM_USED + 1024;  // + slack for the 1024-byte alignment the swizzle needs
static_assert(SMEM_BYTES <= 232448, "shared memory budget (227 KB)");
constexpr int PREFETCH_AHEAD = 2;          // items

// barrier slots (8 bytes each) at OFF_BAR
enum { B_FULL0 = 0, B_FULL1, B_EMPTY0, B_EMPTY1, B_MFULL, B_MEMPTY, B_TFULL0, B_TFULL1, B_TEMPTY0, B_TEMPTY1,
       B_EXPFULL,  // the pending exponents of the next item are in shared memory (meta warp; one buffer: no room for two)
       B_EXPFREE,  // the epilogue has read them
       B_TMEM_PTR };
static_assert((B_TMEM_PTR + 1) * 8 <= 128, "barrier slots");

// instruction descriptor: D fp32 (bit 4), A and B TF32 (2 << 7, 2 << 10), both K-major, N = 64 (>> 3 at bit 17),
// M = 128 (>> 4 at bit 24)
constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((64u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared-memory matrix descriptor: K-major, 128-byte swizzle, 8-row group stride (SBO) 1024 B, version 1 (sm_100)
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)2 << 61);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// Called by ALL lanes of the (converged) issuing warp: the instruction itself is predicated on elect.sync, so the
// descriptor arithmetic around it stays on the uniform datapath instead of a divergent branch.
// COLL: 0 = A read from shared memory and dropped, 1 = A read and kept in the collector buffer (fill),
//       2 = A taken from the collector buffer filled by the previous MMA (lastuse): the same A k-slice feeds
//       x_hi . m_lo and x_hi . m_hi, so it crosses the shared-memory port once
template <int COLL>
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t accumulate) {
  if (COLL == 1)
    asm volatile(
        "{\n\t.reg .pred p, e;\n\t"
        "elect.sync _|e, 0xffffffff;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "@e tcgen05.mma.cta_group::1.kind::tf32.collector::a::fill [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(IDESC), "r"(accumulate)
        : "memory");
  else if (COLL == 2)
    asm volatile(
        "{\n\t.reg .pred p, e;\n\t"
        "elect.sync _|e, 0xffffffff;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "@e tcgen05.mma.cta_group::1.kind::tf32.collector::a::lastuse [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(IDESC), "r"(accumulate)
        : "memory");
  else
    asm volatile(
        "{\n\t.reg .pred p, e;\n\t"
        "elect.sync _|e, 0xffffffff;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "@e tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(IDESC), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile(
      "{\n\t.reg .pred e;\n\t"
      "elect.sync _|e, 0xffffffff;\n\t"
      "@e tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(bar)
      : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,"
      "%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
        "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
        "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void l2_prefetch_bulk(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
__device__ __forceinline__ float4 ldg_nc(const float* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "l"(p));
  return v;
}
// Split x = hi + lo for the three-product TF32 scheme with two plain ALU operations instead of two conversions and a
// subtraction: hi = x with the 13 low mantissa bits cleared (a valid TF32 number whatever the tensor pipe does with low
// bits), lo = x - hi exactly (<= 2^-10 |x|, 13 significant bits of which the pipe keeps 11: residual 2^-21 |x|, against
// 2^-22 with round-to-nearest conversions -- both far inside the 1e-4 bar; the dropped lo.lo term is 2^-20).  The
// conversion unit runs at a fraction of the ALU rate and every operand element and every U value went through it twice.
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }
__device__ __forceinline__ void split4(const float4 v, float4& h, float4& l) {
  h.x = tf32_hi(v.x); l.x = v.x - h.x;
  h.y = tf32_hi(v.y); l.y = v.y - h.y;
  h.z = tf32_hi(v.z); l.z = v.z - h.z;
  h.w = tf32_hi(v.w); l.w = v.w - h.w;
}
__device__ __forceinline__ void sts128(uint32_t addr, const float4 v) {
  asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void sts32(uint32_t addr, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }
__device__ __forceinline__ float lds32(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
  return v;
}
// byte offset of 16-byte chunk `ch` (0..15) of row `row` inside a K-major 128B-swizzled plane of `rows` rows x 64 fp32
__device__ __forceinline__ uint32_t swz_off(int row, int ch, uint32_t rows) {
  return (uint32_t)(ch >> 3) * rows * 128u + (uint32_t)row * 128u + (uint32_t)(((ch & 7) ^ (row & 7)) << 4);
}

// descriptor offset (16-byte units) of k-step ks inside a swizzled plane of `rows` rows
__host__ __device__ constexpr uint64_t koff(int ks, int rows) { return (uint64_t)(((ks >> 2) * rows * 128 + (ks & 3) * 32) >> 4); }

// work items (operation, category, tile), tile fastest; each role walks its CTA's contiguous range incrementally
struct Item {
  int op, c, tile;
  uint32_t n;  // ordinal inside the CTA's range
};

struct Ctx {
  const DevOp* ops;
  int P, S, C, n_tiles;
  uint32_t n_items;
  Item first_item;
  uint32_t smem;  // 1024-aligned shared-memory base (shared-space address)
  uint32_t bar;   // address of barrier slot 0
  __device__ __forceinline__ void advance(Item& it) const {
    ++it.n;
    if (++it.tile == n_tiles) {
      it.tile = 0;
      if (++it.c == C) {
        it.c = 0;
        ++it.op;
      }
    }
  }
  __device__ __forceinline__ bool valid(const Item& it) const { return it.n < n_items; }
  // first item of the range or first tile of an (operation, category): the matrix pair changes
  __device__ __forceinline__ bool new_run(const Item& it) const { return it.n == 0 || it.tile == 0; }
  __device__ __forceinline__ uint32_t barrier(int slot) const { return bar + 8u * slot; }
};

// ---------------------------------------------------------------------------------------------------------------
// producer side.  Producer group g (4 warps) owns child g: its operand tile (2048 16-byte chunks, 16 per thread) and
// its transition matrix (1024 chunks, 8 per thread).  Thread gt of a group takes chunk gt % 16 of rows gt / 16 + 8 j,
// so the swizzled shared-memory offset of its j-th chunk is off0 + 1024 j (row & 7 does not depend on j).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void prefetch_child(const Ctx& cx, Item it, int ahead, int k) {
  for (int d = 0; d < ahead; ++d) cx.advance(it);
  if (!cx.valid(it)) return;
  const DevOp& o = cx.ops[it.op];
  const int p0 = it.tile * TP, n = cx.P - p0 < TP ? cx.P - p0 : TP;
  if (o.kind[k] == KIND_PARTIALS)
    l2_prefetch_bulk(static_cast<const float*>(o.child[k]) + ((size_t)it.c * cx.P + p0) * SP64, (uint32_t)n * 256u);
  else if (o.kind[k] == KIND_BCAST)
    l2_prefetch_bulk(static_cast<const float*>(o.child[k]) + (size_t)p0 * SP64, (uint32_t)n * 256u);
}

// global -> registers: the tile of child k of item `it` (partials), or its compact states (one per row, in r[j].x)
__device__ __forceinline__ void prod_load(const Ctx& cx, const Item& it, int k, int gt, float4 (&r)[XCHUNKS]) {
  const DevOp& o = cx.ops[it.op];
  const int kind = o.kind[k];
  const int p0 = it.tile * TP, n = cx.P - p0 < TP ? cx.P - p0 : TP;
  const int row0 = gt >> 4;
  if (gt == 0) prefetch_child(cx, it, PREFETCH_AHEAD, k);
  if (kind == KIND_PARTIALS || kind == KIND_BCAST) {
    const float* src = static_cast<const float*>(o.child[k]) + ((kind == KIND_PARTIALS ? (size_t)it.c * cx.P : 0) + p0) * SP64 + gt * 4;
#pragma unroll
    for (int j = 0; j < XCHUNKS; ++j)
      r[j] = row0 + 8 * j < n ? ldg_nc(src + j * 512) : make_float4(0.f, 0.f, 0.f, 0.f);
  } else if (kind == KIND_STATES) {
    const uint8_t* st = static_cast<const uint8_t*>(o.child[k]) + p0 + row0;
#pragma unroll
    for (int j = 0; j < XCHUNKS; ++j) r[j].x = __int_as_float(row0 + 8 * j < n ? (int)st[8 * j] : -1);
  }
}

// registers -> shared memory (hi / lo planes, swizzled K-major), then signal the MMA thread
__device__ __forceinline__ void prod_store(const Ctx& cx, const Item& it, int k, int gt, const float4 (&r)[XCHUNKS]) {
  const int kind = cx.ops[it.op].kind[k];
  const uint32_t xhi = cx.smem + OFF_X + (2 * k) * X_PLANE + swz_off(gt >> 4, gt & 15, TP), xlo = xhi + X_PLANE;
  mbar_wait(cx.barrier(B_EMPTY0 + k), (it.n & 1) ^ 1);
  if (kind == KIND_PARTIALS || kind == KIND_BCAST) {
#pragma unroll
    for (int j = 0; j < XCHUNKS; ++j) {
      float4 h, l;
      split4(r[j], h, l);
      sts128(xhi + 1024 * j, h);
      sts128(xlo + 1024 * j, l);
    }
  } else {
    const int S = cx.S, x0 = (gt & 15) * 4;
#pragma unroll
    for (int j = 0; j < XCHUNKS; ++j) {
      const int z = kind == KIND_STATES ? __float_as_int(r[j].x) : -1;  // -1: row beyond the tile or operand absent
      const bool miss = z >= S;  // missing state: every state possible (padding columns stay 0)
      float4 h;
      h.x = (z == x0 || (miss && x0 < S)) ? 1.f : 0.f;
      h.y = (z == x0 + 1 || (miss && x0 + 1 < S)) ? 1.f : 0.f;
      h.z = (z == x0 + 2 || (miss && x0 + 2 < S)) ? 1.f : 0.f;
      h.w = (z == x0 + 3 || (miss && x0 + 3 < S)) ? 1.f : 0.f;
      sts128(xhi + 1024 * j, h);
    }
  }
  fence_async_smem();
  __syncwarp();
  if ((gt & 31) == 0) mbar_arrive(cx.barrier(B_FULL0 + k));
}

__device__ __forceinline__ void prod_load_matrix(const Ctx& cx, const Item& it, int k, int gt, float4 (&m)[MCHUNKS]) {
  const float* src = static_cast<const float*>(cx.ops[it.op].mat[k]) + (size_t)it.c * SP64 * SP64 + gt * 4;
#pragma unroll
  for (int j = 0; j < MCHUNKS; ++j) m[j] = ldg_nc(src + j * 512);
}
__device__ __forceinline__ void prod_store_matrix(const Ctx& cx, int k, int gt, const float4 (&m)[MCHUNKS], uint32_t n_run) {
  const uint32_t mhi = cx.smem + OFF_M + (2 * k) * M_PLANE + swz_off(gt >> 4, gt & 15, 64), mlo = mhi + M_PLANE;
  mbar_wait(cx.barrier(B_MEMPTY), (n_run & 1) ^ 1);
#pragma unroll
  for (int j = 0; j < MCHUNKS; ++j) {
    float4 h, l;
    split4(m[j], h, l);
    sts128(mhi + 1024 * j, h);
    sts128(mlo + 1024 * j, l);
  }
  fence_async_smem();
  __syncwarp();
  if ((gt & 31) == 0) mbar_arrive(cx.barrier(B_MFULL));
}

// ---------------------------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(THREADS, 1) k_post_tc5(const DevOp* __restrict__ ops, int n_ops, int P, int S, int C) {
  extern __shared__ unsigned char tc5_smem_raw[];
  Ctx cx;
  cx.ops = ops; cx.P = P; cx.S = S; cx.C = C;
  cx.n_tiles = (P + TP - 1) / TP;
  {
    const long long total = (long long)n_ops * C * cx.n_tiles;
    const long long base = total / gridDim.x, rem = total % gridDim.x, b = blockIdx.x;
    const long long i0 = b * base + (b < rem ? b : rem);
    cx.n_items = (uint32_t)(base + (b < rem ? 1 : 0));
    const long long oc = i0 / cx.n_tiles;
    cx.first_item = Item{(int)(oc / C), (int)(oc % C), (int)(i0 % cx.n_tiles), 0u};
  }
  if (cx.n_items == 0) return;  // whole CTA leaves before any barrier or TMEM allocation
  cx.smem = (smem_u32(tc5_smem_raw) + 1023u) & ~1023u;
  cx.bar = cx.smem + OFF_BAR;

  // warp index through a shuffle: the compiler then knows it is warp-uniform and keeps the role branches (and the
  // descriptor arithmetic inside them) on the uniform datapath
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(cx.barrier(B_FULL0), PROD_WARPS / 2);
    mbar_init(cx.barrier(B_FULL1), PROD_WARPS / 2);
    mbar_init(cx.barrier(B_EMPTY0), 1);
    mbar_init(cx.barrier(B_EMPTY1), 1);
    mbar_init(cx.barrier(B_MFULL), PROD_WARPS);
    mbar_init(cx.barrier(B_MEMPTY), 1);
    mbar_init(cx.barrier(B_TFULL0), 1);
    mbar_init(cx.barrier(B_TFULL1), 1);
    mbar_init(cx.barrier(B_TEMPTY0), EPI_WARPS);
    mbar_init(cx.barrier(B_TEMPTY1), EPI_WARPS);
    mbar_init(cx.barrier(B_EXPFULL), 1);
    mbar_init(cx.barrier(B_EXPFREE), EPI_WARPS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == N_WARPS - 1) {  // 256 TMEM columns: two accumulator sets of (D_0, D_1) = 2 x 64 columns each
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(cx.barrier(B_TMEM_PTR)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(cx.barrier(B_TMEM_PTR)) : "memory");

  if (warp < EPI_WARPS) {
    // ===== epilogue: warp = 4 half + quarter takes patterns 32 quarter .. +31 (TMEM lanes) x states 32 half .. +31 =====
    const int quarter = warp & 3, half = warp >> 2;
    const uint32_t stage = cx.smem + OFF_STAGE + warp * STAGE_WARP;
    // Pending exponents of both children (deferred rescaling) come from the meta warp through shared memory.  (The
    // epilogue warps used to load the per-category maxima themselves, one item ahead: scattered DRAM loads whose
    // scoreboard every later wait of the warp inherited -- see plk_tc5_pre2.cuh, where a cycle trace showed it.)
    const short* sexp = reinterpret_cast<const short*>(tc5_smem_raw + (cx.smem - smem_u32(tc5_smem_raw)) + OFF_EXP);
    for (Item it = cx.first_item; cx.valid(it);) {
      const uint32_t n = it.n;
      const DevOp& o = ops[it.op];
      const int p0 = it.tile * TP, prow0 = p0 + 32 * quarter, p = prow0 + lane;
      mbar_wait(cx.barrier(B_EXPFULL), n & 1);  // written while the previous item was processed
      const Pow2Pair<float> f0 = pow2_pair(-(int)sexp[32 * quarter + lane], 0.f);
      const Pow2Pair<float> f1 = pow2_pair(-(int)sexp[TP + 32 * quarter + lane], 0.f);
      __syncwarp();
      if (lane == 0) mbar_arrive(cx.barrier(B_EXPFREE));
      const bool one_factor = __all_sync(0xffffffffu, f0.f2 == 1.f && f1.f2 == 1.f);
      float* dest = static_cast<float*>(o.dest) + (size_t)it.c * P * SP64;
      float* scale = static_cast<float*>(o.scale);
      Item nx = it;
      cx.advance(nx);
      const uint32_t a = n & 1;
      mbar_wait(cx.barrier(B_TFULL0 + a), (n >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(32 * quarter) << 16) + a * 128 + half * 32;
      float mx = 0.f;
      {
        uint32_t d0[32], d1[32];
        tmem_ld32(taddr, d0);
        tmem_ld32(taddr + 64, d1);
        tmem_ld_wait();
        // accumulators are in registers: hand the TMEM set back before the stores
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(cx.barrier(B_TEMPTY0 + a));
        if (one_factor) {  // the usual case: each pending exponent fits one power-of-two factor
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            float v[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              v[j] = (__uint_as_float(d0[4 * q + j]) * f0.f1) * (__uint_as_float(d1[4 * q + j]) * f1.f1);
              mx = fmaxf(mx, v[j]);
            }
            sts128(stage + lane * 128 + ((q ^ (lane & 7)) << 4), make_float4(v[0], v[1], v[2], v[3]));
          }
        } else {
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            float v[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              v[j] = ((__uint_as_float(d0[4 * q + j]) * f0.f1) * f0.f2) * ((__uint_as_float(d1[4 * q + j]) * f1.f1) * f1.f2);
              mx = fmaxf(mx, v[j]);
            }
            sts128(stage + lane * 128 + ((q ^ (lane & 7)) << 4), make_float4(v[0], v[1], v[2], v[3]));
          }
        }
      }
      // the upper column half's row maximum travels through shared memory (double-buffered by item parity)
      if (half == 1) sts32(cx.smem + OFF_MAX + (a * TP + 32 * quarter + lane) * 4, mx);
      __syncwarp();
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int idx = j * 32 + lane, r = idx >> 3, ch = idx & 7;
        const float4 v = lds128(stage + r * 128 + ((ch ^ (r & 7)) << 4));
        if (prow0 + r < P) *reinterpret_cast<float4*>(dest + (size_t)(prow0 + r) * SP64 + half * 32 + ch * 4) = v;
      }
      asm volatile("bar.sync 1, %0;" ::"n"(EPI_WARPS * 32) : "memory");
      if (half == 0 && p < P && scale != nullptr)
        scale[(size_t)it.c * P + p] = fmaxf(mx, lds32(cx.smem + OFF_MAX + (a * TP + 32 * quarter + lane) * 4));
      it = nx;
    }
  } else if (warp < EPI_WARPS + PROD_WARPS) {
    // ===== producers: group g = child g =====
    const int pt = threadIdx.x - EPI_WARPS * 32, g = pt >> 7, gt = pt & 127;
    if (gt == 0)
      for (int d = 0; d < PREFETCH_AHEAD; ++d) prefetch_child(cx, cx.first_item, d, g);
    float4 r[XCHUNKS];
    uint32_t n_run = 0;
    Item it = cx.first_item;
    bool loaded = false;
#pragma unroll 1
    while (true) {
      if (cx.new_run(it)) {  // the register pipeline is drained here: r stages the matrix
        static_assert(MCHUNKS <= XCHUNKS, "r doubles as the matrix staging registers");
        float4(&m)[MCHUNKS] = reinterpret_cast<float4(&)[MCHUNKS]>(r);
        prod_load_matrix(cx, it, g, gt, m);
        prod_store_matrix(cx, g, gt, m, n_run);
        ++n_run;
      }
      if (!loaded) prod_load(cx, it, g, gt, r);
      prod_store(cx, it, g, gt, r);
      Item nx = it;
      cx.advance(nx);
      if (!cx.valid(nx)) break;
      loaded = !cx.new_run(nx);
      if (loaded) prod_load(cx, nx, g, gt, r);
      it = nx;
    }
  } else if (warp == META_WARP) {
    // ===== meta warp: exponent of max_c cscale[k][c][p] for the 128 rows of every item, one item ahead (its loads are
    // in flight while it waits for the epilogue to have read the previous item's values) =====
    short* sexp = reinterpret_cast<short*>(tc5_smem_raw + (cx.smem - smem_u32(tc5_smem_raw)) + OFF_EXP);
    auto ldv = [](const float* m) {
      float v;
      asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(m));
      return v;
    };
    for (Item it = cx.first_item; cx.valid(it); cx.advance(it)) {
      const uint32_t n = it.n;
      const DevOp& o = ops[it.op];
      const float* src[2] = {static_cast<const float*>(o.cscale[0]), static_cast<const float*>(o.cscale[1])};
      float4 raw[4][2];  // all loads of the item are issued before the first one is used
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int p = it.tile * TP + lane + 32 * j;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
          if (src[k] != nullptr && p < P) {
            const float* m = src[k] + p;
            v.x = ldv(m);
            if (C > 1) v.y = ldv(m + (size_t)P);
            if (C > 2) v.z = ldv(m + 2 * (size_t)P);
            if (C > 3) v.w = ldv(m + 3 * (size_t)P);
          }
          raw[j][k] = v;
        }
      }
      int ex[4][2];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int p = it.tile * TP + lane + 32 * j;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          float v = fmaxf(fmaxf(raw[j][k].x, raw[j][k].y), fmaxf(raw[j][k].z, raw[j][k].w));
          if (C > 4 && src[k] != nullptr && p < P)
            for (int c = 4; c < C; ++c) v = fmaxf(v, src[k][(size_t)c * P + p]);
          ex[j][k] = exp_of(v);
        }
      }
      if (n > 0) mbar_wait(cx.barrier(B_EXPFREE), (n + 1) & 1);  // item n - 1 was read
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int k = 0; k < 2; ++k) sexp[k * TP + lane + 32 * j] = (short)ex[j][k];
      __syncwarp();
      if (lane == 0) mbar_arrive(cx.barrier(B_EXPFULL));
    }
  } else {
    // ===== MMA issuer: the whole warp runs the loop, one elected lane executes each tcgen05.mma / commit =====
    uint32_t n_run = 0;
    const uint64_t dX[2] = {make_desc(cx.smem + OFF_X), make_desc(cx.smem + OFF_X + 2 * X_PLANE)};
    const uint64_t dM[2] = {make_desc(cx.smem + OFF_M), make_desc(cx.smem + OFF_M + 2 * M_PLANE)};
    for (Item it = cx.first_item; cx.valid(it); cx.advance(it)) {
      const uint32_t n = it.n;
      const DevOp& o = ops[it.op];
      if (cx.new_run(it)) {
        mbar_wait(cx.barrier(B_MFULL), n_run & 1);
        ++n_run;
      }
      const uint32_t a = n & 1;
      mbar_wait(cx.barrier(B_TEMPTY0 + a), ((n >> 1) & 1) ^ 1);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        mbar_wait(cx.barrier(B_FULL0 + k), n & 1);
        tc_fence_after();
        const uint32_t d = tmem_base + a * 128 + k * 64;
        // descriptors differ from the plane's base descriptor only in the 16-byte-unit address field
        const uint64_t dxhi = dX[k], dxlo = dX[k] + (X_PLANE >> 4), dmhi = dM[k], dmlo = dM[k] + (M_PLANE >> 4);
        const bool has_lo = o.kind[k] == KIND_PARTIALS || o.kind[k] == KIND_BCAST;
        uint32_t acc = 0;
        if (has_lo) {  // x_lo . m_hi
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            umma_tf32<0>(d, dxlo + koff(ks, TP), dmhi + koff(ks, 64), acc);
            acc = 1;
          }
        }
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {  // x_hi . m_lo + x_hi . m_hi, the A slice fetched once
          umma_tf32<1>(d, dxhi + koff(ks, TP), dmlo + koff(ks, 64), acc);
          umma_tf32<2>(d, dxhi + koff(ks, TP), dmhi + koff(ks, 64), 1);
          acc = 1;
        }
        umma_commit(cx.barrier(B_EMPTY0 + k));
      }
      umma_commit(cx.barrier(B_TFULL0 + a));
      Item nx = it;
      cx.advance(nx);
      if (cx.valid(nx) && cx.new_run(nx)) umma_commit(cx.barrier(B_MEMPTY));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == N_WARPS - 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem_base) : "memory");
  }
}

inline int launch_post(cudaStream_t stream, const DevOp* d_ops, int n_ops, int P, int S, int C, int sm_count,
                       int64_t* launches) {
  // per device and cheap: no process-wide "done" flag (instances may live on several GPUs)
  if (cudaFuncSetAttribute(k_post_tc5, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess)
    return PLK_ERR_CUDA;
  const long long total = (long long)n_ops * C * ((P + TP - 1) / TP);
  if (total <= 0) return PLK_SUCCESS;
  const int grid = total < sm_count ? (int)total : sm_count;
  k_post_tc5<<<grid, THREADS, SMEM_BYTES, stream>>>(d_ops, n_ops, P, S, C);
  if (cudaGetLastError() != cudaSuccess) return PLK_ERR_CUDA;
  ++*launches;
  return PLK_SUCCESS;
}

}  // namespace tc5
}  // namespace plk
