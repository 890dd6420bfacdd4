/* plk.h -- C ABI of the B200-native phylogenetic-likelihood hot path (libplk.so).
 *
 * What this library computes (citations: P:<line> = PAPER.md line; S8x = SURVEY.md section 8(x)):
 *   - transition matrices from a client-supplied eigendecomposition, cached for reuse over patterns;
 *   - Felsenstein-pruning post-order partial likelihoods over patterns x rate categories x states with
 *     per-pattern rescaling (S8a steps 2-3), level-batched from an operation list;
 *   - the root log-likelihood reduction (S8a step 4);
 *   - the pre-order partials and the linear-time gradient of the log-likelihood with respect to every
 *     branch length as the `pre . Q . post` sandwich (S8a steps 5-6);
 *   - tip-state encoding and unique-site-pattern compression ("unique site patterns"; S8a step 0).
 *
 * Conventions that hold for EVERY entry point
 *   Return value   0 (PLK_SUCCESS) or a negative plk_status; nothing throws across this boundary; no global state.
 *   Host pointers  belong to the caller and are only read / written during the call.  Host-side numbers are
 *                  always `double` whatever the instance precision (conversion happens on upload / download).
 *   Device memory  ONE arena, allocated by the caller (e.g. a torch uint8 tensor) and handed to plk_create; the
 *                  library never calls cudaMalloc / cudaFree.  Arguments named `d_*` are DEVICE pointers owned by
 *                  the caller.  A few KB of pinned host staging are allocated by plk_create with cudaHostAlloc.
 *   Stream         all device work is enqueued on the CUDA stream given to plk_create (a cudaStream_t passed as
 *                  void*; NULL = legacy default stream).  Calls that return values into HOST memory synchronise
 *                  that stream before returning; calls with only device outputs (`*_device`) never synchronise.
 *   Layout         every exposed array is row-major with the state index fastest, then pattern, then category:
 *                  partials[c][p][s]; matrices M[c][s_parent][s_child].  Internally states are padded
 *                  (20 -> 32, 61 -> 64) with zeros; padding never appears at this boundary.
 *   Indices        partials buffers 0..partials_buffer_count-1 (tips are 0..tip_count-1); pre-order buffers
 *                  0..preorder_buffer_count-1; matrix / scale / eigen buffers likewise.  Any index out of range
 *                  -> PLK_ERR_OUT_OF_RANGE; a buffer read before it was written -> PLK_ERR_UNINITIALIZED.
 *   Threads        one instance must not be used from two host threads at once; distinct instances may.
 *   No fallback    there is no CPU path: without a CUDA device plk_create returns PLK_ERR_CUDA.
 */
#ifndef PLK_H_
#define PLK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PLK_API __attribute__((visibility("default")))

typedef enum {
  PLK_SUCCESS = 0,
  PLK_ERR_GENERAL = -1,
  PLK_ERR_OUT_OF_MEMORY = -2,  /* arena too small / no free buffer slot                              */
  PLK_ERR_OUT_OF_RANGE = -3,   /* an index, a count, a shape or a branch length (t < 0, NaN) is invalid */
  PLK_ERR_UNINITIALIZED = -4,  /* a buffer / matrix / model component is read before it was written    */
  PLK_ERR_UNSUPPORTED = -5,    /* state count not in 2..64, unknown flag, path not built                */
  PLK_ERR_FLOATING_POINT = -6, /* NaN / Inf / -Inf in the log-likelihood or a derivative                */
  PLK_ERR_CUDA = -7,           /* a CUDA runtime call failed (no device, launch failure, ...)           */
  PLK_ERR_STOP_CODON = -8,     /* plk_encode_and_compress met a stop codon                              */
  PLK_ERR_STATIC_SCRATCH_LIMIT = -9 /* plk_root_log_likelihoods_static_device: the problem needs more than the
                                  library's fixed static scratch (PLK_STATIC_SCRATCH_DOUBLES / PLK_STATIC_SCALE_MAX) */
} plk_status;

/* limits of plk_root_log_likelihoods_static_device (the one entry point whose scratch is a static device array) */
#define PLK_STATIC_SCRATCH_DOUBLES 8192 /* 64 KB per GPU: k_root blocks = ceil(P * G / 128), G = 1 | 8 | 16 for
                                           4 | 5..32 | 33..64 states => P <= 1 048 576 | 131 072 | 65 536 */
#define PLK_STATIC_SCALE_MAX 2048       /* scale buffers per call */

enum { PLK_FP64 = 0, PLK_FP32 = 1 };                 /* plk_config.precision                          */
enum {                                                /* plk_config.flags (bit set)                    */
  PLK_FLAG_TENSOR_CORES = 1,   /* codon-size (padded 64-state) kernels use the tensor pipe: fp64 -> DMMA,
                                  fp32 -> split-TF32 tcgen05; without it they run on the CUDA cores     */
  PLK_FLAG_NO_LEVEL_BATCH = 2, /* launch one kernel per operation instead of one per dependency level
                                  (reference behaviour for tests; slower)                               */
  PLK_FLAG_LEVEL_BATCH_ONLY = 8,  /* 4-state kernels: always one launch per dependency level                */
  PLK_FLAG_PATTERN_WALK_ONLY = 16, /* 4-state kernels: always ONE launch per call in which every warp keeps its
                                  patterns and walks the whole operation list in the order given (patterns are
                                  independent, so list order is the only dependency).  Without either flag the
                                  library picks the cheaper shape from P, C, the list length and its level count */
  PLK_FLAG_NO_TMA = 32,        /* 4-state kernels: use the register-staged (LDG) kernels instead of the TMA-staged
                                  ones (comparison arm; also what category counts other than 1, 2, 4, 8 run on) */
  PLK_FLAG_NO_TCGEN05 = 64,    /* fp32 + PLK_FLAG_TENSOR_CORES: run the post-order and the fused pre-order + derivative
                                  kernels on the legacy warp-level mma.sync TF32 kernels instead of the tcgen05 /
                                  TMEM kernels (comparison arm)                                             */
  PLK_FLAG_NO_PDL = 128,       /* 4-state gradient pass: plain stream-ordered launches instead of programmatic
                                  dependent launches (the item classes of one dependency level are independent of
                                  each other and otherwise overlap one another's tail; comparison arm)       */
  PLK_FLAG_CACHE_RATE_PRODUCTS = 256, /* P:101 caching variant: reserve a second slot per full partials slot for
                                  Q p_k.  plk_update_partials then also stores Q p_dest of every operation (Q of eigen
                                  buffer 0; plk_cache_rate_products for any other buffer / eigen), and
                                  plk_branch_derivatives evaluates the sandwich from the cached products            */
  PLK_FLAG_ON_THE_FLY_MATRICES = 512, /* P:101 caching variant: reserve the ready flags of
                                  plk_update_partials_on_the_fly (partials_buffer_count * P words); padded state counts
                                  only (S > 4)                                                                      */
  PLK_FLAG_SITE_DERIVATIVES = 4 /* reserve partials_buffer_count * P doubles so that the gradient calls can
                                  return per-pattern derivatives (out_site != NULL); without it such a
                                  request returns PLK_ERR_UNSUPPORTED                                   */
};
enum { PLK_NUCLEOTIDE = 0, PLK_CODON = 1 };          /* plk_encode_and_compress state_kind            */

typedef struct plk_instance plk_instance;            /* opaque */

/* All sizes are fixed at creation (S8b). */
typedef struct {
  int32_t tip_count;              /* N >= 2                                                              */
  int32_t state_count;            /* S: 4 (nucleotide, bandwidth kernels), 5..32 (padded to 32; 20 = amino acids,
                                     CUDA cores) or 33..64 (padded to 64; 61 = codon)                       */
  int32_t pattern_count;          /* P >= 1                                                              */
  int32_t category_count;         /* C >= 1 (<= 16)                                                      */
  int32_t partials_buffer_count;  /* size of the post-order index space (tips first), usually 2N-1       */
  int32_t compact_buffer_count;   /* how many tips will be given as compact states (P bytes each)        */
  int32_t partials_slot_count;    /* full-size slots backing the index space; 0 => partials_buffer_count
                                     - compact_buffer_count.  A slot is bound to an index at first write  */
  int32_t preorder_buffer_count;  /* size of the pre-order index space; 0 => gradient calls unsupported   */
  int32_t preorder_slot_count;    /* full-size slots backing it; 0 => preorder_buffer_count               */
  int32_t matrix_buffer_count;    /* each holds C matrices of S x S                                      */
  int32_t eigen_buffer_count;     /* each holds U, U^-1, lambda and the rate matrix Q                    */
  int32_t scale_buffer_count;     /* each holds P per-pattern scale exponents                            */
  int32_t precision;              /* PLK_FP64 | PLK_FP32: storage + arithmetic of partials and matrices;
                                     log factors, site sums and pattern sums are fp64 in both            */
  int32_t flags;
} plk_config;

/* One post-order operation (S8a step 2): dest = (M1 . child1) o (M2 . child2), per pattern and category, followed
 * by per-pattern rescaling into scale buffer `dest_scale` (S8a step 3) unless dest_scale < 0. */
typedef struct {
  int32_t dest;          /* partials buffer written                      */
  int32_t dest_scale;    /* scale buffer written, or -1 = do not rescale */
  int32_t child1;        /* partials buffer (tip states, tip partials or internal partials) */
  int32_t child1_matrix; /* matrix buffer of the branch above child1     */
  int32_t child2;
  int32_t child2_matrix;
} plk_op;

/* One pre-order operation (S8a step 5), for the child `k` of parent `m` with sibling `j`:
 * q_k[c,p,s] = sum_x M_k[c][x,s] ( q_m[c,p,x] * sum_y M_j[c][x,y] p_j[c,p,y] ), rescaled per pattern. */
typedef struct {
  int32_t dest_pre;       /* pre-order buffer written (q_k); in plk_pre_order_gradient -1 = do not store      */
  int32_t parent_pre;     /* pre-order buffer of the parent (q_m)                                            */
  int32_t matrix;         /* matrix buffer of the branch above k (applied transposed)                        */
  int32_t sibling_post;   /* post-order buffer of the sibling (p_j)                                          */
  int32_t sibling_matrix; /* matrix buffer of the branch above the sibling                                   */
  int32_t node_post;      /* post-order buffer of k itself (p_k): used by plk_pre_order_gradient only        */
} plk_pre_op;

/* ---- instance ------------------------------------------------------------------------------------------- */

/* Bytes of device memory an instance with this configuration needs (0 if the configuration is invalid). */
PLK_API size_t plk_arena_bytes(const plk_config* cfg);

/* Create an instance inside the caller's device arena (>= plk_arena_bytes(cfg), 1024-byte aligned).
 * Errors: _OUT_OF_RANGE (bad sizes), _UNSUPPORTED (state count, flags), _OUT_OF_MEMORY (arena too small),
 * _CUDA (no device).  On error *out is NULL. */
PLK_API int plk_create(const plk_config* cfg, void* d_arena, size_t arena_bytes, void* cuda_stream,
                       plk_instance** out);

/* Release host-side state.  Never frees or touches the arena.  NULL is allowed. */
PLK_API int plk_destroy(plk_instance* inst);

PLK_API const char* plk_error_string(int status);

/* ---- data and model setters (host -> device; S8a "set-up", not hot) --------------------------------------- */

/* Tip `tip` as compact state codes, P values in 0..S; the value S (or larger) means missing / fully ambiguous and
 * contributes 1 for every state (S8c row 15).  Uses one compact slot. */
PLK_API int plk_set_tip_states(plk_instance* inst, int tip, const int32_t* states);

/* The same with one BYTE per pattern (values >= S: missing), which is the layout the kernels read: a plain
 * host -> device copy, enqueued on the instance's stream WITHOUT synchronising.  `states` (P bytes, host memory) is
 * therefore the one exception to the ownership rule above: when it is pinned memory it must stay unchanged until the
 * next call that returns values to the host (or plk_synchronize).  This is the upload an application repeats per
 * evaluation when its alignment changes (bench.py's end-to-end leg). */
PLK_API int plk_set_tip_states_u8(plk_instance* inst, int tip, const uint8_t* states);

/* Tips 0 .. count-1 at once: `states` is HOST memory [count][P] bytes (row t = tip t, values >= S: missing).  Tips
 * that sit in consecutive compact slots -- all of them when they were first set in index order -- travel as ONE pitched
 * asynchronous copy instead of `count` copies (configs[1]: 128 x 100 KB).  Same ownership exception and no
 * synchronisation as plk_set_tip_states_u8.  _OUT_OF_RANGE if one of the tips was set as partials before. */
PLK_API int plk_set_all_tip_states_u8(plk_instance* inst, const uint8_t* states, int count);

/* Tip `tip` as partials [P][S], the same for every category (e.g. one-hot rows, all-ones rows for missing). */
PLK_API int plk_set_tip_partials(plk_instance* inst, int tip, const double* partials);

/* Any post-order buffer as full partials [C][P][S]. */
PLK_API int plk_set_partials(plk_instance* inst, int buffer, const double* partials);

PLK_API int plk_set_pattern_weights(plk_instance* inst, const double* weights /* [P] */);
PLK_API int plk_set_state_frequencies(plk_instance* inst, const double* pi /* [S] */);
PLK_API int plk_set_category_rates(plk_instance* inst, const double* rates /* [C] */);
PLK_API int plk_set_category_weights(plk_instance* inst, const double* weights /* [C] */);

/* Q = U diag(lambda) U^-1 ("numerical eigendecomposition of the infinitesimal rate matrix" is done by the
 * client).  U, Uinv: [S][S] row-major; lambda: [S].  Also rebuilds the rate matrix Q of this eigen buffer as
 * U diag(lambda) Uinv unless plk_set_rate_matrix is called afterwards. */
PLK_API int plk_set_eigen_decomposition(plk_instance* inst, int eigen, const double* U, const double* Uinv,
                                        const double* lambda);

/* The rate matrix Q [S][S] used by the gradient sandwich, overriding the rebuilt one. */
PLK_API int plk_set_rate_matrix(plk_instance* inst, int eigen, const double* Q);

/* Matrix buffer `matrix` directly: [C][S][S], M[c][parent state][child state]. */
PLK_API int plk_set_transition_matrix(plk_instance* inst, int matrix, const double* m);

/* ---- hot path ---------------------------------------------------------------------------------------------- */

/* S8a step 1 / P:101.  For i in 0..count-1 and every category c:
 *   matrix[matrix_idx[i]][c] = U diag(exp(lambda r_c t_i)) U^-1   (fp64 arithmetic, stored in instance precision).
 * branch_lengths: HOST [count], each finite and >= 0 else _OUT_OF_RANGE.  Needs category rates and `eigen`. */
PLK_API int plk_update_transition_matrices(plk_instance* inst, int eigen, const int32_t* matrix_idx,
                                           const double* branch_lengths, int count);
/* Same with the branch lengths already in device memory (fp64 [count]); not range-checked, never synchronises. */
PLK_API int plk_update_transition_matrices_device(plk_instance* inst, int eigen, const int32_t* matrix_idx,
                                                  const double* d_branch_lengths, int count);

/* S8a steps 2-3 / P:27.  `ops` (HOST, count >= 0) may come in any order in which every child is either written
 * before this call or is the dest of an EARLIER op of the list.  The library groups the ops into dependency
 * levels and launches one kernel per level (S8a "level-batched").  Two ops of one call must not share a dest or
 * a dest_scale (_OUT_OF_RANGE).  Never synchronises. */
PLK_API int plk_update_partials(plk_instance* inst, const plk_op* ops, int count);

/* S8f-3 / P:101 ("for phylogeographic problems that typically have a large state-space size but only a single site
 * pattern ... it is more efficient to form the transition probability matrix on-the-fly while calculating the likelihood
 * ... through Felsenstein's pruning algorithm").  The same update as plk_update_partials -- same buffers, same deferred
 * rescaling, results interchangeable -- but no transition matrix is read, formed or stored: for the branch above child k
 * of ops[i], of length branch_lengths[2 i + k] (HOST, finite and >= 0), exp(Q r_c t) is applied to the child's partial as
 * U (exp(lambda r_c t) o (U^-1 x)) from eigen buffer `eigen` (4 S^2 flops per edge, pattern and category; fp64 arithmetic
 * in both precisions).  The child*_matrix fields of the operations are ignored.  The WHOLE list runs in ONE launch
 * (dataflow over ready flags; independent subtrees run concurrently), in the order given.  Needs
 * PLK_FLAG_ON_THE_FLY_MATRICES (else _UNSUPPORTED) and count <= partials_buffer_count.  Never synchronises. */
PLK_API int plk_update_partials_on_the_fly(plk_instance* inst, int eigen, const plk_op* ops, int count,
                                           const double* branch_lengths);

/* S8f-3 / P:101 ("the product of the infinitesimal rate matrix and the post-order partial likelihood vector at each node
 * could be cached directly").  Stores Qp_k[c,p,.] = Q p_k[c,p,.] (Q of eigen buffer `eigen`) for the listed post-order
 * buffers; compact tips need none.  Needs PLK_FLAG_CACHE_RATE_PRODUCTS (else _UNSUPPORTED).  With that flag
 * plk_update_partials calls it for the dests of its operations (eigen buffer 0) and plk_branch_derivatives reads
 * num_p = sum_c w_c r_c q . Qp instead of applying Q; a listed buffer whose product was never cached, or whose partials
 * were overwritten since, gives _UNINITIALIZED there.  Never synchronises. */
PLK_API int plk_cache_rate_products(plk_instance* inst, int eigen, const int32_t* post_idx, int count);

/* S8a step 4.  log l_p = log( sum_c w_c sum_s pi_s p_root[c,p,s] ) + sum over the listed scale buffers of their
 * log factor; logL = sum_p omega_p log l_p.  out_sum: HOST [1]; out_site: HOST [P] or NULL.
 * Returns _FLOATING_POINT (outputs still written) if logL is NaN or infinite. */
PLK_API int plk_root_log_likelihoods(plk_instance* inst, int root_buffer, const int32_t* scale_idx,
                                     int scale_count, double* out_sum, double* out_site);
/* Same, results left in device memory: d_out_sum fp64 [1], d_out_site fp64 [P] or NULL.  No error check on the
 * value, no synchronisation. */
PLK_API int plk_root_log_likelihoods_device(plk_instance* inst, int root_buffer, const int32_t* scale_idx,
                                            int scale_count, double* d_out_sum, double* d_out_site);

/* S8a step 4 for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, kernels and results as plk_root_log_likelihoods_device, but the per-block partial
 * sums of the reduction live in a file-scope `static __device__` array of the library (PLK_STATIC_SCRATCH_DOUBLES
 * doubles = 64 KB, held by every GPU that loads libplk.so until the process exits) instead of the instance arena, and
 * the call performs no device or host allocation at all.  A problem beyond the limits above returns
 * PLK_ERR_STATIC_SCRATCH_LIMIT and launches nothing.  The array is shared by all instances and streams of a device and
 * keeps the last call's contents (every entry that is read is written first by the same call, so nothing needs
 * clearing); calls that overlap on the GPU race on it -- serialise them (one stream, or events).  The arena's device
 * must be current.  Never synchronises, no value check. */
PLK_API int plk_root_log_likelihoods_static_device(plk_instance* inst, int root_buffer, const int32_t* scale_idx,
                                                   int scale_count, double* d_out_sum, double* d_out_site);

/* S8a step 5 / P:43.  Fills pre-order buffer `root_pre_buffer` with q_root[c,p,.] = pi, then applies `ops`
 * (root towards tips; same ordering rule as plk_update_partials with parent_pre in the role of the children).
 * Every q_k is rescaled per pattern by a power of two that is discarded (it cancels in step 6). */
PLK_API int plk_update_pre_partials(plk_instance* inst, int root_pre_buffer, const plk_pre_op* ops, int count);

/* S8a step 6 / P:43.  For i in 0..count-1, with p = post-order buffer post_idx[i] and q = pre-order buffer
 * pre_idx[i] of the same node:  num_p = sum_c w_c r_c q[c,p]^T Q p[c,p],  den_p = sum_c w_c q[c,p]^T p[c,p],
 * out_gradient[i] = sum_p omega_p num_p / den_p  (HOST [count]); out_site (HOST [count][P] or NULL) receives
 * num_p / den_p.  Q is the rate matrix of eigen buffer `eigen`.  _FLOATING_POINT if any gradient is not finite. */
PLK_API int plk_branch_derivatives(plk_instance* inst, int eigen, const int32_t* post_idx, const int32_t* pre_idx,
                                   int count, double* out_gradient, double* out_site);

/* Steps 5 and 6 fused (the benchmarked path): the two sibling ops of one parent are executed by one kernel that
 * reads q_parent and both children's post-order partials once, writes q of those children whose dest_pre >= 0
 * (tips need not be stored) and accumulates both branch derivatives.  out_gradient: HOST [count], in the order of
 * `ops` (the derivative of the branch above ops[i]'s node); out_site: HOST [count][P] or NULL. */
PLK_API int plk_pre_order_gradient(plk_instance* inst, int eigen, int root_pre_buffer, const plk_pre_op* ops,
                                   int count, double* out_gradient, double* out_site);
/* Same with device outputs (fp64), no synchronisation, no value check. */
PLK_API int plk_pre_order_gradient_device(plk_instance* inst, int eigen, int root_pre_buffer,
                                          const plk_pre_op* ops, int count, double* d_out_gradient,
                                          double* d_out_site);

/* S8a steps 1-6 in ONE call (the unit of work of an HMC step): transition matrices for the `matrix_count` listed
 * branches, post-order partials for `ops`, the root log-likelihood over `scale_idx`, and the fused pre-order + derivative
 * pass for `pre_ops` -- exactly plk_update_transition_matrices_device + plk_update_partials +
 * plk_root_log_likelihoods_device + plk_pre_order_gradient_device with the same arguments, same kernels, same results.
 * d_out: DEVICE fp64 [1 + pre_count] = [logL, derivative of the branch above pre_ops[0]'s node, ...].  Small problems
 * are bound by launch latency, so the library caches the whole launch sequence of a call signature (all index arrays,
 * the two device pointers, the model and the slot bindings) as a CUDA graph: the first use of a signature runs eagerly,
 * the second is captured, every later one is a single graph launch.  Capture needs a non-default stream (a stream
 * created by the caller, e.g. torch.cuda.Stream); on the legacy default stream every use runs eagerly.  At most 8
 * signatures are cached per instance (then all are dropped).  Never synchronises, no value check. */
PLK_API int plk_evaluate_device(plk_instance* inst, int eigen, const int32_t* matrix_idx, const double* d_branch_lengths,
                                int matrix_count, const plk_op* ops, int op_count, int root_buffer,
                                const int32_t* scale_idx, int scale_count, int root_pre_buffer, const plk_pre_op* pre_ops,
                                int pre_count, double* d_out);
/* The same with HOST branch lengths [matrix_count] (each finite and >= 0 else _OUT_OF_RANGE) and HOST results:
 * out_logl [1], out_gradient [pre_count].  One upload, one graph launch, one download, one synchronisation.
 * _FLOATING_POINT (outputs still written) if a value is not finite. */
PLK_API int plk_evaluate(plk_instance* inst, int eigen, const int32_t* matrix_idx, const double* branch_lengths,
                         int matrix_count, const plk_op* ops, int op_count, int root_buffer, const int32_t* scale_idx,
                         int scale_count, int root_pre_buffer, const plk_pre_op* pre_ops, int pre_count, double* out_logl,
                         double* out_gradient);

/* S8f-1 / P:29.  Approximate gradient of logL with respect to every element of the rate matrix: the gradient
 * "w.r.t. elements of the rate matrix" evaluated with "a first-order approximation of the derivative of the matrix
 * exponential", d exp(Q tau) / d Q_ij ~= tau exp(Q tau) E_ij, which reduces the sandwich of branch b to an outer product
 * of the pre- and post-order partials of node b (reading 14).  For i in 0..count-1 with
 * p = post-order buffer post_idx[i], q = pre-order buffer pre_idx[i] of the same node and t = branch_lengths[i]:
 *   out_G[a][b] = sum_i t_i sum_p omega_p ( sum_c w_c r_c q[c,p,a] p[c,p,b] ) / ( sum_c w_c q[c,p]^T p[c,p] )
 * out_G: HOST [S][S] row-major (diagonal included).  branch_lengths: HOST [count], finite and >= 0.  Needs the
 * pre-order partials of every listed node (plk_update_pre_partials, or plk_pre_order_gradient with dest_pre >= 0).
 * Exact in every direction dQ that commutes with Q (an overall rate).  _FLOATING_POINT if an element is not finite.
 * With PLK_FLAG_TENSOR_CORES and 33..64 states the pattern contraction runs on the tensor cores (fp64: DMMA, fp32:
 * split TF32; pattern sums in fp64 in a fixed order in every case: bitwise repeatable). */
PLK_API int plk_rate_matrix_gradient(plk_instance* inst, const int32_t* post_idx, const int32_t* pre_idx,
                                     const double* branch_lengths, int count, double* out_G);

/* ---- read-back (tests) -------------------------------------------------------------------------------------- */

/* Partials [C][P][S] of a post-order (pre = 0) or pre-order (pre = 1) buffer; compact tips are expanded to
 * one-hot / all-ones rows.  pre = 2: the cached rate product Q p_k of post-order buffer `buffer`
 * (PLK_FLAG_CACHE_RATE_PRODUCTS; _UNINITIALIZED if it is not current, _UNSUPPORTED for a compact tip). */
PLK_API int plk_get_partials(plk_instance* inst, int buffer, int pre, double* out);
/* Natural-log scale factors [P] of one scale buffer (the stored power-of-two exponent times ln 2). */
PLK_API int plk_get_scale_factors(plk_instance* inst, int scale, double* out);
PLK_API int plk_get_transition_matrix(plk_instance* inst, int matrix, double* out /* [C][S][S] */);
PLK_API int plk_get_rate_matrix(plk_instance* inst, int eigen, double* out /* [S][S] */);

/* Blocks until everything enqueued by this instance has finished (cudaStreamSynchronize). */
PLK_API int plk_synchronize(plk_instance* inst);

/* Number of kernels this instance has launched since creation (bench.py's gpu_launches). */
PLK_API int64_t plk_kernel_launch_count(const plk_instance* inst);

/* ---- host-side helpers (no device needed) -------------------------------------------------------------------- */

/* Dependency levels of a post-order op list as plk_update_partials forms them: out_level[i] = 0 if neither child
 * of ops[i] is the dest of an earlier op, else 1 + max level of the ops producing its children.  Returns the
 * number of levels (>= 0) or a negative status (_OUT_OF_RANGE: duplicate dest, negative index). */
PLK_API int plk_schedule_levels(const plk_op* ops, int count, int32_t* out_level);
/* Same for pre-order ops (dependency: parent_pre written by an earlier op); additionally out_partner[i] = index
 * of the other op with the same parent_pre in the same call (the two are fused into one launch item), or -1. */
PLK_API int plk_schedule_pre_levels(const plk_pre_op* ops, int count, int32_t* out_level, int32_t* out_partner);

/* S8f-1 / P:45 chain rule ("the product of the gradient w.r.t. elements of the rate matrix and the gradient of the matrix
 * elements w.r.t. substitution model parameters", O(K S^2)): out[k] = sum_ab G[a][b] dQ[k][a][b].  G: [S][S] from
 * plk_rate_matrix_gradient; dQ: [K][S][S] = d Q / d theta_k of the client's model (diagonal and normalisation
 * included); out: [K].  Runs on the host. */
PLK_API int plk_chain_rule_rate_matrix(const double* G, const double* dQ, int state_count, int param_count, double* out);

/* S8a step 0.  Encode `taxa` character sequences of `sites` characters each (nucleotide: one site per character;
 * codon: sites must be divisible by 3, one site per triplet) and merge identical columns.
 *   nucleotide  A,C,G,T/U (any case) -> 0..3, anything else -> 4 (missing);
 *   codon       three unambiguous bases -> sense-codon index 0..60 (lexicographic A<C<G<T over the 61 sense codons
 *               of the standard code), any other character in the triplet -> 61; a stop codon -> _STOP_CODON.
 * Patterns are numbered by first occurrence; weight = multiplicity (S8c rows 16-17).
 *   out_states          uint8 [taxa][cap]  (cap = number of columns = sites or sites/3); row stride is `cap`,
 *                       only the first *out_pattern_count entries of each row are meaningful
 *   out_weights         double [cap]
 *   out_site_to_pattern int64 [cap]
 * Runs on the host.  All buffers are the caller's. */
PLK_API int plk_encode_and_compress(int state_kind, int taxa, int64_t sites, const char* const* seqs,
                                    uint8_t* out_states, double* out_weights, int64_t* out_site_to_pattern,
                                    int64_t* out_pattern_count);

#ifdef __cplusplus
}
#endif
#endif /* PLK_H_ */
