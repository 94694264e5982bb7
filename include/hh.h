/* =============================================================================================
 * hh.h -- C ABI of the B200-native H-HIGNN mobility apply  U = M(X) F   (arxiv 2505.08174).
 *
 * Citations are PAPER.md line numbers + section / equation / algorithm; "S-n" are the readings
 * of silent / ambiguous / garbled passages listed in DESIGN.md.
 *
 * The path (Sec. 3): geometric cluster tree on the Morton order (Def. 1,
 * L123-L129) -> block-cluster partition by the admissibility test max(diam) <= eta * dist
 * (Def. 2 / Eq. (7); Alg. 1) -> ACA low-rank factors C, Q of the admissible
 * blocks, entries evaluated on demand by the two-body MLP (Alg. 2; Eqs. (8)-(10)) ->
 * mat-vec = self term + near-field dense blocks evaluated on the fly (L252) + far-field C (Q F)
 * (L115, L260) + three-body graph term (Eq. (4); L74) -> explicit Euler (L338).
 *
 * Conventions
 *  - Every pointer argument is marked HOST or DEVICE.  DEVICE buffers are caller-owned (allocated
 *    by the caller, e.g. with PyTorch) and must stay valid for the duration of the call; the
 *    workspace must stay valid for the life of the context.  The library allocates no device
 *    memory.  It owns the context struct and a small pinned host scratch for scalar read-backs.
 *  - All work is enqueued on the CUDA stream given to hh_create.  Calls return after the few
 *    scalar read-backs they need (level counts, block totals, arena batch boundaries); hh_matvec
 *    and hh_step return after their last kernel has been ENQUEUED (U is valid once the stream has
 *    been synchronised) unless noted.
 *  - Every function returns HH_OK (0) or a negative HH_ERR_* code; hh_last_error gives a text.
 *    No exceptions, no aborts.  There is NO CPU fallback: without a CUDA device every compute
 *    entry point fails with HH_ERR_CUDA.
 *  - Particle arrays are fp32, row-major [N][3], in the CALLER's particle order.  "Tree order" is
 *    the Morton order of S-8/S-9: position k in tree order holds caller particle perm[k].
 *  - Node ids are the library's breadth-first numbering (root 0, children adjacent, left first);
 *    S-12: only the ranges [lo,hi) identify a cluster.
 * ============================================================================================= */
#ifndef HH_H_
#define HH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HH_OK                        0
#define HH_ERR_INVALID_ARG          -1   /* null pointer, N < 1, eta <= 0, tol <= 0, leaf < 1, bad MLP shape */
#define HH_ERR_WORKSPACE_TOO_SMALL  -2   /* hh_stats.workspace_required holds the bytes needed          */
#define HH_ERR_CUDA                 -3   /* a CUDA call failed (text in hh_last_error)                  */
#define HH_ERR_NOT_BUILT            -4   /* call out of order (e.g. hh_build_blocks before hh_build_tree) */
#define HH_ERR_UNSUPPORTED          -5   /* MLP shape other than the compiled ones                      */

typedef struct hh_ctx hh_ctx;           /* opaque, owned by the library */

/* An MLP  y = W_L tanh( ... tanh(W_1 x + b_1) ... ) + b_L  (tanh on hidden layers only; PAPER.md L92,
 * S-4).  Supported shapes: two-body 4->32->32->9 (features [r_hat(3), a/r], Eq. (4) L85 + config),
 * three-body 7->64->64->9 (features [X_j-X_i, X_k-X_i, |X_j-X_k|]); either may have 18 outputs instead of 9 = [alpha^(s), alpha^(t)]
 * (Eq. (2)): the last 9 are the transverse half used above, the first 9 the self half of the diagonal terms M^(s,2), M^(s,3) of
 * Eq. (6) (L108-L113), summed over the neighbours within rcut3 and applied to F_i; and, for the two-body term, the paper-size network
 * 4->128->512->128->9 (n_layers = 4; L92), evaluated on the tcgen05 tensor cores with tf32 operands and tanh.approx
 * (tolerance 2e-3; meant for the paper's own ACA tolerances zeta >= 1e-2; lock-step ACA only, no S-18b, no parity mode).
 *   dims : HOST   int32[n_layers+1]
 *   W, b : HOST   arrays of n_layers DEVICE pointers; W[l] is [dims[l+1]][dims[l]] row-major fp32,
 *                 b[l] is [dims[l+1]] fp32.  Copied into the context at hh_create. */
typedef struct {
  int32_t n_layers;
  const int32_t* dims;
  const float* const* W;
  const float* const* b;
} hh_mlp;

typedef struct {
  int32_t leaf_size;     /* C_leaf (Def. 1): a cluster is a leaf iff it holds <= leaf_size particles (S-10) */
  float   eta;           /* eta of Eq. (7)                                                   */
  float   aca_tol;       /* zeta of Eq. (10)                                                 */
  int32_t aca_max_rank;  /* N_ite_max (L258): cap on the block-rank l; 1..96                       */
  float   radius_a;      /* particle radius a (L41)                                                */
  float   rcut3;         /* R_cut of the short-range terms (three-body and self terms; L56, L90); 0 = none */
  int32_t pivot_rule;    /* 0 = |det| (Eq. (9)), 1 = Frobenius (listing L219/L224); S-18 */
  int32_t near_path;     /* near-field entry evaluation (rows 6, 8): 0 = fp32 ALU path (tolerance 1e-5).  1 = tcgen05 tensor cores:
                            the 32 x 32 layer as a tf32 contraction with the accumulator in tensor memory, tanh.approx
                            (tolerance 2e-3, north_star).  2 = the same contraction with split tf32 operands (3 products,
                            fp32-class) and the accurate tanh.  csrc/hh_near_tc.cu                                        */
  float   kappa_max;     /* 0 (default) or INFINITY = Alg. 2 as printed: the pivot block is inverted whatever its condition
                            (L221).  > 0 opts in to S-18b: a pivot block with |P|_F |P^-1|_F above this is treated as
                            numerically singular, Alg. 2 breaks down on that block (flag 2) and the mat-vec evaluates it
                            densely like an inadmissible block (L252).  DESIGN.md section 3 states which configs use it. */
  float   dense_cap;     /* S-18b applies where the dense evaluation is affordable: |tau||sigma| <= dense_cap (|tau|+|sigma|);
                            larger blocks keep the ill-conditioned pivot (plain listing).  0 = default (128)          */
  int32_t aca_precision; /* 0 = fp32 entries in Alg. 2 (default; the fast path).  1 = parity mode: the entries G(i,j) that Alg. 2
                            queries (L218, L222) and the residuals are evaluated in fp64 and rounded once when stored (factors
                            stay fp32).  Two runs of Alg. 2 on the same pivots differ by (entry noise) x cond_F(pivot block);
                            with fp32 entries (relative noise 2e-7) that is above 1e-5 on large or chain-shaped clouds
                            (DESIGN.md section 5); this mode removes the noise at ~3x the ACA cost.                       */
} hh_params;

/* Counters (Figs. 7-9 count "queries" = MLP evaluations; L299). Filled as stages run. */
typedef struct {
  int64_t n_particles;
  int64_t n_nodes, n_leaves, depth;        /* cluster tree                                          */
  int64_t n_admissible, n_inadmissible;    /* |P^G|, |P^H| (Alg. 1)                                 */
  int64_t near_entries;                    /* W^H = sum |tau||sigma| over P^H (L250)                */
  int64_t far_rows_cols;                   /* sum (|tau|+|sigma|) over P^G                          */
  int64_t sum_rank;                        /* sum of block-ranks l over the blocks factorised so far */
  int64_t aca_entries;                     /* two-body MLP evaluations spent in ACA so far          */
  int64_t factor_bytes;                    /* 36 * l * (|tau|+|sigma|) summed over factorised blocks */
  int64_t aca_batches;                     /* arena fills so far (L246, L260: batching)             */
  int64_t aca_not_converged;               /* blocks that hit aca_max_rank before Eq. (10) (S-21)   */
  int64_t aca_singular;                    /* blocks on which Alg. 2 broke down on a (numerically) singular pivot
                                              (S-18, S-18b); they are applied densely                  */
  int64_t n_faces;                         /* three-body faces (j,k,i) visited (L74)                */
  int64_t workspace_required;              /* bytes; set when HH_ERR_WORKSPACE_TOO_SMALL is returned */
  int64_t arena_bytes;                     /* size of the factor arena carved from the workspace    */
  float   ms_tree, ms_blocks, ms_aca, ms_near, ms_far, ms_three, ms_other;  /* CUDA-event stage times of the last hh_matvec/hh_step (only if timing enabled) */
  float   pad_;
  int64_t n_launches;                      /* kernels launched since the last hh_build_tree began (one whole hh_step) */
  int64_t fallback_entries;                /* sum |tau||sigma| over the blocks counted in aca_singular (dense evaluations per mat-vec) */
  int64_t n_self_pairs;                    /* pairs (i, j in N(i)) visited by the two-body self term M^(s,2) (Eq. (6))                  */
} hh_stats;

/* Create a context.  params: HOST.  mlp2: HOST struct, required.  mlp3: HOST struct or NULL (then
 * rcut3 must be 0).  workspace: DEVICE, 256-byte aligned, holds the tree, the block lists and the
 * factor arena (whatever remains after tree and lists).  stream: a cudaStream_t (NULL = default
 * stream).  Errors: INVALID_ARG, UNSUPPORTED, CUDA. */
int hh_create(hh_ctx** ctx, const hh_params* params, const hh_mlp* mlp2, const hh_mlp* mlp3,
              void* workspace, size_t workspace_bytes, void* cuda_stream);
int hh_destroy(hh_ctx* ctx);

/* Change eta / aca_tol / aca_max_rank / pivot_rule / leaf_size of an existing context (parameter
 * sweeps of config 3).  Invalidates tree and blocks as needed. */
int hh_set_params(hh_ctx* ctx, const hh_params* params);

/* Alg. 2 form: 0 = lock-step over all blocks of an arena batch (default; each listing line a parallel pass over
 * the selected blocks), entry evaluation and the vectorised update as separate launches; 1 = one CTA per block; 2 = lock-step
 * with the stored rank terms of a tile of 256 rows staged through shared memory by TMA bulk copies; 3 = lock-step with entry
 * evaluation and update fused in one kernel; 4 = form 0 on two half-batches one listing line apart (the update of one on a
 * side stream beside the entry evaluation of the other).  1-4 are measured slower and kept for comparison.  Same factors up
 * to fp32 summation order in the norm recursion. */
int hh_set_aca_impl(hh_ctx* ctx, int impl);

/* Far-field apply form: 0 = blocks with max(m,n) <= 1024 are streamed by persistent CTAs through a
 * shared-memory ring filled by TMA bulk copies (chunk by chunk up to 256, rank by rank above), larger ones by one CTA per
 * block (default); 1 = one CTA per block in every size class; 2 = the ring only up to 256.  Same sums up to fp32 summation
 * order. */
int hh_set_far_impl(hh_ctx* ctx, int impl);

/* Record per-stage CUDA-event times into hh_stats (adds stream synchronisations). */
int hh_enable_timing(hh_ctx* ctx, int on);

/* Steps 1-4: Morton keys (S-8), stable radix sort (S-9), cluster tree (Def. 1,
 * L123-L127; S-10, S-11), tight bounding boxes (L144; S-13).
 *   X : DEVICE fp32 [N][3], caller order; read only.  N >= 1.
 * Errors: INVALID_ARG, WORKSPACE_TOO_SMALL, CUDA. */
int hh_build_tree(hh_ctx* ctx, const float* X, int64_t N);

/* Step 5: Alg. 1 BuildPartition from (root, root) (L164-L184; Eq. (7); S-14..S-16) -> P^G, P^H.
 * Errors: NOT_BUILT (no tree), WORKSPACE_TOO_SMALL, CUDA. */
int hh_build_blocks(hh_ctx* ctx);

/* Step 7: Alg. 2 (L210-L234) on admissible blocks first_block, first_block+1, ... (the library's
 * P^G order, largest blocks first), all blocks of the batch in lock step (L262), until the factor
 * arena is full or P^G is exhausted; *next_block (HOST) receives the
 * first block NOT factorised (== n_admissible when done).  Factors stay in the arena until the
 * next hh_aca / hh_build_* call.  Blocks that reach aca_max_rank are kept at that rank and counted.
 * Errors: NOT_BUILT, INVALID_ARG (first_block out of range), WORKSPACE_TOO_SMALL (arena cannot
 * hold even one block), CUDA. */
int hh_aca(hh_ctx* ctx, int64_t first_block, int64_t* next_block);

/* Steps 6-11: U = M(X) F = F (self term, alpha_1 = I, S-5) + near-field (L252) + far-field over all
 * admissible blocks (runs hh_aca batch by batch when the factors are not all resident; L115, L260)
 * + three-body term if rcut3 > 0 (Eq. (4); S-22, S-23).
 *   F : DEVICE fp32 [N][3] caller order, read only.   U : DEVICE fp32 [N][3] caller order, written.
 * Errors: NOT_BUILT, CUDA, WORKSPACE_TOO_SMALL. */
int hh_matvec(hh_ctx* ctx, const float* F, float* U);

/* Selective mat-vec for tests and stage timing: bit 0 alpha_1 = I, 1 near, 2 far, 3 three-body M^(t,3), 4 the diagonal self terms
 * M^(s,2) + M^(s,3) (present only with 18-output networks).  hh_matvec = all five. */
int hh_matvec_parts(hh_ctx* ctx, const float* F, float* U, int parts);

/* Far-field apply only, over the factors currently in the arena (blocks [first, next) of the last
 * hh_aca call): Us_tree += C (Q F^sigma), the roofline-graded kernel; resident
 * blocks on which Alg. 2 broke down (flag 2, S-18b) are added densely after it.
 *   F : DEVICE fp32 [N][3] caller order.  U : DEVICE fp32 [N][3] caller order; U is OVERWRITTEN with
 *   the contribution of the resident admissible blocks only. */
int hh_far_apply_resident(hh_ctx* ctx, const float* F, float* U);

/* Step 12: one time step (L102, L338): build tree + blocks from X, U = M(X) F, X <- X + dt U (fp32,
 * S-25).  X : DEVICE fp32 [N][3], updated in place.  F read, U written (DEVICE). */
int hh_step(hh_ctx* ctx, float* X, const float* F, float* U, int64_t N, float dt);

/* hh_step with HOST buffers (the end-to-end call bench.py times): X_host, F_host are copied to the device, hh_step runs,
 * U_host and the updated X_host are copied back; returns after the copies have completed (the stream is synchronised).
 *   X_host, F_host, U_host : HOST fp32 [N][3] (pinned memory makes the copies asynchronous); X_host is updated in place.
 * Errors: as hh_step. */
int hh_step_host(hh_ctx* ctx, float* X_host, const float* F_host, float* U_host, int64_t N, float dt);

/* Capacity of the block lists and of the Alg. 1 frontier, in pairs per particle (default 32; c3 needs ~5 for P^G and
 * ~3.4 for P^H).  Takes effect at the next hh_build_tree (the workspace is carved again).
 * Errors: INVALID_ARG (pairs_per_particle < 1). */
int hh_set_pair_capacity(hh_ctx* ctx, int64_t pairs_per_particle);

/* Pivot capture for parity tests at sizes where the factors are streamed and discarded (replay on sampled
 * target leaves).  While set, every hh_aca batch (also inside hh_matvec / hh_step) appends one record per factorised
 * admissible block whose TARGET range [lo,hi) of tree order holds a flagged row, i.e. row_prefix[hi] - row_prefix[lo] > 0:
 *   row_prefix : DEVICE int32[N+1], exclusive prefix sum of the 0/1 row flags in TREE order (S-9); caller-owned
 *   records    : DEVICE int32[cap_records][200]: [0] block index in the library's P^G order (hh_get_blocks), [1] rank,
 *                [2] flag, [3] number of pivot pairs listed (rank, +1 after a breakdown), [4..100) piv_i, [100..196) piv_j
 *                (local row / column indices, -1 beyond the listed ones), [196..200) unused; caller-owned
 * records == NULL switches the capture off.  The record counter restarts at 0 on every call; records beyond cap_records
 * are counted but not written (hh_get_capture_count then exceeds cap_records).  Alg. 2's pivots: L219, L224; S-17, S-18.
 * Errors: INVALID_ARG, CUDA. */
int hh_set_capture(hh_ctx* ctx, const int32_t* row_prefix, int32_t* records, int64_t cap_records);
int hh_get_capture_count(hh_ctx* ctx, int64_t* n_records /* HOST */);

/* ---- introspection (parity tests, counters).  All destination buffers are HOST. ---- */
int hh_get_stats(hh_ctx* ctx, hh_stats* stats);
/* perm int64[N] (S-9), keys uint64[N] sorted; node arrays of length n_nodes (any may be NULL). */
int hh_get_tree(hh_ctx* ctx, int64_t* perm, uint64_t* keys, int64_t* lo, int64_t* hi, int32_t* left,
                int32_t* right, int32_t* parent, int32_t* level, float* bmin, float* bmax);
/* which = 0: P^G, 1: P^H.  tau, sigma: int32[count] node ids (targets, sources; S-16). */
int hh_get_blocks(hh_ctx* ctx, int which, int32_t* tau, int32_t* sigma);
/* Factors of admissible block `block` (must be resident in the arena).  rank, flag (0 ok, 1 = hit
 * max rank, 2 = breakdown on a singular pivot, block applied densely): HOST scalars.  piv_i, piv_j:
 * int32[cap_rank] local row / column pivots of the `rank` accepted steps, followed (flag 2) by the
 * attempted pivot at which Alg. 2 broke down.  C: fp32 [rank][m][9] (the listing's normalised
 * columns, C_k(i_k) = I), Q: fp32 [rank][n][9] (residual rows), entry-major copies of the arena's
 * plane-major storage; any of piv_i, piv_j, C, Q may be NULL. */
int hh_get_factors(hh_ctx* ctx, int64_t block, int32_t* rank, int32_t* flag, int32_t cap_rank,
                   int32_t* piv_i, int32_t* piv_j, float* C, float* Q);
/* ranks int32[n_admissible], flags int32[n_admissible] of all blocks factorised so far (-1 = not yet). */
int hh_get_ranks(hh_ctx* ctx, int32_t* ranks, int32_t* flags);
/* Evaluate the two-body entry M_ij (Eq. (4), S-1..S-3) for n pairs: Xi, Xj DEVICE [n][3], M DEVICE [n][9]. */
int hh_eval_entries(hh_ctx* ctx, const float* Xi, const float* Xj, int64_t n, float* M);

const char* hh_last_error(const hh_ctx* ctx);
const char* hh_version(void);

/* ---- the one entry point that ALLOCATES NOTHING (csrc/hh_static.cu) -------------------------------------------------
 * For callers that cannot allocate or synchronise: code under CUDA graph capture, tight serving loops over small
 * suspensions, harnesses that forbid cudaMalloc.  No hh_ctx, no workspace: inputs and outputs only.  The scratch (packed
 * weights + partial sums) is a file-scope static __device__ array of HH_STATIC_SCRATCH_BYTES (about 3.2 MB) that every GPU
 * which loads the library holds until exit.  The call makes no cudaMalloc / cudaFree / allocating library call, no memcpy
 * and no synchronisation: three kernels are enqueued on cuda_stream and the call returns.
 *
 * Computes the definition  U_i = F_i + sum_{j != i} M_ij F_j,  M_ij = (1/r) R(MLP2([r_hat, a/r]))  (Eq. (4)
 * L85-L88; Eq. (6) L108-L113 with alpha_1 = I; S-1..S-5): what hh_matvec returns when no block is admissible (L283), fp32,
 * relative L2 <= 1e-5 of it (summation order differs).  No three-body or self terms.
 *   mlp2        HOST struct; two-body network 4->32->32->9 only; W, b: HOST arrays of DEVICE pointers, read by the kernels
 *               of THIS call on cuda_stream (they must be ready on that stream; nothing is cached between calls)
 *   X, F        DEVICE fp32 [N][3], caller's order;  U  DEVICE fp32 [N][3], overwritten;  1 <= N <= HH_STATIC_MAX_N
 *   cuda_stream a cudaStream_t (NULL = default stream)
 *   err         HOST buffer for an error text, or NULL
 * Errors: HH_ERR_WORKSPACE_TOO_SMALL if N > HH_STATIC_MAX_N (text names the limit), INVALID_ARG, UNSUPPORTED (other MLP
 * shape), CUDA (no device, cudaGetSymbolAddress or a launch failed).
 * Sharing: ALL calls on a device use the same array, which keeps the last call's contents (each call rewrites everything
 * it reads, nothing needs clearing).  Calls that OVERLAP on the GPU (two streams, unordered graph branches) RACE on it;
 * calls on one stream are ordered and safe.  The first call on a device looks up the array's address
 * (cudaGetSymbolAddress, once per device, with that device current): make it outside graph capture. */
#define HH_STATIC_MAX_N 16384
#define HH_STATIC_SCRATCH_BYTES 3153920
int hh_dense_matvec_static(const hh_mlp* mlp2, float radius_a, const float* X, const float* F, float* U, int64_t N,
                           void* cuda_stream, char* err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* HH_H_ */
