// hh_internal.cuh -- shared declarations of the CUDA path (context, workspace layout, primitives).
// Product code.  Shares nothing with oracle/.  Citations: PAPER.md line numbers; S-n = DESIGN.md readings.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "../../include/hh.h"

typedef uint32_t u32;
typedef uint64_t u64;

#define HH_MAX_RANK 96                          /* cap on N_ite_max (L258)                         */
#define HH_RC 4                                 /* ranks per arena chunk                           */
#define HH_MAX_CHUNKS (HH_MAX_RANK / HH_RC)     /* 24                                              */
#define HH_UNIT_FLOATS 32                       /* arena allocation unit = 128 B                   */
#define HH_TAB_STRIDE 32                        /* u32 per resident block: 24 chunk offsets + pivot offset + pad */
#define HH_TAB_PIV 24
#define HH_MAX_LEAF 256                         /* largest supported C_leaf                        */
#define HH_MAX_LEVELS 128
#ifndef HH_FAR_MID_MAX
#define HH_FAR_MID_MAX 1024                     /* far-field apply: blocks with 256 < max(m,n) <= this go through k_far_mid (hh_far.cu) */
#endif
#define HH_CAP_STRIDE 200                      /* int32 per captured pivot record (hh.h: hh_set_capture) */

/* packed MLP weights (floats) as laid out for the kernels: W1 [H][INP], b1 [H], W2 [H][H], b2 [H],
 * W3T [H][12] (9 outputs of hidden unit o, 3 pad), b3 [12]                                        */
#define HH_MLP_FLOATS(INP, H) ((H) * (INP) + (H) + (H) * (H) + (H) + (H) * 12 + 12)
#define HH_MLP2_INP 4
#define HH_MLP2_H 32
#define HH_MLP3_INP 8
#define HH_MLP3_H 64
#define HH_MLP2_FLOATS HH_MLP_FLOATS(HH_MLP2_INP, HH_MLP2_H)   /* 1612 */
#define HH_MLP3_FLOATS HH_MLP_FLOATS(HH_MLP3_INP, HH_MLP3_H)   /* 5516 */

struct Cnt3 { u32 g, h, c; };
__host__ __device__ inline Cnt3 operator+(Cnt3 a, Cnt3 b) { return Cnt3{a.g + b.g, a.h + b.h, a.c + b.c}; }

/* device-side scalars (one 256-B slot at the start of the workspace) + pinned host mirror */
struct DevScalars {
  float bb[6];              /* min xyz, max xyz of X as order-preserving uints while reducing, floats after */
  u32 bbu[6];
  u32 n_split;              /* tree: nodes split at the current level                                 */
  u32 pad0;
  Cnt3 lvl;                 /* Alg. 1: totals of the current level (admissible, inadmissible, children) */
  u32 n_leaves;
  u64 arena_cursor;         /* in units                                                               */
  u32 fail_min;             /* first block whose arena allocation failed                              */
  u32 batch_end;            /* result of the batch-range search                                       */
  u32 class_bound[4];       /* first block of ACA class 1,2,3 in the sorted P^G (class 0 starts at 0) */
  u64 sum_rank, aca_entries, factor_bytes, n_faces;
  u32 not_conv, singular, deg_overflow;
  u32 aca_err;              /* k2_step_t: 1 = an mbarrier wait timed out                                                 */
  u32 far_err;              /* k_far_ring / k_far_fill: 1 = an mbarrier wait timed out, 2 = item list overflow          */
  u64 near_entries, far_rows_cols;
  u32 max_rank_seen, n_dense;
  u64 fallback_entries;
  u64 n_self_pairs;         /* pairs (i, j in N(i)) visited by the two-body self term */
  u64 cap_count;            /* pivot records written by hh_set_capture's kernel (may exceed the caller's capacity) */
  u32 batch_mid;            /* lock-step ACA, two half-batches in flight: first block of the second half (half of the rows + columns each) */
  u32 ab[6];                /* per half: active blocks [0,1], row granules [2,3], column granules [4,5]                     */
  u64 batch_units, batch_units1;  /* lock-step ACA: padded rows + columns of the batch [first, batch_end) resp. of block `first` alone */
};

struct hh_ctx {
  hh_params p;
  cudaStream_t stream;
  char* ws;  size_t ws_bytes;
  char err[512];
  int have_mlp3;
  int timing;
  int aca_impl;                         /* 0 = lock-step, entries and vectorised update in separate launches (hh_aca2.cu), 1 = one CTA per block (hh_aca.cu), 2 = lock-step, stored terms staged by TMA, 3 = lock-step, fused k2_step */
  int n_sm;                             /* cudaDevAttrMultiProcessorCount of the context's device (grid sizing) */
  int three_smem_set;                   /* k_three's dynamic shared-memory attribute has been set on this device */
  int64_t pairs_per_particle;
  /* state */
  int64_t N, Ncap;
  int tree_ok, blocks_ok;
  int n_nodes, n_levels, n_leaves;
  int lvl_start[HH_MAX_LEVELS + 1];
  int64_t nG, nH, cap_pairs;
  int64_t res_first, res_next;          /* resident factor range [first, next) of sorted P^G */
  double l_pred;                        /* predicted rank for batch sizing                   */
  double l_pred_first;                  /* what the FIRST batch of a mat-vec (the largest blocks) needed last time: the next mat-vec starts from it
                                           instead of the last batch's prediction (leaf-size blocks, half the rank), which made every step's first batch
                                           overflow the arena and run twice (c3: 750 ms of a 5.4 s step) */
  u32 class_bound[5];
  u32 mid_bound;                        /* first block of sorted P^G with max(m,n) <= HH_FAR_MID_MAX */
  hh_stats st;
  int64_t n_launches;                   /* kernels launched since the last hh_build_tree began (claim for bench.py) */
  /* pinned host scratch */
  DevScalars* h_sc;
  cudaEvent_t ev[8];
  cudaStream_t stream2;                 /* side stream of the two-half lock-step ACA (hh_set_aca_impl 4): carries the update kernel of one half while the other half's entries are evaluated */
  cudaEvent_t ev_ab[2];
  /* carved device pointers */
  DevScalars* d_sc;
  float *w2, *w3;                       /* packed weights                                     */
  float *w2s, *w3s;                     /* self halves of 18-output networks, packed as 9-output sets (Eq. (2)) */
  int have_self2, have_self3;
  float* w2tc;                          /* W2 as the tensor-core B operand: tf32 hi | lo, core-matrix layout (near_path 1, 2) */
  int mlp2_wide;                        /* the two-body MLP is the paper-size 4-128-512-128-9 (hh_wide.cuh)  */
  float* w2w;                           /* its packed weights (hh_pack_wide)                                    */
  double* w2d;                          /* the two-body weights as fp64 (aca_precision = 1)   */
  u64 *keys[2]; u32 *idx[2];            /* radix ping-pong                                    */
  u32* hist;  size_t hist_cap;          /* radix histograms / generic scan tile sums          */
  void* tilesum;                        /* tile sums for scans (Cnt3 / u64)                   */
  float *Xs, *Fs, *Us;                  /* tree order                                         */
  u32* perm;
  u32 *nlo, *nhi; int *nleft, *nparent, *nlevel; u32* nsplit; u32* nflag;
  float *bmin, *bmax;                   /* [nodes][3]                                         */
  u32* leaf_nodes;
  uint2 *PG, *PH;                       /* (tau, sigma) node ids; PG sorted by size desc, PH by tau */
  u32 *near_begin, *near_end;           /* per node: range in PH                              */
  int* ranks; int* flags;               /* per admissible block                               */
  u32* dense_list; u32* dense_cnt; u32 n_dense;         /* resident blocks on which Alg. 2 broke down (S-18b): applied densely */
  u64* unit_prefix;                     /* prefix of (m_pad + n_pad) over sorted PG, nG+1     */
  char* scratch; size_t scratch_bytes;  /* frontier ping-pong during build; == arena region    */
  float* arena; u64 arena_units;        /* after the resident table                            */
  u32* tab;                             /* resident block table, HH_TAB_STRIDE u32 per block   */
  /* far-field ring kernel (hh_far.cu): item list of the resident blocks of the leaf-size classes */
  int far_impl;                         /* 0 = ring kernel for max(m,n) <= 256 (default), 1 = one CTA per block everywhere */
  int far_built, far_smem_set, aca_smem_set;
  u32* far_cnt; uint4* far_items; size_t far_items_cap;
  /* three-body cell list */
  u32 *cell_of, *cell_start, *cell_order; int64_t n_cells_cap;
  /* pivot capture for at-size parity tests (hh_set_capture) */
  const int32_t* cap_prefix; int32_t* cap_rec; int64_t cap_max;
  /* host staging for *_host calls */
  float *stageX, *stageF, *stageU;
};

#define HH_CUDA(call)                                                                     \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      snprintf(ctx->err, sizeof ctx->err, "%s:%d %s -> %s", __FILE__, __LINE__, #call,   \
               cudaGetErrorString(e_));                                                   \
      return HH_ERR_CUDA;                                                                 \
    }                                                                                     \
  } while (0)
#define HH_TRY(call) do { int r_ = (call); if (r_ != HH_OK) return r_; } while (0)
#define HH_LAUNCH_CHECK() HH_CUDA(cudaGetLastError())
/* every kernel launch is written  k<<<HH_N + grid, block, smem, stream>>>(...)  and counts itself */
#define HH_N (++ctx->n_launches, 0u)

static inline int hh_fail(hh_ctx* ctx, int code, const char* msg) {
  snprintf(ctx->err, sizeof ctx->err, "%s", msg);
  return code;
}
static inline unsigned cdiv(int64_t a, int64_t b) { return (unsigned)((a + b - 1) / b); }

/* ---- primitives (hh_prims.cu) ---- */
int hh_scan_u32(hh_ctx* ctx, const u32* in, u32* out, int64_t n, u32* total_dev /*may be null*/);
int hh_scan_u64(hh_ctx* ctx, const u64* in, u64* out, int64_t n, u64* total_dev);
int hh_scan_cnt3(hh_ctx* ctx, Cnt3* tiles, int64_t ntiles, Cnt3* total_dev);   /* in place, exclusive */
/* stable LSD radix sort of (key, val) on bits [bit_lo, bit_hi); result index (0/1) of ping-pong in *which */
int hh_sort_pairs(hh_ctx* ctx, u64* keys[2], u32* vals[2], int64_t n, int bit_lo, int bit_hi, int* which);

/* ---- stages ---- */
int hh_tree_build(hh_ctx* ctx, const float* X, int64_t N);
int hh_blocks_build(hh_ctx* ctx);
int hh_near_apply(hh_ctx* ctx);                                       /* Us += near-field           */
int hh_near_apply_wide(hh_ctx* ctx);                                  /* paper-size MLP (hh_wide.cu) */
int hh_entries_eval_wide(hh_ctx* ctx, const float* Xi, const float* Xj, int64_t n, float* M);
int hh_pack_wide(hh_ctx* ctx, const hh_mlp* m, float* out);
size_t hh_wide_floats(void);
int hh_near_apply_tc(hh_ctx* ctx);                                    /* the same on tcgen05 tensor cores (hh_near_tc.cu) */
void hh_pack_w2_tc(const float* W2, float* out);                      /* host: W2 [32][32] -> 2 x 1024 floats */
int hh_dense_apply(hh_ctx* ctx);                                      /* Us += resident blocks on which ACA broke down, densely */
int hh_aca_batch(hh_ctx* ctx, int64_t first, int64_t* next);      /* one CTA per block (hh_aca.cu)        */
int hh_aca2_batch(hh_ctx* ctx, int64_t first, int64_t* next);     /* lock-step over the batch (hh_aca2.cu) */
int hh_aca_batch_finish(hh_ctx* ctx, int64_t first, u32 end, int64_t* next);   /* stats, dense list, rank prediction */
int hh_far_apply(hh_ctx* ctx);                                        /* Us += resident far-field   */
int hh_three_apply(hh_ctx* ctx, int modes);                          /* Us += short-range terms (tree order): bit 0 M^(t,3), 1 M^(s,3), 2 M^(s,2) */
int hh_entries_eval(hh_ctx* ctx, const float* Xi, const float* Xj, int64_t n, float* M);
int hh_factors_fetch(hh_ctx* ctx, int64_t block, int32_t* rank, int32_t* flag, int32_t cap_rank,
                     int32_t* piv_i, int32_t* piv_j, float* C, float* Q);

/* ---- device helpers ---- */
#ifdef __CUDACC__
__device__ __forceinline__ u32 lane_id() { return threadIdx.x & 31; }

/* exclusive scan of one u32 per thread across the block; returns exclusive prefix, *total = block sum.
 * smem: 33 u32.  All threads must call. */
template <typename T>
__device__ __forceinline__ T block_excl_scan(T v, T* smem /* >= 33 */, T* total) {
  const u32 lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  T inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    T t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (u32)o) inc += t;
  }
  if (lane == 31) smem[w] = inc;
  __syncthreads();
  if (w == 0) {
    T s = lane < nw ? smem[lane] : T(0);
    T si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      T t = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= (u32)o) si += t;
    }
    smem[lane] = si - s;
    if (lane == 31) smem[32] = si;
  }
  __syncthreads();
  T base = smem[w];
  *total = smem[32];
  __syncthreads();
  return base + inc - v;
}
#endif
