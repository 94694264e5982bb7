// hh_tree.cu -- SURVEY 8(a) rows 1-4: Morton keys (S-8), stable radix sort (S-9), cluster tree
// (Def. 1; S-10, S-11), tight bounding boxes (L144; S-13).
#include "hh_internal.cuh"

__device__ __forceinline__ u32 f2ord(float f) { u32 u = __float_as_uint(f); return (u & 0x80000000u) ? ~u : (u | 0x80000000u); }
__device__ __forceinline__ float ord2f(u32 o) { u32 u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o; return __uint_as_float(u); }

__global__ void k_init_bbox(DevScalars* sc) {
  if (threadIdx.x < 3) { sc->bbu[threadIdx.x] = 0xffffffffu; sc->bbu[3 + threadIdx.x] = 0u; }
}

// min/max of the centres: fp32 min/max are exact and order-free.
__global__ void __launch_bounds__(256) k_bbox(const float* __restrict__ X, int64_t N, DevScalars* sc) {
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
    for (int c = 0; c < 3; ++c) { float v = X[3 * i + c]; lo[c] = fminf(lo[c], v); hi[c] = fmaxf(hi[c], v); }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c)
    for (int o = 16; o; o >>= 1) {
      lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o));
      hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
    }
  if ((threadIdx.x & 31) == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      if (lo[c] != INFINITY) atomicMin(&sc->bbu[c], f2ord(lo[c]));
      if (hi[c] != -INFINITY) atomicMax(&sc->bbu[3 + c], f2ord(hi[c]));
    }
  }
}

__device__ __forceinline__ u64 spread21(u64 v) {   // bit b -> bit 3b
  v &= 0x1fffffull;
  v = (v | (v << 32)) & 0x1f00000000ffffull;
  v = (v | (v << 16)) & 0x1f0000ff0000ffull;
  v = (v | (v << 8)) & 0x100f00f00f00f00full;
  v = (v | (v << 4)) & 0x10c30c30c30c30c3ull;
  v = (v | (v << 2)) & 0x1249249249249249ull;
  return v;
}

// S-8: root cube anchored at the minimum corner, quantised in fp64 with individually rounded
// sub / div / mul (nothing to contract), 21 bits per axis, x in the top bit of each triple.
__global__ void __launch_bounds__(256) k_morton(const float* __restrict__ X, int64_t N, const DevScalars* __restrict__ sc,
                                                 u64* __restrict__ keys, u32* __restrict__ idx) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  double lo[3], ext = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = (double)ord2f(sc->bbu[c]);
    double e = __dsub_rn((double)ord2f(sc->bbu[3 + c]), lo[c]);
    ext = e > ext ? e : ext;
  }
  u64 q[3] = {0, 0, 0};
  if (ext > 0.0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double t = __dmul_rn(__ddiv_rn(__dsub_rn((double)X[3 * i + c], lo[c]), ext), 2097152.0);
      double f = floor(t);
      q[c] = (f >= 2097151.0) ? 2097151ull : (u64)f;
    }
  }
  keys[i] = (spread21(q[0]) << 2) | (spread21(q[1]) << 1) | spread21(q[2]);
  idx[i] = (u32)i;
}

__global__ void __launch_bounds__(256) k_gather_x(const float* __restrict__ X, const u32* __restrict__ idx, int64_t N,
                                                   float* __restrict__ Xs, u32* __restrict__ perm) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  u32 p = idx[k];
  perm[k] = p;
  Xs[3 * k] = X[3 * (size_t)p]; Xs[3 * k + 1] = X[3 * (size_t)p + 1]; Xs[3 * k + 2] = X[3 * (size_t)p + 2];
}

__global__ void k_init_root(u32* nlo, u32* nhi, int* nleft, int* nparent, int* nlevel, u32 N) {
  nlo[0] = 0; nhi[0] = N; nleft[0] = -1; nparent[0] = -1; nlevel[0] = 0;
}

// Def. 1 + S-10/S-11: a node with more than C_leaf particles is split at the highest bit in which its
// first and last keys differ (geometric bisection of the root cube cycling x,y,z; empty halves skipped).
__global__ void __launch_bounds__(256) k_split(const u64* __restrict__ keys, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                int* __restrict__ nleft, u32* __restrict__ nsplit, u32* __restrict__ nflag,
                                                int start, int count, u32 leaf) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  int id = start + t;
  u32 lo = nlo[id], hi = nhi[id];
  if (hi - lo <= leaf) { nleft[id] = -1; nflag[id] = 0; return; }
  u64 a = keys[lo], b = keys[hi - 1];
  u32 m;
  if (a == b) {
    m = lo + (hi - lo) / 2;
  } else {
    int bit = 63 - __clzll((long long)(a ^ b));
    u32 l = lo, r = hi - 1;              // keys[l] has bit 0, keys[r] has bit 1; find first with bit 1
    while (r - l > 1) {
      u32 mid = l + (r - l) / 2;
      if ((keys[mid] >> bit) & 1ull) r = mid; else l = mid;
    }
    m = r;
  }
  nsplit[id] = m;
  nleft[id] = -2;
  nflag[id] = 1;
}

__global__ void __launch_bounds__(256) k_children(u32* __restrict__ nlo, u32* __restrict__ nhi, int* __restrict__ nleft,
                                                   int* __restrict__ nparent, int* __restrict__ nlevel,
                                                   const u32* __restrict__ nsplit, const u32* __restrict__ nrank,
                                                   int start, int count, int level) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  int id = start + t;
  if (nleft[id] != -2) return;
  int L = start + count + 2 * (int)nrank[id];
  u32 lo = nlo[id], hi = nhi[id], m = nsplit[id];
  nleft[id] = L;
  nlo[L] = lo; nhi[L] = m; nlo[L + 1] = m; nhi[L + 1] = hi;
  nleft[L] = -1; nleft[L + 1] = -1;
  nparent[L] = id; nparent[L + 1] = id;
  nlevel[L] = level + 1; nlevel[L + 1] = level + 1;
}

__global__ void __launch_bounds__(256) k_leaf_flag(const int* __restrict__ nleft, int n, u32* __restrict__ flag) {
  int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id < n) flag[id] = nleft[id] < 0 ? 1u : 0u;
}
__global__ void __launch_bounds__(256) k_leaf_compact(const int* __restrict__ nleft, const u32* __restrict__ rank, int n,
                                                       u32* __restrict__ leaf_nodes) {
  int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id < n && nleft[id] < 0) leaf_nodes[rank[id]] = (u32)id;
}

// S-13: tight AABB of the centres.  One warp per leaf.
__global__ void __launch_bounds__(256) k_leaf_boxes(const float* __restrict__ Xs, const u32* __restrict__ leaf_nodes, int n_leaves,
                                                     const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                     float* __restrict__ bmin, float* __restrict__ bmax) {
  int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_leaves) return;
  u32 id = leaf_nodes[w];
  u32 lo = nlo[id], hi = nhi[id];
  float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (u32 k = lo + lane; k < hi; k += 32)
#pragma unroll
    for (int c = 0; c < 3; ++c) { float v = Xs[3 * (size_t)k + c]; mn[c] = fminf(mn[c], v); mx[c] = fmaxf(mx[c], v); }
#pragma unroll
  for (int c = 0; c < 3; ++c)
    for (int o = 16; o; o >>= 1) {
      mn[c] = fminf(mn[c], __shfl_xor_sync(0xffffffffu, mn[c], o));
      mx[c] = fmaxf(mx[c], __shfl_xor_sync(0xffffffffu, mx[c], o));
    }
  if (lane < 3) { bmin[3 * (size_t)id + lane] = mn[lane]; bmax[3 * (size_t)id + lane] = mx[lane]; }
}

__global__ void __launch_bounds__(256) k_merge_boxes(const int* __restrict__ nleft, float* __restrict__ bmin, float* __restrict__ bmax,
                                                      int start, int count) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  int id = start + t;
  int L = nleft[id];
  if (L < 0) return;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    bmin[3 * (size_t)id + c] = fminf(bmin[3 * (size_t)L + c], bmin[3 * (size_t)L + 3 + c]);
    bmax[3 * (size_t)id + c] = fmaxf(bmax[3 * (size_t)L + c], bmax[3 * (size_t)L + 3 + c]);
  }
}

int hh_tree_build(hh_ctx* ctx, const float* X, int64_t N) {
  cudaStream_t s = ctx->stream;
  ctx->tree_ok = ctx->blocks_ok = 0;
  ctx->res_first = ctx->res_next = 0;
  ctx->N = N;
  // rows 1-2: keys, sort, gather
  k_init_bbox<<<HH_N + 1, 32, 0, s>>>(ctx->d_sc);
  unsigned gb = cdiv(N, 256);
  k_bbox<<<HH_N + (gb < 8u * ctx->n_sm ? gb : 8u * ctx->n_sm), 256, 0, s>>>(X, N, ctx->d_sc);
  k_morton<<<HH_N + gb, 256, 0, s>>>(X, N, ctx->d_sc, ctx->keys[0], ctx->idx[0]);
  HH_LAUNCH_CHECK();
  int which = 0;
  HH_TRY(hh_sort_pairs(ctx, ctx->keys, ctx->idx, N, 0, 64, &which));
  if (which) {   // keep the sorted keys in keys[0]
    u64* tk = ctx->keys[0]; ctx->keys[0] = ctx->keys[1]; ctx->keys[1] = tk;
    u32* ti = ctx->idx[0]; ctx->idx[0] = ctx->idx[1]; ctx->idx[1] = ti;
  }
  k_gather_x<<<HH_N + gb, 256, 0, s>>>(X, ctx->idx[0], N, ctx->Xs, ctx->perm);
  // row 3: level-synchronous top-down tree, children adjacent, breadth-first numbering
  k_init_root<<<HH_N + 1, 1, 0, s>>>(ctx->nlo, ctx->nhi, ctx->nleft, ctx->nparent, ctx->nlevel, (u32)N);
  HH_LAUNCH_CHECK();
  int start = 0, count = 1, level = 0;
  int64_t node_cap = 2 * ctx->Ncap;
  ctx->lvl_start[0] = 0;
  while (count > 0) {
    if (level >= HH_MAX_LEVELS) return hh_fail(ctx, HH_ERR_INVALID_ARG, "cluster tree deeper than HH_MAX_LEVELS");
    k_split<<<HH_N + cdiv(count, 256), 256, 0, s>>>(ctx->keys[0], ctx->nlo, ctx->nhi, ctx->nleft, ctx->nsplit, ctx->nflag, start, count,
                                             (u32)ctx->p.leaf_size);
    HH_TRY(hh_scan_u32(ctx, ctx->nflag + start, ctx->nflag + start, count, &ctx->d_sc->n_split));
    HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->n_split, &ctx->d_sc->n_split, sizeof(u32), cudaMemcpyDeviceToHost, s));
    HH_CUDA(cudaStreamSynchronize(s));
    int nsp = (int)ctx->h_sc->n_split;
    if ((int64_t)start + count + 2 * (int64_t)nsp > node_cap) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "node capacity exceeded");
    if (nsp > 0)
      k_children<<<HH_N + cdiv(count, 256), 256, 0, s>>>(ctx->nlo, ctx->nhi, ctx->nleft, ctx->nparent, ctx->nlevel, ctx->nsplit,
                                                  ctx->nflag, start, count, level);
    start += count;
    count = 2 * nsp;
    ++level;
    ctx->lvl_start[level] = start;
  }
  ctx->n_levels = level;          // levels 0 .. level-1 are non-empty
  ctx->n_nodes = start;
  // leaves, in node order
  int nn = ctx->n_nodes;
  k_leaf_flag<<<HH_N + cdiv(nn, 256), 256, 0, s>>>(ctx->nleft, nn, ctx->nflag);
  HH_TRY(hh_scan_u32(ctx, ctx->nflag, ctx->nflag, nn, &ctx->d_sc->n_leaves));
  k_leaf_compact<<<HH_N + cdiv(nn, 256), 256, 0, s>>>(ctx->nleft, ctx->nflag, nn, ctx->leaf_nodes);
  HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->n_leaves, &ctx->d_sc->n_leaves, sizeof(u32), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  ctx->n_leaves = (int)ctx->h_sc->n_leaves;
  // row 4: boxes, leaves then bottom-up
  k_leaf_boxes<<<HH_N + cdiv((int64_t)ctx->n_leaves * 32, 256), 256, 0, s>>>(ctx->Xs, ctx->leaf_nodes, ctx->n_leaves, ctx->nlo, ctx->nhi,
                                                                      ctx->bmin, ctx->bmax);
  for (int l = ctx->n_levels - 2; l >= 0; --l) {
    int c = ctx->lvl_start[l + 1] - ctx->lvl_start[l];
    k_merge_boxes<<<HH_N + cdiv(c, 256), 256, 0, s>>>(ctx->nleft, ctx->bmin, ctx->bmax, ctx->lvl_start[l], c);
  }
  HH_LAUNCH_CHECK();
  ctx->st.n_particles = N;
  ctx->st.n_nodes = ctx->n_nodes;
  ctx->st.n_leaves = ctx->n_leaves;
  ctx->st.depth = ctx->n_levels - 1;
  ctx->tree_ok = 1;
  return HH_OK;
}
