// hh_blocks.cu -- SURVEY 8(a) row 5: Alg. 1 BuildPartition as a level-synchronous,
// order-preserving frontier expansion; admissibility = Def. 2 / Eq. (7) on bounding boxes (L139-L148;
// S-14, S-15).  Afterwards P^G is ordered by block size (largest first; ACA size classes and arena
// batches are contiguous ranges of it) and P^H by target leaf (one near-field CTA per leaf).
#include "hh_internal.cuh"

#define BK_T 256

struct TreeView {
  const u32 *lo, *hi;
  const int* left;
  const float *bmin, *bmax;
};

// Eq. (7): max(diam^2) <= eta^2 dist^2 in fp64, summation order x,y,z, each operation individually
// rounded (no FMA contraction), so the decision is bit-identical to any IEEE fp64 evaluation in that order.
__device__ __forceinline__ bool admissible(const TreeView& tv, u32 t, u32 s, double eta2) {
  if (t == s) return false;                                               // S-15
  double da = 0.0, db = 0.0, dist = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double amin = (double)tv.bmin[3 * (size_t)t + c], amax = (double)tv.bmax[3 * (size_t)t + c];
    double bmn = (double)tv.bmin[3 * (size_t)s + c], bmx = (double)tv.bmax[3 * (size_t)s + c];
    double ea = __dsub_rn(amax, amin), eb = __dsub_rn(bmx, bmn);
    da = __dadd_rn(da, __dmul_rn(ea, ea));
    db = __dadd_rn(db, __dmul_rn(eb, eb));
    double g1 = __dsub_rn(amin, bmx), g2 = __dsub_rn(bmn, amax);
    double g = fmax(0.0, fmax(g1, g2));
    dist = __dadd_rn(dist, __dmul_rn(g, g));
  }
  return fmax(da, db) <= __dmul_rn(eta2, dist);
}

// 0: admissible, 1: inadmissible leaf pair, 2: split tau, 3: split sigma, 4: split both
__device__ __forceinline__ int classify(const TreeView& tv, uint2 p, double eta2) {
  if (admissible(tv, p.x, p.y, eta2)) return 0;
  bool tl = tv.left[p.x] < 0, sl = tv.left[p.y] < 0;
  if (tl && sl) return 1;
  if (sl) return 2;
  if (tl) return 3;
  return 4;
}

__global__ void __launch_bounds__(BK_T) k_bp_count(TreeView tv, const uint2* __restrict__ fr, int64_t n, double eta2,
                                                    Cnt3* __restrict__ tiles) {
  __shared__ u32 sm[33];
  int64_t i = (int64_t)blockIdx.x * BK_T + threadIdx.x;
  int code = i < n ? classify(tv, fr[i], eta2) : -1;
  u32 g = code == 0, h = code == 1, c = code >= 4 ? 4u : (code >= 2 ? 2u : 0u);
  u32 tg, th, tc;
  block_excl_scan<u32>(g, sm, &tg);
  block_excl_scan<u32>(h, sm, &th);
  block_excl_scan<u32>(c, sm, &tc);
  if (threadIdx.x == 0) tiles[blockIdx.x] = Cnt3{tg, th, tc};
}

__global__ void __launch_bounds__(BK_T) k_bp_fill(TreeView tv, const uint2* __restrict__ fr, int64_t n, double eta2,
                                                   const Cnt3* __restrict__ tiles, uint2* __restrict__ PG, uint2* __restrict__ PH,
                                                   uint2* __restrict__ next) {
  __shared__ u32 sm[33];
  int64_t i = (int64_t)blockIdx.x * BK_T + threadIdx.x;
  uint2 p = i < n ? fr[i] : make_uint2(0, 0);
  int code = i < n ? classify(tv, p, eta2) : -1;
  u32 g = code == 0, h = code == 1, c = code >= 4 ? 4u : (code >= 2 ? 2u : 0u);
  u32 tg, th, tc;
  u32 eg = block_excl_scan<u32>(g, sm, &tg);
  u32 eh = block_excl_scan<u32>(h, sm, &th);
  u32 ec = block_excl_scan<u32>(c, sm, &tc);
  Cnt3 base = tiles[blockIdx.x];
  if (code == 0) PG[base.g + eg] = p;
  else if (code == 1) PH[base.h + eh] = p;
  else if (code == 2) {
    int L = tv.left[p.x];
    next[base.c + ec] = make_uint2(L, p.y); next[base.c + ec + 1] = make_uint2(L + 1, p.y);
  } else if (code == 3) {
    int L = tv.left[p.y];
    next[base.c + ec] = make_uint2(p.x, L); next[base.c + ec + 1] = make_uint2(p.x, L + 1);
  } else if (code == 4) {
    int Lt = tv.left[p.x], Ls = tv.left[p.y];
    uint2* o = next + base.c + ec;
    o[0] = make_uint2(Lt, Ls); o[1] = make_uint2(Lt, Ls + 1); o[2] = make_uint2(Lt + 1, Ls); o[3] = make_uint2(Lt + 1, Ls + 1);
  }
}

__global__ void k_set_root_pair(uint2* fr) { fr[0] = make_uint2(0, 0); }

// ---- post-processing -------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_g_keys(const uint2* __restrict__ PG, int64_t n, const u32* __restrict__ nlo,
                                                 const u32* __restrict__ nhi, u64* __restrict__ keys, u32* __restrict__ vals) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  uint2 p = PG[k];
  u32 m = nhi[p.x] - nlo[p.x], q = nhi[p.y] - nlo[p.y];
  u32 mx = m > q ? m : q;
  keys[k] = (u64)(0xffffffffu - mx);          // ascending key = descending size; stable -> ties keep Alg. 1 order
  vals[k] = (u32)k;
}
__global__ void __launch_bounds__(256) k_h_keys(const uint2* __restrict__ PH, int64_t n, u64* __restrict__ keys, u32* __restrict__ vals) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  keys[k] = (u64)PH[k].x;
  vals[k] = (u32)k;
}
__global__ void __launch_bounds__(256) k_gather_pairs(const uint2* __restrict__ in, const u32* __restrict__ vals, int64_t n,
                                                       uint2* __restrict__ out) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) out[k] = in[vals[k]];
}

__device__ __forceinline__ u32 pad8(u32 v) { return (v + 7u) & ~7u; }

// per sorted admissible block: arena units per unit rank, class boundaries, counters
__global__ void __launch_bounds__(256) k_g_post(const uint2* __restrict__ PG, int64_t n, const u32* __restrict__ nlo,
                                                 const u32* __restrict__ nhi, u64* __restrict__ units, int* __restrict__ ranks,
                                                 int* __restrict__ flags, DevScalars* sc) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  u64 rc = 0;
  if (k < n) {
    uint2 p = PG[k];
    u32 m = nhi[p.x] - nlo[p.x], q = nhi[p.y] - nlo[p.y];
    units[k] = (u64)(pad8(m) + pad8(q));
    ranks[k] = -1;
    flags[k] = 0;
    rc = (u64)m + q;
    u32 mx = m > q ? m : q;
    u32 pmx = 0xffffffffu;
    if (k > 0) { uint2 pp = PG[k - 1]; u32 a = nhi[pp.x] - nlo[pp.x], b = nhi[pp.y] - nlo[pp.y]; pmx = a > b ? a : b; }
    const u32 th[4] = {256u, 128u, 64u, HH_FAR_MID_MAX};          // [3]: first block of the far-field apply's mid-size class (hh_far.cu)
#pragma unroll
    for (int c = 0; c < 4; ++c) if (mx <= th[c] && pmx > th[c]) sc->class_bound[c] = (u32)k;
  }
  for (int o = 16; o; o >>= 1) rc += __shfl_xor_sync(0xffffffffu, rc, o);
  if ((threadIdx.x & 31) == 0 && rc) atomicAdd((unsigned long long*)&sc->far_rows_cols, (unsigned long long)rc);
}

__global__ void __launch_bounds__(256) k_h_post(const uint2* __restrict__ PH, int64_t n, const u32* __restrict__ nlo,
                                                 const u32* __restrict__ nhi, u32* __restrict__ near_begin, u32* __restrict__ near_end,
                                                 DevScalars* sc) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  u64 w = 0;
  if (k < n) {
    uint2 p = PH[k];
    w = (u64)(nhi[p.x] - nlo[p.x]) * (u64)(nhi[p.y] - nlo[p.y]);
    if (k == 0 || PH[k - 1].x != p.x) near_begin[p.x] = (u32)k;
    if (k == n - 1 || PH[k + 1].x != p.x) near_end[p.x] = (u32)k + 1;
  }
  for (int o = 16; o; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
  if ((threadIdx.x & 31) == 0 && w) atomicAdd((unsigned long long*)&sc->near_entries, (unsigned long long)w);
}

__global__ void k_blocks_init(DevScalars* sc, u32 nG) {
  sc->class_bound[0] = sc->class_bound[1] = sc->class_bound[2] = sc->class_bound[3] = nG;
  sc->near_entries = 0; sc->far_rows_cols = 0;
}

static int bits_for(u64 maxval) { int b = 8; while (b < 64 && (maxval >> b)) b += 8; return b; }

int hh_blocks_build(hh_ctx* ctx) {
  if (!ctx->tree_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_build_blocks before hh_build_tree");
  cudaStream_t s = ctx->stream;
  ctx->blocks_ok = 0;
  ctx->res_first = ctx->res_next = 0;
  TreeView tv{ctx->nlo, ctx->nhi, ctx->nleft, ctx->bmin, ctx->bmax};
  const double eta2 = (double)ctx->p.eta * (double)ctx->p.eta;
  // frontier ping-pong lives in the scratch (== arena) region
  int64_t fcap = (int64_t)(ctx->scratch_bytes / 2 / sizeof(uint2));
  uint2* fr[2] = {(uint2*)ctx->scratch, (uint2*)ctx->scratch + fcap};
  Cnt3* tiles = (Cnt3*)ctx->tilesum;
  k_set_root_pair<<<HH_N + 1, 1, 0, s>>>(fr[0]);
  int64_t n = 1, nG = 0, nH = 0;
  int cur = 0;
  while (n > 0) {
    int64_t nt = (n + BK_T - 1) / BK_T;
    k_bp_count<<<HH_N + (unsigned)nt, BK_T, 0, s>>>(tv, fr[cur], n, eta2, tiles);
    HH_TRY(hh_scan_cnt3(ctx, tiles, nt, &ctx->d_sc->lvl));
    HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->lvl, &ctx->d_sc->lvl, sizeof(Cnt3), cudaMemcpyDeviceToHost, s));
    HH_CUDA(cudaStreamSynchronize(s));
    Cnt3 t = ctx->h_sc->lvl;
    if (nG + t.g > ctx->cap_pairs || nH + t.h > ctx->cap_pairs || (int64_t)t.c > fcap) {
      int64_t need = nG + t.g > nH + t.h ? nG + t.g : nH + t.h;
      if ((int64_t)t.c > need) need = t.c;
      ctx->st.workspace_required = (int64_t)ctx->ws_bytes + need * 64;
      return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "block lists / frontier exceed the pair capacity (raise pairs_per_particle or the workspace)");
    }
    k_bp_fill<<<HH_N + (unsigned)nt, BK_T, 0, s>>>(tv, fr[cur], n, eta2, tiles, ctx->PG + nG, ctx->PH + nH, fr[cur ^ 1]);
    HH_LAUNCH_CHECK();
    nG += t.g; nH += t.h; n = t.c; cur ^= 1;
  }
  ctx->nG = nG; ctx->nH = nH;
  k_blocks_init<<<HH_N + 1, 1, 0, s>>>(ctx->d_sc, (u32)nG);
  // sort buffers carved from the scratch region
  int64_t nmax = nG > nH ? nG : nH;
  size_t need = (size_t)nmax * (2 * sizeof(u64) + 2 * sizeof(u32) + sizeof(uint2)) + 1024;
  if (need > ctx->scratch_bytes) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "scratch too small for block-list sort");
  u64* k2[2] = {(u64*)ctx->scratch, (u64*)ctx->scratch + nmax};
  u32* v2[2] = {(u32*)(k2[1] + nmax), (u32*)(k2[1] + nmax) + nmax};
  uint2* tmp = (uint2*)(((uintptr_t)(v2[1] + nmax) + 15) & ~(uintptr_t)15);
  int which;
  if (nG > 0) {
    k_g_keys<<<HH_N + cdiv(nG, 256), 256, 0, s>>>(ctx->PG, nG, ctx->nlo, ctx->nhi, k2[0], v2[0]);
    HH_TRY(hh_sort_pairs(ctx, k2, v2, nG, 0, 32, &which));
    k_gather_pairs<<<HH_N + cdiv(nG, 256), 256, 0, s>>>(ctx->PG, v2[which], nG, tmp);
    HH_CUDA(cudaMemcpyAsync(ctx->PG, tmp, (size_t)nG * sizeof(uint2), cudaMemcpyDeviceToDevice, s));
    k_g_post<<<HH_N + cdiv(nG, 256), 256, 0, s>>>(ctx->PG, nG, ctx->nlo, ctx->nhi, ctx->unit_prefix, ctx->ranks, ctx->flags, ctx->d_sc);
    HH_TRY(hh_scan_u64(ctx, ctx->unit_prefix, ctx->unit_prefix, nG + 1, nullptr));
  }
  if (nH > 0) {
    HH_CUDA(cudaMemsetAsync(ctx->near_begin, 0, sizeof(u32) * ctx->n_nodes, s));
    HH_CUDA(cudaMemsetAsync(ctx->near_end, 0, sizeof(u32) * ctx->n_nodes, s));
    k_h_keys<<<HH_N + cdiv(nH, 256), 256, 0, s>>>(ctx->PH, nH, k2[0], v2[0]);
    HH_TRY(hh_sort_pairs(ctx, k2, v2, nH, 0, bits_for((u64)ctx->n_nodes), &which));
    k_gather_pairs<<<HH_N + cdiv(nH, 256), 256, 0, s>>>(ctx->PH, v2[which], nH, tmp);
    HH_CUDA(cudaMemcpyAsync(ctx->PH, tmp, (size_t)nH * sizeof(uint2), cudaMemcpyDeviceToDevice, s));
    k_h_post<<<HH_N + cdiv(nH, 256), 256, 0, s>>>(ctx->PH, nH, ctx->nlo, ctx->nhi, ctx->near_begin, ctx->near_end, ctx->d_sc);
  }
  HH_LAUNCH_CHECK();
  HH_CUDA(cudaMemcpyAsync(ctx->h_sc, ctx->d_sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  ctx->class_bound[0] = 0;
  for (int c = 0; c < 3; ++c) ctx->class_bound[c + 1] = ctx->h_sc->class_bound[c];
  ctx->class_bound[4] = (u32)nG;
  ctx->mid_bound = ctx->h_sc->class_bound[3] < ctx->h_sc->class_bound[0] ? ctx->h_sc->class_bound[3] : ctx->h_sc->class_bound[0];   // <= first block of class 1
  // boundaries are "first index with size <= threshold"; a class that never starts keeps nG, and a
  // later class may start earlier only if sizes skip a class entirely -> make monotone
  for (int c = 3; c >= 1; --c) if (ctx->class_bound[c] > ctx->class_bound[c + 1]) ctx->class_bound[c] = ctx->class_bound[c + 1];
  ctx->st.n_admissible = nG;
  ctx->st.n_inadmissible = nH;
  ctx->st.near_entries = (int64_t)ctx->h_sc->near_entries;
  ctx->st.far_rows_cols = (int64_t)ctx->h_sc->far_rows_cols;
  ctx->st.sum_rank = ctx->st.aca_entries = ctx->st.factor_bytes = ctx->st.aca_batches = 0;
  ctx->st.aca_not_converged = ctx->st.aca_singular = 0;
  ctx->blocks_ok = 1;
  return HH_OK;
}
