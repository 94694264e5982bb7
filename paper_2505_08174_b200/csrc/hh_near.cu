// hh_near.cu -- SURVEY 8(a) rows 6 and 8: inadmissible (near-field) blocks evaluated on the fly and never
// stored: U_i += sum_{j in sigma, j != i} M_ij F_j with M_ij from the two-body MLP
// (Eq. (4); S-1..S-5).  One CTA per target leaf walks that leaf's source leaves (P^H sorted by tau);
// the (target, source) pairs of a tile of sources are flattened over the threads so that ragged leaves
// waste no lanes; every thread evaluates two entries at a time (see hh_mlp.cuh).
#include "hh_mlp.cuh"

#define NR_T 256
#define NR_TILE 512

__global__ void __launch_bounds__(NR_T, 2) k_near(const float* __restrict__ gw, float a, const u32* __restrict__ leaf_nodes,
                                                const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                const uint2* __restrict__ PH, const u32* __restrict__ near_begin,
                                                const u32* __restrict__ near_end, const float* __restrict__ Xs,
                                                const float* __restrict__ Fs, float* __restrict__ Us) {
  __shared__ __align__(16) float sw[HH_MLP2_FLOATS];
  __shared__ float tX[HH_MAX_LEAF * 3], sU[HH_MAX_LEAF * 3];
  __shared__ float sXj[NR_TILE * 3], sFj[NR_TILE * 3];
  __shared__ u32 sJ[NR_TILE];
  __shared__ u32 segStart[33], segLo[32];
  __shared__ u32 s_nb;
  const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const u32 node = leaf_nodes[blockIdx.x];
  const u32 tlo = nlo[node], m = nhi[node] - tlo;
  load_weights(sw, gw, HH_MLP2_FLOATS);
  for (u32 t = tid; t < 3 * m; t += NR_T) { tX[t] = Xs[3 * (size_t)tlo + t]; sU[t] = 0.f; }
  u32 b = near_begin[node];
  const u32 bend = near_end[node];
  __syncthreads();
  while (b < bend) {
    if (warp == 0) {
      u32 blk = b + lane;
      u32 lo = 0, sz = 0;
      if (blk < bend) { u32 sg = PH[blk].y; lo = nlo[sg]; sz = nhi[sg] - lo; }
      u32 inc = sz;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { u32 t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (u32)o) inc += t; }
      bool fits = blk < bend && inc <= NR_TILE;
      u32 nb = __popc(__ballot_sync(0xffffffffu, fits));      // fits is a prefix property (sizes > 0)
      segStart[lane] = inc - sz;
      segLo[lane] = lo;
      if (lane == nb - 1) segStart[nb] = inc;
      if (lane == 0) s_nb = nb;
    }
    __syncthreads();
    const u32 nb = s_nb, nt = segStart[nb];
    for (u32 s = tid; s < nt; s += NR_T) {
      u32 g = 0;
      while (g + 1 < nb && segStart[g + 1] <= s) ++g;
      u32 j = segLo[g] + (s - segStart[g]);
      sJ[s] = j;
#pragma unroll
      for (int c = 0; c < 3; ++c) { sXj[3 * s + c] = Xs[3 * (size_t)j + c]; sFj[3 * s + c] = Fs[3 * (size_t)j + c]; }
    }
    __syncthreads();
    const u32 pairs = m * nt;
    for (u32 p0 = tid; p0 < pairs; p0 += 2 * NR_T) {
      u32 pp[2] = {p0, p0 + NR_T};
      bool ok[2] = {true, pp[1] < pairs};
      if (!ok[1]) pp[1] = p0;
      u32 ii[2], jj[2];
      float xi[2][3], xj[2][3], M[2][9];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        jj[e] = pp[e] / m; ii[e] = pp[e] - jj[e] * m;
#pragma unroll
        for (int c = 0; c < 3; ++c) { xi[e][c] = tX[3 * ii[e] + c]; xj[e][c] = sXj[3 * jj[e] + c]; }
      }
      entry2_eval<2>(sw, a, xi, xj, M);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (ok[e] && tlo + ii[e] != sJ[jj[e]]) {                         // S-5: the pair i == j is skipped
          const float f0 = sFj[3 * jj[e]], f1 = sFj[3 * jj[e] + 1], f2 = sFj[3 * jj[e] + 2];
#pragma unroll
          for (int al = 0; al < 3; ++al)
            atomicAdd(&sU[3 * ii[e] + al], fmaf(M[e][3 * al], f0, fmaf(M[e][3 * al + 1], f1, M[e][3 * al + 2] * f2)));
        }
      }
    }
    __syncthreads();
    b += nb;
  }
  for (u32 t = tid; t < 3 * m; t += NR_T) atomicAdd(&Us[3 * (size_t)tlo + t], sU[t]);
}

int hh_near_apply(hh_ctx* ctx) {
  if (ctx->n_leaves <= 0 || ctx->nH <= 0) return HH_OK;
  if (ctx->mlp2_wide) return hh_near_apply_wide(ctx);
  if (ctx->p.near_path != 0) return hh_near_apply_tc(ctx);
  k_near<<<HH_N + ctx->n_leaves, NR_T, 0, ctx->stream>>>(ctx->w2, ctx->p.radius_a, ctx->leaf_nodes, ctx->nlo, ctx->nhi, ctx->PH,
                                                  ctx->near_begin, ctx->near_end, ctx->Xs, ctx->Fs, ctx->Us);
  HH_LAUNCH_CHECK();
  return HH_OK;
}

// S-18b: admissible blocks on which Alg. 2 broke down (numerically singular pivot) are evaluated densely, exactly
// like the inadmissible ones (L252).  Each such block is cut into tiles of HH_MAX_LEAF rows x NR_TILE columns; the tiles
// of all blocks form one flat list (prefix over the blocks, binary search per CTA), so a 4096 x 4096 block spreads
// over the whole GPU instead of one SM.
__global__ void __launch_bounds__(256) k_dense_count(const u32* __restrict__ list, u32 n, const uint2* __restrict__ PG,
                                                      const u32* __restrict__ nlo, const u32* __restrict__ nhi, u32* __restrict__ cnt) {
  u32 t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const uint2 blk = PG[list[t]];
  const u32 m = nhi[blk.x] - nlo[blk.x], q = nhi[blk.y] - nlo[blk.y];
  cnt[t] = ((m + HH_MAX_LEAF - 1) / HH_MAX_LEAF) * ((q + NR_TILE - 1) / NR_TILE);
}

__global__ void __launch_bounds__(NR_T, 2) k_dense(const float* __restrict__ gw, float a, const u32* __restrict__ list, u32 n_list,
                                                    const u32* __restrict__ tile_prefix, const u32* __restrict__ total_tiles,
                                                    const uint2* __restrict__ PG, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                    const float* __restrict__ Xs, const float* __restrict__ Fs, float* __restrict__ Us) {
  __shared__ __align__(16) float sw[HH_MLP2_FLOATS];
  __shared__ float tX[HH_MAX_LEAF * 3], sU[HH_MAX_LEAF * 3];
  __shared__ float sXj[NR_TILE * 3], sFj[NR_TILE * 3];
  const u32 tid = threadIdx.x;
  load_weights(sw, gw, HH_MLP2_FLOATS);
  const u32 total = *total_tiles;
  for (u32 tile = blockIdx.x; tile < total; tile += gridDim.x) {
    u32 lo = 0, hi = n_list - 1;                                   // last block whose first tile is <= tile
    while (lo < hi) { u32 mid = (lo + hi + 1) / 2; if (tile_prefix[mid] <= tile) lo = mid; else hi = mid - 1; }
    const uint2 blk = PG[list[lo]];
    const u32 tlo = nlo[blk.x], m = nhi[blk.x] - tlo;
    const u32 slo = nlo[blk.y], n = nhi[blk.y] - slo;
    const u32 ct = (n + NR_TILE - 1) / NR_TILE, local = tile - tile_prefix[lo];
    const u32 r0 = (local / ct) * HH_MAX_LEAF, j0 = (local % ct) * NR_TILE;
    const u32 mt = min((u32)HH_MAX_LEAF, m - r0), nt = min((u32)NR_TILE, n - j0);
    __syncthreads();
    for (u32 t = tid; t < 3 * mt; t += NR_T) { tX[t] = Xs[3 * (size_t)(tlo + r0) + t]; sU[t] = 0.f; }
    for (u32 t = tid; t < 3 * nt; t += NR_T) { sXj[t] = Xs[3 * (size_t)(slo + j0) + t]; sFj[t] = Fs[3 * (size_t)(slo + j0) + t]; }
    __syncthreads();
    const u32 pairs = mt * nt;
    for (u32 p0 = tid; p0 < pairs; p0 += 2 * NR_T) {
      u32 pp[2] = {p0, p0 + NR_T};
      bool ok[2] = {true, pp[1] < pairs};
      if (!ok[1]) pp[1] = p0;
      u32 ii[2], jj[2];
      float xi[2][3], xj[2][3], M[2][9];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        jj[e] = pp[e] / mt; ii[e] = pp[e] - jj[e] * mt;
#pragma unroll
        for (int c = 0; c < 3; ++c) { xi[e][c] = tX[3 * ii[e] + c]; xj[e][c] = sXj[3 * jj[e] + c]; }
      }
      entry2_eval<2>(sw, a, xi, xj, M);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (ok[e] && tlo + r0 + ii[e] != slo + j0 + jj[e]) {
          const float f0 = sFj[3 * jj[e]], f1 = sFj[3 * jj[e] + 1], f2 = sFj[3 * jj[e] + 2];
#pragma unroll
          for (int al = 0; al < 3; ++al)
            atomicAdd(&sU[3 * ii[e] + al], fmaf(M[e][3 * al], f0, fmaf(M[e][3 * al + 1], f1, M[e][3 * al + 2] * f2)));
        }
      }
    }
    __syncthreads();
    for (u32 t = tid; t < 3 * mt; t += NR_T) atomicAdd(&Us[3 * (size_t)(tlo + r0) + t], sU[t]);
  }
}

int hh_dense_apply(hh_ctx* ctx) {
  if (ctx->res_next <= ctx->res_first || ctx->n_dense == 0) return HH_OK;
  const u32 n = ctx->n_dense;
  u32* cnt = ctx->dense_cnt;
  k_dense_count<<<HH_N + cdiv(n, 256), 256, 0, ctx->stream>>>(ctx->dense_list, n, ctx->PG, ctx->nlo, ctx->nhi, cnt);
  HH_TRY(hh_scan_u32(ctx, cnt, cnt, n, &ctx->d_sc->n_split));
  k_dense<<<HH_N + ctx->n_sm * 2, NR_T, 0, ctx->stream>>>(ctx->w2, ctx->p.radius_a, ctx->dense_list, n, cnt, &ctx->d_sc->n_split, ctx->PG,
                                                    ctx->nlo, ctx->nhi, ctx->Xs, ctx->Fs, ctx->Us);
  HH_LAUNCH_CHECK();
  return HH_OK;
}

// Two-body entries for explicit pairs (parity tests of the entry function).
__global__ void __launch_bounds__(128) k_entries(const float* __restrict__ gw, float a, const float* __restrict__ Xi,
                                                  const float* __restrict__ Xj, int64_t n, float* __restrict__ M) {
  __shared__ __align__(16) float sw[HH_MLP2_FLOATS];
  load_weights(sw, gw, HH_MLP2_FLOATS);
  __syncthreads();
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  float xi[1][3], xj[1][3], out[1][9];
#pragma unroll
  for (int c = 0; c < 3; ++c) { xi[0][c] = Xi[3 * t + c]; xj[0][c] = Xj[3 * t + c]; }
  entry2_eval<1>(sw, a, xi, xj, out);
#pragma unroll
  for (int r = 0; r < 9; ++r) M[9 * t + r] = out[0][r];
}

int hh_entries_eval(hh_ctx* ctx, const float* Xi, const float* Xj, int64_t n, float* M) {
  k_entries<<<HH_N + cdiv(n, 128), 128, 0, ctx->stream>>>(ctx->w2, ctx->p.radius_a, Xi, Xj, n, M);
  HH_LAUNCH_CHECK();
  return HH_OK;
}
