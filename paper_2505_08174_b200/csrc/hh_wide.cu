// hh_wide.cu -- kernels around the paper-size MLP tile of hh_wide.cuh: near-field apply,
// entry evaluation for the lock-step ACA (the paper's own structure, L262: gather coordinates -> network inference -> scatter
// into C / Q; here the "inference" is the tensor-core tile and the scatter goes straight into the rank-k slot of the arena),
// and explicit pairs for the entry test.
#include <string.h>
#include "hh_wide.cuh"

#define WN_T WD_T            /* 256 threads: two warpgroups per 128-entry tile */
#define WN_TILE 256

struct WideNearSmem {
  WideSmem W;
  float tX[HH_MAX_LEAF * 3], sU[HH_MAX_LEAF * 3];
  float sXj[WN_TILE * 3], sFj[WN_TILE * 3];
  u32 sJ[WN_TILE];
  u32 segStart[33], segLo[32];
  u32 s_nb;
};

__device__ __forceinline__ void wide_features(const float* xi, const float* xj, float a, float (&x)[4], float& inv) {
  const float rx = xj[0] - xi[0], ry = xj[1] - xi[1], rz = xj[2] - xi[2];
  float d = sqrtf(fmaf(rx, rx, fmaf(ry, ry, rz * rz)));
  d = fmaxf(d, 1e-12f * a);
  inv = 1.0f / d;
  x[0] = rx * inv; x[1] = ry * inv; x[2] = rz * inv; x[3] = a * inv;
}

// rows 6, 8 with the paper-size MLP: one CTA per target leaf, 128 (target, source) pairs per tile (the loop of k_near_tc)
__global__ void __launch_bounds__(WN_T) k_near_wide(const float* __restrict__ gw, float a, const u32* __restrict__ leaf_nodes,
                                                     const u32* __restrict__ nlo, const u32* __restrict__ nhi, const uint2* __restrict__ PH,
                                                     const u32* __restrict__ near_begin, const u32* __restrict__ near_end,
                                                     const float* __restrict__ Xs, const float* __restrict__ Fs, float* __restrict__ Us,
                                                     u32* __restrict__ err_flag) {
  extern __shared__ __align__(1024) unsigned char wn_raw[];
  WideNearSmem& S = *reinterpret_cast<WideNearSmem*>(wn_raw);
  const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const u32 node = leaf_nodes[blockIdx.x];
  const u32 tlo = nlo[node], m = nhi[node] - tlo;
  wide_setup(S.W, gw);
  for (u32 t = tid; t < 3 * m; t += WN_T) { S.tX[t] = Xs[3 * (size_t)tlo + t]; S.sU[t] = 0.f; }
  bool alive = true;
  u32 b = near_begin[node];
  const u32 bend = near_end[node];
  while (b < bend) {
    __syncthreads();
    if (warp == 0) {
      u32 blk = b + lane;
      u32 lo = 0, sz = 0;
      if (blk < bend) { u32 sg = PH[blk].y; lo = nlo[sg]; sz = nhi[sg] - lo; }
      u32 inc = sz;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { u32 t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (u32)o) inc += t; }
      bool fits = blk < bend && inc <= WN_TILE;
      u32 nb = __popc(__ballot_sync(0xffffffffu, fits));
      S.segStart[lane] = inc - sz;
      S.segLo[lane] = lo;
      if (lane == nb - 1) S.segStart[nb] = inc;
      if (lane == 0) S.s_nb = nb;
    }
    __syncthreads();
    const u32 nb = S.s_nb, nt = S.segStart[nb];
    for (u32 s = tid; s < nt; s += WN_T) {
      u32 g = 0;
      while (g + 1 < nb && S.segStart[g + 1] <= s) ++g;
      u32 j = S.segLo[g] + (s - S.segStart[g]);
      S.sJ[s] = j;
#pragma unroll
      for (int c = 0; c < 3; ++c) { S.sXj[3 * s + c] = Xs[3 * (size_t)j + c]; S.sFj[3 * s + c] = Fs[3 * (size_t)j + c]; }
    }
    __syncthreads();
    const u32 pairs = m * nt;
    for (u32 p0 = 0; p0 < pairs; p0 += 128) {
      const u32 p = p0 + (tid & 127u);
      const bool valid = p < pairs && tid < 128u;                            // the result lives in the first warpgroup
      const u32 pc = p < pairs ? p : 0u;
      const u32 jj = pc / m, ii = pc - jj * m;
      float x[4], inv, out[9];
      wide_features(&S.tX[3 * ii], &S.sXj[3 * jj], a, x, inv);
      alive = wide_tile(S.W, gw, x, out) && alive;
      if (valid && tlo + ii != S.sJ[jj]) {                                   // S-5
        const float f0 = S.sFj[3 * jj], f1 = S.sFj[3 * jj + 1], f2 = S.sFj[3 * jj + 2];
#pragma unroll
        for (int al = 0; al < 3; ++al)
          atomicAdd(&S.sU[3 * ii + al], inv * fmaf(out[3 * al], f0, fmaf(out[3 * al + 1], f1, out[3 * al + 2] * f2)));
      }
    }
    b += nb;
  }
  __syncthreads();
  for (u32 t = tid; t < 3 * m; t += WN_T) atomicAdd(&Us[3 * (size_t)tlo + t], S.sU[t]);
  if (!alive && tid == 0) atomicExch(err_flag, 1u);
  wide_teardown(S.W);
}

// explicit pairs (hh_eval_entries)
__global__ void __launch_bounds__(WN_T) k_entries_wide(const float* __restrict__ gw, float a, const float* __restrict__ Xi, const float* __restrict__ Xj,
                                                        int64_t n, float* __restrict__ M, u32* __restrict__ err_flag) {
  extern __shared__ __align__(1024) unsigned char wn_raw[];
  WideSmem& S = *reinterpret_cast<WideSmem*>(wn_raw);
  wide_setup(S, gw);
  bool alive = true;
  for (int64_t t0 = (int64_t)blockIdx.x * 128; t0 < n; t0 += (int64_t)gridDim.x * 128) {
    const int64_t t = t0 + (threadIdx.x & 127);
    const int64_t tc = t < n ? t : n - 1;
    float xi[3], xj[3], x[4], inv, out[9];
#pragma unroll
    for (int c = 0; c < 3; ++c) { xi[c] = Xi[3 * tc + c]; xj[c] = Xj[3 * tc + c]; }
    wide_features(xi, xj, a, x, inv);
    alive = wide_tile(S, gw, x, out) && alive;
    if (t < n && threadIdx.x < 128) {
#pragma unroll
      for (int r = 0; r < 9; ++r) M[9 * t + r] = out[r] * inv;
    }
  }
  if (!alive && threadIdx.x == 0) atomicExch(err_flag, 1u);
  wide_teardown(S);
}

// ------------------------------------------------------------------------------ host side
// Pack a 4 -> 128 -> 512 -> 128 -> 9 MLP (hh_mlp: W[l] row-major [out][in], DEVICE pointers) into the layout of hh_wide.cuh:
// W1, b1, b2, b3, W4T, b4 as they are; W2 and W3 rounded to tf32 (cvt.rna) and cut into the 8 chunks of the tile, each chunk
// in the K-major core-matrix layout its TMA bulk copy drops into shared memory.  `out` receives WD_TOTAL floats.
int hh_pack_wide(hh_ctx* ctx, const hh_mlp* m, float* out) {
  if (m->n_layers != 4 || !m->dims || !m->W || !m->b) return HH_ERR_UNSUPPORTED;
  const int want[5] = {WD_IN, WD_H1, WD_H2, WD_H3, 9};
  for (int l = 0; l < 5; ++l) if (m->dims[l] != want[l]) return HH_ERR_UNSUPPORTED;
  size_t wn[4] = {(size_t)WD_H1 * WD_IN, (size_t)WD_H2 * WD_H1, (size_t)WD_H3 * WD_H2, (size_t)9 * WD_H3};
  size_t bn[4] = {WD_H1, WD_H2, WD_H3, 9};
  float* W[4]; float* B[4];
  for (int l = 0; l < 4; ++l) {
    if (!m->W[l] || !m->b[l]) return HH_ERR_INVALID_ARG;
    W[l] = (float*)malloc(wn[l] * sizeof(float)); B[l] = (float*)malloc(bn[l] * sizeof(float));
    if (!W[l] || !B[l]) return HH_ERR_INVALID_ARG;
    HH_CUDA(cudaMemcpyAsync(W[l], m->W[l], wn[l] * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
    HH_CUDA(cudaMemcpyAsync(B[l], m->b[l], bn[l] * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
  }
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  auto rna = [](float v) { u32 b; memcpy(&b, &v, 4); b = (b + 0x1000u) & 0xffffe000u; float r; memcpy(&r, &b, 4); return r; };
  memset(out, 0, sizeof(float) * WD_TOTAL);
  memcpy(out + WD_OFF_W1, W[0], wn[0] * sizeof(float));
  memcpy(out + WD_OFF_B1, B[0], bn[0] * sizeof(float));
  memcpy(out + WD_OFF_B2, B[1], bn[1] * sizeof(float));
  memcpy(out + WD_OFF_B3, B[2], bn[2] * sizeof(float));
  for (int h = 0; h < WD_H3; ++h) for (int r = 0; r < 9; ++r) out[WD_OFF_W4 + h * 12 + r] = W[3][(size_t)r * WD_H3 + h];
  memcpy(out + WD_OFF_B4, B[3], 9 * sizeof(float));
  for (int n = 0; n < WD_H2; ++n)                                 // W2 [512][128]: chunk c = n / 64, row nn = n % 64
    for (int k = 0; k < WD_H1; ++k) {
      const int c = n / WD_NC, nn = n % WD_NC;
      out[WD_OFF_W2 + (size_t)c * WD_NC * WD_H1 + (nn / 8) * 1024 + (k / 4) * 32 + (nn % 8) * 4 + (k % 4)] = rna(W[1][(size_t)n * WD_H1 + k]);
    }
  for (int n = 0; n < WD_H3; ++n)                                 // W3 [128][512]: K-chunk c = k / 64, kk = k % 64
    for (int k = 0; k < WD_H2; ++k) {
      const int c = k / WD_NC, kk = k % WD_NC;
      out[WD_OFF_W3 + (size_t)c * WD_H3 * WD_NC + (n / 8) * 512 + (kk / 4) * 32 + (n % 8) * 4 + (kk % 4)] = rna(W[2][(size_t)n * WD_H2 + k]);
    }
  for (int l = 0; l < 4; ++l) { free(W[l]); free(B[l]); }
  return HH_OK;
}
size_t hh_wide_floats(void) { return WD_TOTAL; }

static int wide_check(hh_ctx* ctx, const char* what) {
  HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->deg_overflow, &ctx->d_sc->deg_overflow, sizeof(u32), cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  if (ctx->h_sc->deg_overflow) return hh_fail(ctx, HH_ERR_CUDA, what);
  return HH_OK;
}

int hh_near_apply_wide(hh_ctx* ctx) {
  if (ctx->n_leaves <= 0 || ctx->nH <= 0) return HH_OK;
  const size_t smem = sizeof(WideNearSmem) + 1024;
  HH_CUDA(cudaFuncSetAttribute(k_near_wide, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  HH_CUDA(cudaMemsetAsync(&ctx->d_sc->deg_overflow, 0, sizeof(u32), ctx->stream));
  k_near_wide<<<HH_N + ctx->n_leaves, WN_T, smem, ctx->stream>>>(ctx->w2w, ctx->p.radius_a, ctx->leaf_nodes, ctx->nlo, ctx->nhi, ctx->PH, ctx->near_begin,
                                                                 ctx->near_end, ctx->Xs, ctx->Fs, ctx->Us, &ctx->d_sc->deg_overflow);
  HH_LAUNCH_CHECK();
  return wide_check(ctx, "paper-size MLP near-field: an mbarrier wait timed out (MMA or TMA never completed)");
}

int hh_entries_eval_wide(hh_ctx* ctx, const float* Xi, const float* Xj, int64_t n, float* M) {
  const size_t smem = sizeof(WideSmem) + 1024;
  HH_CUDA(cudaFuncSetAttribute(k_entries_wide, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  HH_CUDA(cudaMemsetAsync(&ctx->d_sc->deg_overflow, 0, sizeof(u32), ctx->stream));
  const unsigned tiles = cdiv(n, 128);
  k_entries_wide<<<HH_N + (tiles < (unsigned)ctx->n_sm ? tiles : (unsigned)ctx->n_sm), WN_T, smem, ctx->stream>>>(ctx->w2w, ctx->p.radius_a, Xi, Xj, n, M,
                                                                                                                   &ctx->d_sc->deg_overflow);
  HH_LAUNCH_CHECK();
  return wide_check(ctx, "paper-size MLP entries: an mbarrier wait timed out");
}
