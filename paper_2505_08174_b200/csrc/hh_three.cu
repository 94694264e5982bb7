// hh_three.cu -- SURVEY 8(a) row 10: short-range three-body graph term (Eq. (4), faces L74;
// S-22, S-23):  U_i += R(MLP3([X_j-X_i, X_k-X_i, |X_j-X_k|])) F_j / (|X_j-X_k| |X_k-X_i|) for every ordered
// face (j,k,i), i != j, i,j in N(k) = { p != k : |X_p - X_k| < R_cut }.  Neighbour search: uniform cell list
// (cell side >= R_cut) built with the radix sort; one warp per centre k gathers N(k) with ballots, then its
// lanes take the d(d-1) faces.  The cutoff is an integer decision taken in fp32 in the fixed order
// ((dx*dx + dy*dy) + dz*dz) < rcut*rcut with individually rounded operations (S-22).
#include "hh_mlp.cuh"

#define TB_T 128
#define TB_CAP 256          /* neighbours kept per centre */

__device__ __forceinline__ float ord2f3(u32 o) { u32 u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o; return __uint_as_float(u); }

struct CellGrid { float lo[3]; float inv[3]; int nc[3]; };

__device__ __forceinline__ void cell_coords(const CellGrid& G, const float* x, int* c) {
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    int v = (int)floorf((x[d] - G.lo[d]) * G.inv[d]);
    c[d] = v < 0 ? 0 : (v >= G.nc[d] ? G.nc[d] - 1 : v);
  }
}

__global__ void __launch_bounds__(256) k_cell_ids(const float* __restrict__ Xs, int64_t N, CellGrid G, u64* __restrict__ keys,
                                                   u32* __restrict__ vals) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  float x[3] = {Xs[3 * k], Xs[3 * k + 1], Xs[3 * k + 2]};
  int c[3];
  cell_coords(G, x, c);
  keys[k] = (u64)(((int64_t)c[0] * G.nc[1] + c[1]) * G.nc[2] + c[2]);
  vals[k] = (u32)k;
}

// cell_start[c] = first sorted position whose cell id is >= c  (length ncells + 1)
__global__ void __launch_bounds__(256) k_cell_start(const u64* __restrict__ keys, int64_t N, u32 ncells, u32* __restrict__ cell_start) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p > N) return;
  u32 cprev = p == 0 ? 0u : (u32)keys[p - 1] + 1u;
  u32 ccur = p == N ? ncells : (u32)keys[p];
  for (u32 c = cprev; c <= ccur; ++c) cell_start[c] = (u32)p;
}

__device__ __forceinline__ bool within_cut(const float* A, const float* B, float rc2) {
  float dx = __fsub_rn(A[0], B[0]), dy = __fsub_rn(A[1], B[1]), dz = __fsub_rn(A[2], B[2]);
  float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
  return d2 < rc2;
}

// MODE 0: the transverse three-body term M^(t,3) (row 10).  MODE 1: the three-body SELF term M^(s,3) of Eq. (6) (L108-L113): the same
// faces, the self half of the 18-output network (packed as a second 9-output weight set), acting on F_i.  MODE 2: the two-body SELF
// term M^(s,2): U_k += [ sum_{j in N(k)} alpha_2^(s)(X_k, X_j) ] F_k, the self half of the 18-output two-body network on the same
// neighbour lists (Eq. (2); all three cut-off terms share R_cut, L56).
template <int MODE>
__global__ void __launch_bounds__(TB_T) k_three(const float* __restrict__ gw, float a, const float* __restrict__ Xs, const float* __restrict__ Fs,
                                                 float* __restrict__ Us, int64_t N, CellGrid G, const u32* __restrict__ cell_start,
                                                 const u32* __restrict__ order, float rcut, DevScalars* sc) {
  extern __shared__ __align__(16) float dyn[];
  float* sw = dyn;                                               // HH_MLP3_FLOATS (MODE 2: HH_MLP2_FLOATS used)
  u32* nbl = (u32*)(dyn + HH_MLP3_FLOATS);                       // [warps][TB_CAP]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  load_weights(sw, gw, MODE == 2 ? HH_MLP2_FLOATS : HH_MLP3_FLOATS);
  __syncthreads();
  const int64_t k = (int64_t)blockIdx.x * (TB_T / 32) + warp;
  if (k >= N) return;
  u32* nb = nbl + warp * TB_CAP;
  const float xk[3] = {Xs[3 * k], Xs[3 * k + 1], Xs[3 * k + 2]};
  const float rc2 = __fmul_rn(rcut, rcut);
  int ck[3];
  cell_coords(G, xk, ck);
  u32 d = 0;
  for (int dx = -1; dx <= 1; ++dx)
    for (int dy = -1; dy <= 1; ++dy) {
      int cx = ck[0] + dx, cy = ck[1] + dy;
      if (cx < 0 || cy < 0 || cx >= G.nc[0] || cy >= G.nc[1]) continue;
      int z0 = max(ck[2] - 1, 0), z1 = min(ck[2] + 1, G.nc[2] - 1);             // the z-run of cells is contiguous
      u32 c0 = (u32)(((int64_t)cx * G.nc[1] + cy) * G.nc[2] + z0), c1 = c0 + (u32)(z1 - z0);
      u32 pb = cell_start[c0], pe = cell_start[c1 + 1];
      for (u32 p0 = pb; p0 < pe; p0 += 32) {
        u32 p = p0 + lane;
        bool in = false;
        u32 q = 0;
        if (p < pe) {
          q = order[p];
          const float xq[3] = {Xs[3 * (size_t)q], Xs[3 * (size_t)q + 1], Xs[3 * (size_t)q + 2]};
          in = (int64_t)q != k && within_cut(xq, xk, rc2);
        }
        u32 bal = __ballot_sync(0xffffffffu, in);
        u32 pos = d + __popc(bal & ((1u << lane) - 1u));
        if (in && pos < TB_CAP) nb[pos] = q;
        d += __popc(bal);
      }
    }
  __syncwarp();
  if (d > TB_CAP) { if (lane == 0) atomicAdd(&sc->deg_overflow, 1u); return; }
  if (MODE == 2) {
    if (d < 1) return;
    if (lane == 0) atomicAdd((unsigned long long*)&sc->n_self_pairs, (unsigned long long)d);
    float S[9];
#pragma unroll
    for (int r = 0; r < 9; ++r) S[r] = 0.f;
    for (u32 f = lane; f < d; f += 32) {
      const u32 j = nb[f];
      float xi[1][3], xj[1][3], M[1][9];
#pragma unroll
      for (int c = 0; c < 3; ++c) { xi[0][c] = xk[c]; xj[0][c] = Xs[3 * (size_t)j + c]; }
      entry2_eval<1>(sw, a, xi, xj, M);
#pragma unroll
      for (int r = 0; r < 9; ++r) S[r] += M[0][r];
    }
#pragma unroll
    for (int r = 0; r < 9; ++r)
#pragma unroll
      for (int o = 16; o; o >>= 1) S[r] += __shfl_xor_sync(0xffffffffu, S[r], o);
    if (lane < 3) {
      const float f0 = Fs[3 * k], f1 = Fs[3 * k + 1], f2 = Fs[3 * k + 2];
      atomicAdd(&Us[3 * k + lane], fmaf(S[3 * lane], f0, fmaf(S[3 * lane + 1], f1, S[3 * lane + 2] * f2)));
    }
    return;
  }
  if (d < 2) return;
  const u32 nf = d * (d - 1);
  if (lane == 0 && MODE == 0) atomicAdd((unsigned long long*)&sc->n_faces, (unsigned long long)nf);
  for (u32 f = lane; f < nf; f += 32) {
    u32 a = f / (d - 1), b = f - a * (d - 1);
    if (b >= a) ++b;
    const u32 i = nb[a], j = nb[b];
    float x[1][HH_MLP3_INP], out[1][9];
    float djk = 0.f, dki = 0.f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float xi = Xs[3 * (size_t)i + c], xj = Xs[3 * (size_t)j + c];
      x[0][c] = xj - xi;
      x[0][3 + c] = xk[c] - xi;
      const float e = xj - xk[c];
      djk = fmaf(e, e, djk);
      dki = fmaf(x[0][3 + c], x[0][3 + c], dki);
    }
    djk = sqrtf(djk); dki = sqrtf(dki);
    x[0][6] = djk; x[0][7] = 0.f;
    mlp_eval<HH_MLP3_INP, HH_MLP3_H, 1>(sw, x, out);
    const float s = 1.0f / (djk * dki);
    const size_t jf = MODE == 1 ? (size_t)i : (size_t)j;           // the self half multiplies F_i, the transverse half F_j
    const float f0 = Fs[3 * jf], f1 = Fs[3 * jf + 1], f2 = Fs[3 * jf + 2];
#pragma unroll
    for (int al = 0; al < 3; ++al)
      atomicAdd(&Us[3 * (size_t)i + al], s * fmaf(out[0][3 * al], f0, fmaf(out[0][3 * al + 1], f1, out[0][3 * al + 2] * f2)));
  }
}

// modes: bit 0 transverse three-body (row 10), bit 1 three-body self term, bit 2 two-body self term
int hh_three_apply(hh_ctx* ctx, int modes) {
  if ((modes & 1) && !ctx->have_mlp3) return hh_fail(ctx, HH_ERR_INVALID_ARG, "three-body term needs a three-body MLP");
  if (!ctx->have_self3) modes &= ~2;
  if (!ctx->have_self2) modes &= ~4;
  if (!modes) return HH_OK;
  cudaStream_t s = ctx->stream;
  const int64_t N = ctx->N;
  const float rcut = ctx->p.rcut3;
  HH_CUDA(cudaMemcpyAsync(ctx->h_sc, ctx->d_sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  // bounding box of the cloud (left by hh_build_tree) -> cell grid with side >= rcut and at most n_cells_cap cells
  CellGrid G;
  double ext[3], cs = (double)rcut * 1.0001;
  for (int c = 0; c < 3; ++c) {
    u32 a = ctx->h_sc->bbu[c], b = ctx->h_sc->bbu[3 + c];
    u32 ua = (a & 0x80000000u) ? (a & 0x7fffffffu) : ~a, ub = (b & 0x80000000u) ? (b & 0x7fffffffu) : ~b;
    float lo, hi;
    memcpy(&lo, &ua, 4); memcpy(&hi, &ub, 4);
    G.lo[c] = lo;
    ext[c] = (double)hi - (double)lo;
  }
  for (;;) {
    double tot = 1.0;
    for (int c = 0; c < 3; ++c) {
      int64_t n = (int64_t)floor(ext[c] / cs) + 1;
      if (n < 1) n = 1;
      G.nc[c] = (int)(n > 2000000 ? 2000000 : n);
      tot *= (double)G.nc[c];
    }
    if (tot <= (double)ctx->n_cells_cap) break;
    cs *= 1.26;
  }
  for (int c = 0; c < 3; ++c) {
    double cw = ext[c] / (double)G.nc[c] * 1.000001;
    if (cw < cs) cw = cs;
    G.inv[c] = (float)(1.0 / cw);
  }
  const u32 ncells = (u32)((int64_t)G.nc[0] * G.nc[1] * G.nc[2]);
  if (modes & 1) HH_CUDA(cudaMemsetAsync(&ctx->d_sc->n_faces, 0, sizeof(u64), s));
  if (modes & 4) HH_CUDA(cudaMemsetAsync(&ctx->d_sc->n_self_pairs, 0, sizeof(u64), s));
  HH_CUDA(cudaMemsetAsync(&ctx->d_sc->deg_overflow, 0, sizeof(u32), s));
  k_cell_ids<<<HH_N + cdiv(N, 256), 256, 0, s>>>(ctx->Xs, N, G, ctx->keys[1], ctx->idx[1]);
  // sort (cell id, particle) with the radix ping-pong buffers; keys[0] (the Morton keys) must survive, so the
  // sort runs in scratch-free buffers: keys[1]/idx[1] and the cell_of / cell_order arrays as the second pair
  u64* k2[2] = {ctx->keys[1], (u64*)ctx->stageU};                // stageU (12 N bytes) holds N u64 keys
  u32* v2[2] = {ctx->idx[1], ctx->cell_of};
  int bits = 8;
  while (bits < 64 && ((u64)ncells >> bits)) bits += 8;
  int which = 0;
  HH_TRY(hh_sort_pairs(ctx, k2, v2, N, 0, bits, &which));
  k_cell_start<<<HH_N + cdiv(N + 1, 256), 256, 0, s>>>(k2[which], N, ncells, ctx->cell_start);
  size_t smem = (size_t)HH_MLP3_FLOATS * sizeof(float) + (TB_T / 32) * TB_CAP * sizeof(u32);
  if (!ctx->three_smem_set) {
    HH_CUDA(cudaFuncSetAttribute(k_three<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    HH_CUDA(cudaFuncSetAttribute(k_three<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    HH_CUDA(cudaFuncSetAttribute(k_three<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ctx->three_smem_set = 1;
  }
  const float a = ctx->p.radius_a;
  if (modes & 1) k_three<0><<<HH_N + cdiv(N, TB_T / 32), TB_T, smem, s>>>(ctx->w3, a, ctx->Xs, ctx->Fs, ctx->Us, N, G, ctx->cell_start, v2[which], rcut, ctx->d_sc);
  if (modes & 2) k_three<1><<<HH_N + cdiv(N, TB_T / 32), TB_T, smem, s>>>(ctx->w3s, a, ctx->Xs, ctx->Fs, ctx->Us, N, G, ctx->cell_start, v2[which], rcut, ctx->d_sc);
  if (modes & 4) k_three<2><<<HH_N + cdiv(N, TB_T / 32), TB_T, smem, s>>>(ctx->w2s, a, ctx->Xs, ctx->Fs, ctx->Us, N, G, ctx->cell_start, v2[which], rcut, ctx->d_sc);
  HH_LAUNCH_CHECK();
  HH_CUDA(cudaMemcpyAsync(ctx->h_sc, ctx->d_sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  if (modes & 1) ctx->st.n_faces = (int64_t)ctx->h_sc->n_faces;
  if (modes & 4) ctx->st.n_self_pairs = (int64_t)ctx->h_sc->n_self_pairs;
  if (ctx->h_sc->deg_overflow) return hh_fail(ctx, HH_ERR_UNSUPPORTED, "three-body: a particle has more than 256 neighbours within R_cut");
  return HH_OK;
}
