// hh_api.cu -- the C ABI of include/hh.h: context, workspace carving, stage drivers, introspection.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include <vector>
#include "hh_internal.cuh"

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Carver {
  char* base; size_t off, cap; bool ok;
  template <typename T> T* take(size_t count) {
    off = align_up(off, 256);
    T* p = (T*)(base + off);
    off += count * sizeof(T);
    if (off > cap) ok = false;
    return p;
  }
};

// Fixed (per-N) arrays first, the rest of the workspace is the scratch / factor arena.
static int carve(hh_ctx* ctx, int64_t N) {
  // every carved pointer changes below: whatever was built for the previous layout is gone, also when this fails
  ctx->tree_ok = ctx->blocks_ok = 0;
  ctx->res_first = ctx->res_next = 0;
  ctx->n_dense = 0;
  ctx->N = 0;
  ctx->far_items = nullptr; ctx->far_cnt = nullptr; ctx->far_items_cap = 0; ctx->far_built = 0;
  Carver c{ctx->ws, 0, ctx->ws_bytes, true};
  ctx->Ncap = N;
  ctx->cap_pairs = ctx->pairs_per_particle * N + 4096;
  size_t nodes = (size_t)2 * N + 2;
  ctx->d_sc = c.take<DevScalars>(1);
  ctx->w2 = c.take<float>(HH_MLP2_FLOATS);
  ctx->w3 = c.take<float>(HH_MLP3_FLOATS);
  ctx->w2s = c.take<float>(HH_MLP2_FLOATS);
  ctx->w3s = c.take<float>(HH_MLP3_FLOATS);
  ctx->w2d = c.take<double>(HH_MLP2_FLOATS);
  ctx->w2tc = c.take<float>(2 * 1024);
  ctx->w2w = c.take<float>(hh_wide_floats());
  for (int k = 0; k < 2; ++k) { ctx->keys[k] = c.take<u64>(N); ctx->idx[k] = c.take<u32>(N); }
  ctx->hist_cap = (size_t)((ctx->cap_pairs > N ? ctx->cap_pairs : N) / 8 + 8192);
  ctx->hist = c.take<u32>(ctx->hist_cap);
  ctx->tilesum = c.take<char>(ctx->ws_bytes / 256 + 65536);
  ctx->Xs = c.take<float>(3 * N); ctx->Fs = c.take<float>(3 * N); ctx->Us = c.take<float>(3 * N);
  ctx->perm = c.take<u32>(N);
  ctx->nlo = c.take<u32>(nodes); ctx->nhi = c.take<u32>(nodes);
  ctx->nleft = c.take<int>(nodes); ctx->nparent = c.take<int>(nodes); ctx->nlevel = c.take<int>(nodes);
  ctx->nsplit = c.take<u32>(nodes); ctx->nflag = c.take<u32>(nodes);
  ctx->bmin = c.take<float>(3 * nodes); ctx->bmax = c.take<float>(3 * nodes);
  ctx->leaf_nodes = c.take<u32>(nodes);
  ctx->near_begin = c.take<u32>(nodes); ctx->near_end = c.take<u32>(nodes);
  ctx->PG = c.take<uint2>(ctx->cap_pairs); ctx->PH = c.take<uint2>(ctx->cap_pairs);
  ctx->ranks = c.take<int>(ctx->cap_pairs); ctx->flags = c.take<int>(ctx->cap_pairs);
  ctx->dense_list = c.take<u32>(ctx->cap_pairs); ctx->dense_cnt = c.take<u32>(ctx->cap_pairs + 1);
  ctx->unit_prefix = c.take<u64>(ctx->cap_pairs + 1);
  ctx->n_cells_cap = 4 * N + 4096;
  ctx->cell_of = c.take<u32>(N); ctx->cell_order = c.take<u32>(N); ctx->cell_start = c.take<u32>(ctx->n_cells_cap + 1);
  ctx->stageX = c.take<float>(3 * N); ctx->stageF = c.take<float>(3 * N); ctx->stageU = c.take<float>(3 * N);
  c.off = align_up(c.off, 4096);
  size_t min_scratch = (size_t)64 << 20;
  ctx->st.workspace_required = (int64_t)(c.off + min_scratch);
  if (!c.ok || c.off + min_scratch > ctx->ws_bytes) {
    ctx->Ncap = 0;
    return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "workspace too small for the per-particle arrays (see hh_stats.workspace_required)");
  }
  ctx->scratch = ctx->ws + c.off;
  ctx->scratch_bytes = ctx->ws_bytes - c.off;
  ctx->st.arena_bytes = (int64_t)ctx->scratch_bytes;
  return HH_OK;
}

static int check_params(const hh_params* p) {
  if (!p) return 0;
  if (p->leaf_size < 1 || p->leaf_size > HH_MAX_LEAF) return 0;
  if (!(p->eta > 0.f) || !isfinite(p->eta)) return 0;
  if (!(p->aca_tol > 0.f) || !isfinite(p->aca_tol)) return 0;
  if (p->aca_max_rank < 1 || p->aca_max_rank > HH_MAX_RANK) return 0;
  if (!(p->radius_a > 0.f) || !isfinite(p->radius_a)) return 0;
  if (!(p->rcut3 >= 0.f) || !isfinite(p->rcut3)) return 0;
  if (p->pivot_rule != 0 && p->pivot_rule != 1) return 0;
  if (p->near_path < 0 || p->near_path > 2) return 0;
  if (!(p->kappa_max >= 0.f)) return 0;
  if (!(p->dense_cap >= 0.f)) return 0;
  if (p->aca_precision != 0 && p->aca_precision != 1) return 0;                           /* 0 = default, INFINITY allowed, NaN / negative not */
  return 1;
}

// copy an MLP to the host and pack it as MlpOff<INP,H> describes (input dim zero-padded to INP)
// An 18-output network emits [alpha^(s), alpha^(t)] (Eq. (2)): `out` receives the transverse half (outputs 9..17, what the
// H-matrix and the transverse three-body term use), `out_self` the self half (outputs 0..8) as a second 9-output weight set.
static int pack_mlp(hh_ctx* ctx, const hh_mlp* m, int in, int INP, int H, std::vector<float>& out, std::vector<float>* out_self = nullptr) {
  if (m->n_layers != 3 || !m->dims || !m->W || !m->b) return HH_ERR_UNSUPPORTED;
  if (m->dims[0] != in || m->dims[1] != H || m->dims[2] != H || (m->dims[3] != 9 && m->dims[3] != 18)) return HH_ERR_UNSUPPORTED;
  const int nout = m->dims[3], off = nout == 18 ? 9 : 0;
  std::vector<float> W1((size_t)H * in), b1(H), W2((size_t)H * H), b2(H), W3((size_t)nout * H), b3(nout);
  float* dst[6] = {W1.data(), b1.data(), W2.data(), b2.data(), W3.data(), b3.data()};
  const float* src[6] = {m->W[0], m->b[0], m->W[1], m->b[1], m->W[2], m->b[2]};
  size_t cnt[6] = {W1.size(), b1.size(), W2.size(), b2.size(), W3.size(), b3.size()};
  for (int k = 0; k < 6; ++k) {
    if (!src[k]) return HH_ERR_INVALID_ARG;
    HH_CUDA(cudaMemcpyAsync(dst[k], src[k], cnt[k] * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
  }
  HH_CUDA(cudaStreamSynchronize(ctx->stream));                    // the weights must be ready on ctx->stream
  out.assign((size_t)HH_MLP_FLOATS(INP, H), 0.f);
  size_t o = 0;
  for (int r = 0; r < H; ++r) for (int c = 0; c < in; ++c) out[o + (size_t)r * INP + c] = W1[(size_t)r * in + c];
  o += (size_t)H * INP;
  for (int r = 0; r < H; ++r) out[o + r] = b1[r];
  o += H;
  for (size_t t = 0; t < W2.size(); ++t) out[o + t] = W2[t];
  o += (size_t)H * H;
  for (int r = 0; r < H; ++r) out[o + r] = b2[r];
  o += H;
  if (out_self) { out_self->clear(); if (nout == 18) *out_self = out; }
  for (int h = 0; h < H; ++h) for (int r = 0; r < 9; ++r) out[o + (size_t)h * 12 + r] = W3[(size_t)(off + r) * H + h];
  if (out_self && nout == 18)
    for (int h = 0; h < H; ++h) for (int r = 0; r < 9; ++r) (*out_self)[o + (size_t)h * 12 + r] = W3[(size_t)r * H + h];
  o += (size_t)H * 12;
  for (int r = 0; r < 9; ++r) out[o + r] = b3[off + r];
  if (out_self && nout == 18) for (int r = 0; r < 9; ++r) (*out_self)[o + r] = b3[r];
  return HH_OK;
}

// ------------------------------------------------------------------------------ small kernels
__global__ void __launch_bounds__(256) k_gather_f(const float* __restrict__ F, const u32* __restrict__ perm, int64_t N,
                                                   float* __restrict__ Fs, float* __restrict__ Us) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  size_t p = perm[k];
#pragma unroll
  for (int c = 0; c < 3; ++c) { Fs[3 * k + c] = F[3 * p + c]; Us[3 * k + c] = 0.f; }
}
// row 11: self term alpha_1 = I (S-5) and scatter back to the caller's order
__global__ void __launch_bounds__(256) k_unpermute(const float* __restrict__ Us, const float* __restrict__ Fs,
                                                    const u32* __restrict__ perm, int64_t N, int self, int accumulate,
                                                    float* __restrict__ U) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  size_t p = perm[k];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    float v = Us[3 * k + c] + (self ? Fs[3 * k + c] : 0.f);
    U[3 * p + c] = accumulate ? U[3 * p + c] + v : v;
  }
}
// row 12: explicit Euler X <- X + dt U in fp32, separately rounded product and sum (S-25, L338)
__global__ void __launch_bounds__(256) k_euler(float* __restrict__ X, const float* __restrict__ U, int64_t n3, float dt) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n3) X[t] = __fadd_rn(X[t], __fmul_rn(dt, U[t]));
}

// ------------------------------------------------------------------------------ context
extern "C" int hh_create(hh_ctx** out, const hh_params* params, const hh_mlp* mlp2, const hh_mlp* mlp3, void* workspace,
                         size_t workspace_bytes, void* cuda_stream) {
  if (!out) return HH_ERR_INVALID_ARG;
  *out = nullptr;
  if (!check_params(params) || !mlp2 || !workspace) return HH_ERR_INVALID_ARG;
  if (((uintptr_t)workspace & 255) != 0) return HH_ERR_INVALID_ARG;
  if (!mlp3 && params->rcut3 > 0.f && !(mlp2->n_layers == 3 && mlp2->dims && mlp2->dims[3] == 18)) return HH_ERR_INVALID_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return HH_ERR_CUDA; }   // no CPU fallback
  hh_ctx* ctx = new (std::nothrow) hh_ctx();
  if (!ctx) return HH_ERR_INVALID_ARG;
  memset(ctx, 0, sizeof *ctx);
  ctx->p = *params;
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->ws = (char*)workspace;
  ctx->ws_bytes = workspace_bytes;
  ctx->pairs_per_particle = 32;
  ctx->l_pred = ctx->l_pred_first = 32.0;
  *out = ctx;
  {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) {
      cudaGetLastError();
      return hh_fail(ctx, HH_ERR_CUDA, "cannot query the SM count of the current device");
    }
    ctx->n_sm = nsm;
  }                                       // returned even on failure so hh_last_error works
  int r = carve(ctx, 1);
  if (r != HH_OK) return r;
  HH_CUDA(cudaMallocHost((void**)&ctx->h_sc, sizeof(DevScalars)));
  HH_CUDA(cudaMemsetAsync(ctx->d_sc, 0, sizeof(DevScalars), ctx->stream));
  for (int k = 0; k < 8; ++k) HH_CUDA(cudaEventCreate(&ctx->ev[k]));
  HH_CUDA(cudaStreamCreateWithFlags(&ctx->stream2, cudaStreamNonBlocking));
  for (int k = 0; k < 2; ++k) HH_CUDA(cudaEventCreateWithFlags(&ctx->ev_ab[k], cudaEventDisableTiming));
  std::vector<float> pk;
  if (mlp2->n_layers == 4) {                        // the paper-size network: tensor-core tile of hh_wide.cuh
    if (params->kappa_max > 0.f || params->aca_precision != 0)
      return hh_fail(ctx, HH_ERR_UNSUPPORTED, "the paper-size MLP path has neither the S-18b dense fallback nor the fp64 parity mode");
    std::vector<float> pw(hh_wide_floats());
    r = hh_pack_wide(ctx, mlp2, pw.data());
    if (r != HH_OK) return hh_fail(ctx, r, "a 4-layer two-body MLP must be 4->128->512->128->9 with device weight pointers");
    HH_CUDA(cudaMemcpyAsync(ctx->w2w, pw.data(), pw.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    HH_CUDA(cudaStreamSynchronize(ctx->stream));
    ctx->mlp2_wide = 1;
  } else {
  std::vector<float> pks;
  r = pack_mlp(ctx, mlp2, 4, HH_MLP2_INP, HH_MLP2_H, pk, &pks);
  if (r != HH_OK) return hh_fail(ctx, r, "two-body MLP must be 4->32->32->9 / 18 (or 4->128->512->128->9) with device weight pointers");
  if (!pks.empty()) {
    HH_CUDA(cudaMemcpyAsync(ctx->w2s, pks.data(), pks.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    ctx->have_self2 = 1;
  }
  HH_CUDA(cudaMemcpyAsync(ctx->w2, pk.data(), pk.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
  std::vector<double> pkd(pk.begin(), pk.end());
  std::vector<float> w2tc(2 * 1024);
  hh_pack_w2_tc(pk.data() + HH_MLP2_H * HH_MLP2_INP + HH_MLP2_H, w2tc.data());     // W2 follows W1 and b1 in the packed layout
  HH_CUDA(cudaMemcpyAsync(ctx->w2tc, w2tc.data(), w2tc.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
  HH_CUDA(cudaMemcpyAsync(ctx->w2d, pkd.data(), pkd.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  }
  if (mlp3) {
    std::vector<float> pks3;
    r = pack_mlp(ctx, mlp3, 7, HH_MLP3_INP, HH_MLP3_H, pk, &pks3);
    if (r != HH_OK) return hh_fail(ctx, r, "three-body MLP must be 7->64->64->9 / 18 with device weight pointers");
    if (!pks3.empty()) {
      HH_CUDA(cudaMemcpyAsync(ctx->w3s, pks3.data(), pks3.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
      HH_CUDA(cudaStreamSynchronize(ctx->stream));
      ctx->have_self3 = 1;
    }
    HH_CUDA(cudaMemcpyAsync(ctx->w3, pk.data(), pk.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    HH_CUDA(cudaStreamSynchronize(ctx->stream));
    ctx->have_mlp3 = 1;
  }
  ctx->Ncap = 0;
  return HH_OK;
}

extern "C" int hh_destroy(hh_ctx* ctx) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (ctx->h_sc) cudaFreeHost(ctx->h_sc);
  for (int k = 0; k < 8; ++k) if (ctx->ev[k]) cudaEventDestroy(ctx->ev[k]);
  for (int k = 0; k < 2; ++k) if (ctx->ev_ab[k]) cudaEventDestroy(ctx->ev_ab[k]);
  if (ctx->stream2) cudaStreamDestroy(ctx->stream2);
  delete ctx;
  return HH_OK;
}

extern "C" int hh_set_params(hh_ctx* ctx, const hh_params* params) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!check_params(params)) return hh_fail(ctx, HH_ERR_INVALID_ARG, "invalid parameters");
  if (params->rcut3 > 0.f && !ctx->have_mlp3 && !ctx->have_self2) return hh_fail(ctx, HH_ERR_INVALID_ARG, "rcut3 > 0 needs a three-body MLP or an 18-output two-body MLP");
  if (ctx->mlp2_wide && (params->kappa_max > 0.f || params->aca_precision != 0))
    return hh_fail(ctx, HH_ERR_UNSUPPORTED, "the paper-size MLP path has neither the S-18b dense fallback nor the fp64 parity mode");
  if (params->leaf_size != ctx->p.leaf_size) ctx->tree_ok = ctx->blocks_ok = 0;
  if (params->eta != ctx->p.eta) ctx->blocks_ok = 0;
  ctx->res_first = ctx->res_next = 0;               // factors depend on tol / rank cap / rule / kappa_max
  ctx->n_dense = 0;
  ctx->l_pred = ctx->l_pred_first = 32.0;
  ctx->p = *params;
  return HH_OK;
}

extern "C" int hh_set_pair_capacity(hh_ctx* ctx, int64_t pairs_per_particle) {
  if (!ctx || pairs_per_particle < 1) return HH_ERR_INVALID_ARG;
  ctx->pairs_per_particle = pairs_per_particle;
  ctx->Ncap = 0; ctx->tree_ok = ctx->blocks_ok = 0;
  return HH_OK;
}

// 0 = lock-step over the batch, entries (k2_eval) and vectorised update (k2_upd) as separate launches (default),
// 1 = one CTA per admissible block (the first form), 2 = lock-step with the stored terms staged through shared memory by TMA
// bulk copies, 3 = lock-step with entries and update fused in one kernel (k2_step), 4 = form 0 on two half-batches (a2_two_halves);
// 1-4 measured slower, kept for comparison
extern "C" int hh_set_aca_impl(hh_ctx* ctx, int impl) {
  if (!ctx || impl < 0 || impl > 4) return HH_ERR_INVALID_ARG;
  if (impl == 1 && ctx->mlp2_wide) return hh_fail(ctx, HH_ERR_UNSUPPORTED, "the paper-size MLP runs in the lock-step form only");
  ctx->aca_impl = impl;
  ctx->res_first = ctx->res_next = 0;
  return HH_OK;
}

// 0 = ring kernels (TMA bulk copies into a shared-memory ring, persistent CTAs) for blocks with max(m,n) <= 1024 (default),
// 1 = one CTA per block in every size class (round 1's kernel), 2 = ring kernel only up to 256; 1, 2 kept for comparison
extern "C" int hh_set_far_impl(hh_ctx* ctx, int impl) {
  if (!ctx || impl < 0 || impl > 2) return HH_ERR_INVALID_ARG;
  ctx->far_impl = impl;
  return HH_OK;
}

// error flag of the ring kernel and its item list (one 4-byte read-back per mat-vec)
static int far_check(hh_ctx* ctx) {
  HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->far_err, &ctx->d_sc->far_err, sizeof(u32), cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  if (ctx->h_sc->far_err == 2) return hh_fail(ctx, HH_ERR_CUDA, "far-field ring kernel: item list overflow (internal)");
  if (ctx->h_sc->far_err) return hh_fail(ctx, HH_ERR_CUDA, "far-field ring kernel: an mbarrier wait timed out");
  return HH_OK;
}

extern "C" int hh_set_capture(hh_ctx* ctx, const int32_t* row_prefix, int32_t* records, int64_t cap_records) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (records && (!row_prefix || cap_records < 1)) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_set_capture: records without row_prefix / capacity");
  ctx->cap_prefix = records ? row_prefix : nullptr;
  ctx->cap_rec = records;
  ctx->cap_max = records ? cap_records : 0;
  HH_CUDA(cudaMemsetAsync(&ctx->d_sc->cap_count, 0, sizeof(u64), ctx->stream));
  return HH_OK;
}

extern "C" int hh_get_capture_count(hh_ctx* ctx, int64_t* n_records) {
  if (!ctx || !n_records) return HH_ERR_INVALID_ARG;
  u64 n = 0;
  HH_CUDA(cudaMemcpyAsync(&n, &ctx->d_sc->cap_count, sizeof n, cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  *n_records = (int64_t)n;
  return HH_OK;
}

extern "C" int hh_enable_timing(hh_ctx* ctx, int on) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  ctx->timing = on;
  return HH_OK;
}

extern "C" const char* hh_last_error(const hh_ctx* ctx) { return ctx ? ctx->err : "null context"; }
extern "C" const char* hh_version(void) { return "hh-b200 0.1 (sm_100a)"; }

// ------------------------------------------------------------------------------ stage drivers
#define T0(i) do { if (ctx->timing) cudaEventRecord(ctx->ev[i], ctx->stream); } while (0)
static float ev_ms(hh_ctx* ctx, int a, int b) {
  float ms = 0.f;
  cudaEventSynchronize(ctx->ev[b]);
  cudaEventElapsedTime(&ms, ctx->ev[a], ctx->ev[b]);
  return ms;
}

extern "C" int hh_build_tree(hh_ctx* ctx, const float* X, int64_t N) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!X || N < 1 || N > 0x7fffffff / 4) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_build_tree: X null or N out of range");
  if (N > ctx->Ncap || N * 4 < ctx->Ncap) HH_TRY(carve(ctx, N));
  ctx->n_launches = 0;
  T0(0);
  HH_TRY(hh_tree_build(ctx, X, N));
  T0(1);
  if (ctx->timing) ctx->st.ms_tree = ev_ms(ctx, 0, 1);
  return HH_OK;
}

extern "C" int hh_build_blocks(hh_ctx* ctx) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  T0(0);
  HH_TRY(hh_blocks_build(ctx));
  T0(1);
  if (ctx->timing) ctx->st.ms_blocks = ev_ms(ctx, 0, 1);
  return HH_OK;
}

extern "C" int hh_aca(hh_ctx* ctx, int64_t first_block, int64_t* next_block) {
  if (!ctx || !next_block) return HH_ERR_INVALID_ARG;
  if (!ctx->blocks_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_aca before hh_build_blocks");
  if (first_block < 0 || first_block > ctx->nG) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_aca: first_block out of range");
  if (first_block == ctx->nG) { *next_block = ctx->nG; ctx->res_first = ctx->res_next = ctx->nG; return HH_OK; }
  T0(2);
  HH_TRY(ctx->aca_impl == 1 ? hh_aca_batch(ctx, first_block, next_block) : hh_aca2_batch(ctx, first_block, next_block));
  T0(3);
  if (ctx->timing) ctx->st.ms_aca += ev_ms(ctx, 2, 3);
  return HH_OK;
}

extern "C" int hh_matvec_parts(hh_ctx* ctx, const float* F, float* U, int parts) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!F || !U) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_matvec: null F or U");
  if (!ctx->blocks_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_matvec before hh_build_blocks");
  cudaStream_t s = ctx->stream;
  const int64_t N = ctx->N;
  if (ctx->timing) { ctx->st.ms_aca = ctx->st.ms_near = ctx->st.ms_far = ctx->st.ms_three = ctx->st.ms_other = 0.f; }
  T0(4);
  k_gather_f<<<HH_N + cdiv(N, 256), 256, 0, s>>>(F, ctx->perm, N, ctx->Fs, ctx->Us);
  HH_LAUNCH_CHECK();
  T0(5);
  if (ctx->timing) ctx->st.ms_other += ev_ms(ctx, 4, 5);
  if (parts & 2) {
    T0(4);
    HH_TRY(hh_near_apply(ctx));
    T0(5);
    if (ctx->timing) ctx->st.ms_near = ev_ms(ctx, 4, 5);
  }
  if ((parts & 4) && ctx->nG > 0) {
    bool resident_all = ctx->res_first == 0 && ctx->res_next == ctx->nG;
    if (resident_all) {
      T0(4);
      HH_TRY(hh_far_apply(ctx));
      T0(5);
      if (ctx->timing) ctx->st.ms_far += ev_ms(ctx, 4, 5);
      T0(4);
      HH_TRY(hh_dense_apply(ctx));
      T0(5);
      if (ctx->timing) ctx->st.ms_near += ev_ms(ctx, 4, 5);
    } else {
      // factors are streamed through the arena batch by batch (L246, L260, L334)
      ctx->st.sum_rank = ctx->st.aca_entries = ctx->st.factor_bytes = ctx->st.aca_batches = 0;
      ctx->st.aca_not_converged = ctx->st.aca_singular = ctx->st.fallback_entries = 0;
      int64_t first = 0;
      while (first < ctx->nG) {
        int64_t next = first;
        HH_TRY(hh_aca(ctx, first, &next));
        if (next <= first) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "factor arena cannot hold a single admissible block");
        T0(4);
        HH_TRY(hh_far_apply(ctx));
        T0(5);
        if (ctx->timing) ctx->st.ms_far += ev_ms(ctx, 4, 5);
        T0(4);
        HH_TRY(hh_dense_apply(ctx));
        T0(5);
        if (ctx->timing) ctx->st.ms_near += ev_ms(ctx, 4, 5);
        first = next;
      }
    }
  }
  if ((parts & 4) && ctx->nG > 0) HH_TRY(far_check(ctx));
  const int short_modes = ((parts & 8) && ctx->have_mlp3 ? 1 : 0) | ((parts & 16) ? 6 : 0);
  if (short_modes && ctx->p.rcut3 > 0.f) {
    T0(4);
    HH_TRY(hh_three_apply(ctx, short_modes));
    T0(5);
    if (ctx->timing) ctx->st.ms_three = ev_ms(ctx, 4, 5);
  }
  T0(4);
  k_unpermute<<<HH_N + cdiv(N, 256), 256, 0, s>>>(ctx->Us, ctx->Fs, ctx->perm, N, parts & 1, 0, U);
  HH_LAUNCH_CHECK();
  T0(5);
  if (ctx->timing) ctx->st.ms_other += ev_ms(ctx, 4, 5);
  return HH_OK;
}

extern "C" int hh_matvec(hh_ctx* ctx, const float* F, float* U) { return hh_matvec_parts(ctx, F, U, 31); }

extern "C" int hh_far_apply_resident(hh_ctx* ctx, const float* F, float* U) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!F || !U) return hh_fail(ctx, HH_ERR_INVALID_ARG, "null F or U");
  if (!ctx->blocks_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_far_apply_resident before hh_build_blocks");
  const int64_t N = ctx->N;
  k_gather_f<<<HH_N + cdiv(N, 256), 256, 0, ctx->stream>>>(F, ctx->perm, N, ctx->Fs, ctx->Us);
  T0(4);
  HH_TRY(hh_far_apply(ctx));
  T0(5);
  if (ctx->timing) ctx->st.ms_far = ev_ms(ctx, 4, 5);
  HH_TRY(hh_dense_apply(ctx));
  k_unpermute<<<HH_N + cdiv(N, 256), 256, 0, ctx->stream>>>(ctx->Us, ctx->Fs, ctx->perm, N, 0, 0, U);
  HH_LAUNCH_CHECK();
  return far_check(ctx);
}

extern "C" int hh_step(hh_ctx* ctx, float* X, const float* F, float* U, int64_t N, float dt) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!X || !F || !U || !isfinite(dt)) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_step: null pointer or non-finite dt");
  HH_TRY(hh_build_tree(ctx, X, N));
  HH_TRY(hh_build_blocks(ctx));
  HH_TRY(hh_matvec(ctx, F, U));
  k_euler<<<HH_N + cdiv(3 * N, 256), 256, 0, ctx->stream>>>(X, U, 3 * N, dt);
  HH_LAUNCH_CHECK();
  return HH_OK;
}

// End-to-end variant with HOST buffers: copies X, F in, runs hh_step, copies X, U out, synchronises.
extern "C" int hh_step_host(hh_ctx* ctx, float* X_host, const float* F_host, float* U_host, int64_t N, float dt) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!X_host || !F_host || !U_host || N < 1) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_step_host: null pointer");
  if (N > ctx->Ncap || N * 4 < ctx->Ncap) HH_TRY(carve(ctx, N));
  size_t b = (size_t)3 * N * sizeof(float);
  HH_CUDA(cudaMemcpyAsync(ctx->stageX, X_host, b, cudaMemcpyHostToDevice, ctx->stream));
  HH_CUDA(cudaMemcpyAsync(ctx->stageF, F_host, b, cudaMemcpyHostToDevice, ctx->stream));
  HH_TRY(hh_step(ctx, ctx->stageX, ctx->stageF, ctx->stageU, N, dt));
  HH_CUDA(cudaMemcpyAsync(U_host, ctx->stageU, b, cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaMemcpyAsync(X_host, ctx->stageX, b, cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  return HH_OK;
}

// ------------------------------------------------------------------------------ introspection
extern "C" int hh_get_stats(hh_ctx* ctx, hh_stats* st) {
  if (!ctx || !st) return HH_ERR_INVALID_ARG;
  *st = ctx->st;
  st->n_launches = ctx->n_launches;
  return HH_OK;
}

template <typename S, typename D>
static int fetch(hh_ctx* ctx, const S* dev, size_t n, D* host) {
  if (!host || n == 0) return HH_OK;
  std::vector<S> tmp(n);
  HH_CUDA(cudaMemcpyAsync(tmp.data(), dev, n * sizeof(S), cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  for (size_t i = 0; i < n; ++i) host[i] = (D)tmp[i];
  return HH_OK;
}

extern "C" int hh_get_tree(hh_ctx* ctx, int64_t* perm, uint64_t* keys, int64_t* lo, int64_t* hi, int32_t* left, int32_t* right,
                           int32_t* parent, int32_t* level, float* bmin, float* bmax) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!ctx->tree_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_get_tree before hh_build_tree");
  size_t N = (size_t)ctx->N, nn = (size_t)ctx->n_nodes;
  HH_TRY(fetch(ctx, ctx->perm, N, perm));
  HH_TRY(fetch(ctx, ctx->keys[0], N, keys));
  HH_TRY(fetch(ctx, ctx->nlo, nn, lo));
  HH_TRY(fetch(ctx, ctx->nhi, nn, hi));
  HH_TRY(fetch(ctx, ctx->nleft, nn, left));
  if (right) {
    HH_TRY(fetch(ctx, ctx->nleft, nn, right));
    for (size_t i = 0; i < nn; ++i) if (right[i] >= 0) right[i] += 1;
  }
  HH_TRY(fetch(ctx, ctx->nparent, nn, parent));
  HH_TRY(fetch(ctx, ctx->nlevel, nn, level));
  HH_TRY(fetch(ctx, ctx->bmin, 3 * nn, bmin));
  HH_TRY(fetch(ctx, ctx->bmax, 3 * nn, bmax));
  return HH_OK;
}

extern "C" int hh_get_blocks(hh_ctx* ctx, int which, int32_t* tau, int32_t* sigma) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!ctx->blocks_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_get_blocks before hh_build_blocks");
  if (which != 0 && which != 1) return hh_fail(ctx, HH_ERR_INVALID_ARG, "which must be 0 (P^G) or 1 (P^H)");
  size_t n = (size_t)(which == 0 ? ctx->nG : ctx->nH);
  if (n == 0) return HH_OK;
  std::vector<uint2> tmp(n);
  HH_CUDA(cudaMemcpyAsync(tmp.data(), which == 0 ? ctx->PG : ctx->PH, n * sizeof(uint2), cudaMemcpyDeviceToHost, ctx->stream));
  HH_CUDA(cudaStreamSynchronize(ctx->stream));
  for (size_t i = 0; i < n; ++i) { if (tau) tau[i] = (int32_t)tmp[i].x; if (sigma) sigma[i] = (int32_t)tmp[i].y; }
  return HH_OK;
}

extern "C" int hh_get_ranks(hh_ctx* ctx, int32_t* ranks, int32_t* flags) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!ctx->blocks_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_get_ranks before hh_build_blocks");
  HH_TRY(fetch(ctx, ctx->ranks, (size_t)ctx->nG, ranks));
  HH_TRY(fetch(ctx, ctx->flags, (size_t)ctx->nG, flags));
  return HH_OK;
}

extern "C" int hh_get_factors(hh_ctx* ctx, int64_t block, int32_t* rank, int32_t* flag, int32_t cap_rank, int32_t* piv_i,
                              int32_t* piv_j, float* C, float* Q) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!ctx->blocks_ok) return hh_fail(ctx, HH_ERR_NOT_BUILT, "hh_get_factors before hh_build_blocks");
  if (block < ctx->res_first || block >= ctx->res_next) return hh_fail(ctx, HH_ERR_INVALID_ARG, "block is not resident in the arena");
  return hh_factors_fetch(ctx, block, rank, flag, cap_rank, piv_i, piv_j, C, Q);
}

extern "C" int hh_eval_entries(hh_ctx* ctx, const float* Xi, const float* Xj, int64_t n, float* M) {
  if (!ctx) return HH_ERR_INVALID_ARG;
  if (!Xi || !Xj || !M || n < 0) return hh_fail(ctx, HH_ERR_INVALID_ARG, "hh_eval_entries: null pointer");
  if (n == 0) return HH_OK;
  return ctx->mlp2_wide ? hh_entries_eval_wide(ctx, Xi, Xj, n, M) : hh_entries_eval(ctx, Xi, Xj, n, M);
}
