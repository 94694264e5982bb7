// hh_prims.cu -- device-wide exclusive scans and a stable LSD radix sort (keys u64, values u32).
// Integer plumbing for SURVEY 8(a) rows 2, 3, 5 (north_star: "integer tree and block-list construction
// via warp-level scans and ballots").  Everything is ordered, hence deterministic.
#include "hh_internal.cuh"

#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) k_tile_sum(const T* __restrict__ in, T* __restrict__ tsum, int64_t n) {
  __shared__ T sm[33];
  int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
  T s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < n) s += in[base + k];
  T tot;
  block_excl_scan<T>(s, sm, &tot);
  if (threadIdx.x == 0) tsum[blockIdx.x] = tot;
}

// single block: in-place exclusive scan of `a[0..n)`, total -> *total (if non-null)
template <typename T>
__global__ void __launch_bounds__(1024) k_scan_single(T* a, int64_t n, T* total) {
  __shared__ T sm[33];
  T carry = 0;
  for (int64_t b = 0; b < n; b += 1024) {
    int64_t i = b + threadIdx.x;
    T v = i < n ? a[i] : T(0);
    T tot;
    T ex = block_excl_scan<T>(v, sm, &tot);
    if (i < n) a[i] = carry + ex;
    carry += tot;
  }
  if (threadIdx.x == 0 && total) *total = carry;
}

__global__ void __launch_bounds__(1024) k_scan_single_cnt3(Cnt3* a, int64_t n, Cnt3* total) {
  __shared__ u32 sm[33];
  Cnt3 carry{0, 0, 0};
  for (int64_t b = 0; b < n; b += 1024) {
    int64_t i = b + threadIdx.x;
    Cnt3 v = i < n ? a[i] : Cnt3{0, 0, 0};
    u32 tg, th, tc;
    u32 eg = block_excl_scan<u32>(v.g, sm, &tg);
    u32 eh = block_excl_scan<u32>(v.h, sm, &th);
    u32 ec = block_excl_scan<u32>(v.c, sm, &tc);
    if (i < n) a[i] = Cnt3{carry.g + eg, carry.h + eh, carry.c + ec};
    carry = carry + Cnt3{tg, th, tc};
  }
  if (threadIdx.x == 0 && total) *total = carry;
}

template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) k_tile_scan(const T* in, T* out, const T* __restrict__ tsum, int64_t n) {
  __shared__ T sm[33];
  int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
  T v[SCAN_ITEMS];
  T s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? in[base + k] : T(0); s += v[k]; }
  T tot;
  T ex = block_excl_scan<T>(s, sm, &tot) + tsum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) out[base + k] = ex; ex += v[k]; }
}

template <typename T>
static int scan_impl(hh_ctx* ctx, const T* in, T* out, int64_t n, T* total_dev) {
  if (n <= 0) {
    if (total_dev) HH_CUDA(cudaMemsetAsync(total_dev, 0, sizeof(T), ctx->stream));
    return HH_OK;
  }
  int64_t nt = (n + SCAN_TILE - 1) / SCAN_TILE;
  T* ts = (T*)ctx->tilesum;
  k_tile_sum<T><<<HH_N + (unsigned)nt, SCAN_THREADS, 0, ctx->stream>>>(in, ts, n);
  k_scan_single<T><<<HH_N + 1, 1024, 0, ctx->stream>>>(ts, nt, total_dev);
  k_tile_scan<T><<<HH_N + (unsigned)nt, SCAN_THREADS, 0, ctx->stream>>>(in, out, ts, n);
  HH_LAUNCH_CHECK();
  return HH_OK;
}

int hh_scan_u32(hh_ctx* ctx, const u32* in, u32* out, int64_t n, u32* total_dev) { return scan_impl<u32>(ctx, in, out, n, total_dev); }
int hh_scan_u64(hh_ctx* ctx, const u64* in, u64* out, int64_t n, u64* total_dev) { return scan_impl<u64>(ctx, in, out, n, total_dev); }

int hh_scan_cnt3(hh_ctx* ctx, Cnt3* tiles, int64_t ntiles, Cnt3* total_dev) {
  k_scan_single_cnt3<<<HH_N + 1, 1024, 0, ctx->stream>>>(tiles, ntiles, total_dev);
  HH_LAUNCH_CHECK();
  return HH_OK;
}

// ------------------------------------------------------------------------------ radix sort
// Each warp owns a contiguous segment of RS_SEG items and walks it 32 at a time in order, so the
// per-(digit, warp) counters give a stable scatter (S-9: ties by original index).
#define RS_SEG 2048
#define RS_WARPS 8

__global__ void __launch_bounds__(RS_WARPS * 32) k_rs_hist(const u64* __restrict__ keys, int64_t n, int shift,
                                                            u32* __restrict__ hist, u32 NW) {
  __shared__ u32 sh[RS_WARPS][256];
  const u32 w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const u32 gw = blockIdx.x * RS_WARPS + w;
  for (int d = lane; d < 256; d += 32) sh[w][d] = 0;
  __syncwarp();
  if (gw >= NW) return;
  int64_t beg = (int64_t)gw * RS_SEG, end = beg + RS_SEG < n ? beg + RS_SEG : n;
  for (int64_t b = beg; b < end; b += 32) {
    int64_t i = b + lane;
    bool valid = i < end;
    u32 d = valid ? (u32)((keys[i] >> shift) & 0xFF) : 0x100u;
    u32 peers = __match_any_sync(0xffffffffu, d);
    if (valid && lane == (u32)(__ffs(peers) - 1)) sh[w][d] += __popc(peers);
    __syncwarp();
  }
  for (int d = lane; d < 256; d += 32) hist[(size_t)d * NW + gw] = sh[w][d];
}

__global__ void __launch_bounds__(RS_WARPS * 32) k_rs_scatter(const u64* __restrict__ keys, const u32* __restrict__ vals,
                                                               u64* __restrict__ okeys, u32* __restrict__ ovals,
                                                               int64_t n, int shift, const u32* __restrict__ hist, u32 NW) {
  __shared__ u32 sh[RS_WARPS][256];
  const u32 w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const u32 gw = blockIdx.x * RS_WARPS + w;
  if (gw >= NW) return;
  for (int d = lane; d < 256; d += 32) sh[w][d] = hist[(size_t)d * NW + gw];
  __syncwarp();
  int64_t beg = (int64_t)gw * RS_SEG, end = beg + RS_SEG < n ? beg + RS_SEG : n;
  const u32 lt = (1u << lane) - 1u;
  for (int64_t b = beg; b < end; b += 32) {
    int64_t i = b + lane;
    bool valid = i < end;
    u64 k = valid ? keys[i] : 0;
    u32 v = valid ? vals[i] : 0;
    u32 d = valid ? (u32)((k >> shift) & 0xFF) : 0x100u;
    u32 peers = __match_any_sync(0xffffffffu, d);
    u32 pos = valid ? sh[w][d] + __popc(peers & lt) : 0;
    __syncwarp();
    if (valid && lane == (u32)(__ffs(peers) - 1)) sh[w][d] += __popc(peers);
    __syncwarp();
    if (valid) { okeys[pos] = k; ovals[pos] = v; }
  }
}

int hh_sort_pairs(hh_ctx* ctx, u64* keys[2], u32* vals[2], int64_t n, int bit_lo, int bit_hi, int* which) {
  int cur = 0;
  if (n > 0) {
    u32 NW = (u32)((n + RS_SEG - 1) / RS_SEG);
    if ((size_t)NW * 256 > ctx->hist_cap) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "radix histogram buffer too small");
    unsigned grid = (NW + RS_WARPS - 1) / RS_WARPS;
    for (int shift = bit_lo; shift < bit_hi; shift += 8) {
      k_rs_hist<<<HH_N + grid, RS_WARPS * 32, 0, ctx->stream>>>(keys[cur], n, shift, ctx->hist, NW);
      HH_TRY(hh_scan_u32(ctx, ctx->hist, ctx->hist, (int64_t)NW * 256, nullptr));
      k_rs_scatter<<<HH_N + grid, RS_WARPS * 32, 0, ctx->stream>>>(keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n, shift,
                                                           ctx->hist, NW);
      cur ^= 1;
    }
    HH_LAUNCH_CHECK();
  }
  *which = cur;
  return HH_OK;
}
