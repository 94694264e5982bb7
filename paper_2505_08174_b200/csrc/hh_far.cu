// hh_far.cu -- SURVEY 8(a) row 9, the roofline-graded kernel: far-field apply over the factors resident in
// the arena, U^tau += C (Q F^sigma) per admissible block.  Bandwidth-bound: every
// factor byte is read exactly once, as coalesced float4 (Q) / 128-B warp rows (C) from plane-major storage;
// F^sigma is staged in shared memory tile by tile; t = Q F^sigma (3 floats per rank) never leaves the SM.
#include "hh_internal.cuh"

#define FAR_SUB 512            /* columns per (rank, sub-tile) warp work unit                 */

__device__ __forceinline__ u32 pad8f(u32 v) { return (v + 7u) & ~7u; }
__device__ __forceinline__ float4 ldg_stream(const float4* p) {   // streamed once: do not allocate in L1
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ float ldg_stream1(const float* p) {
  float v;
  asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}

// T threads; JT = source columns staged per tile (>= the largest n of the size class, or 2048 with tiling)
template <int T, int JT>
__global__ void __launch_bounds__(T, 1024 / T) k_far(const uint2* __restrict__ PG, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                            const int* __restrict__ ranks, const int* __restrict__ flags, const u32* __restrict__ tab, const float* __restrict__ arena,
                                            const float* __restrict__ Fs, float* __restrict__ Us, u32 first, u32 begin) {
  __shared__ __align__(16) float sF[3][JT];        // component-major force tile
  __shared__ float st[HH_MAX_RANK * 3];                // t_k = Q_k F^sigma
  __shared__ u32 sch[HH_MAX_CHUNKS];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = T / 32;
  const u32 g = begin + blockIdx.x;
  const int l = ranks[g];
  if (l <= 0 || flags[g] == 2) return;             // nothing factorised / Alg. 2 broke down (applied densely, S-18b)
  const uint2 blk = PG[g];
  const u32 tlo = nlo[blk.x], m = nhi[blk.x] - tlo;
  const u32 slo = nlo[blk.y], n = nhi[blk.y] - slo;
  const u32 mp = pad8f(m), np = pad8f(n);
  const u32* row = tab + (size_t)(g - first) * HH_TAB_STRIDE;
  if (tid < HH_MAX_CHUNKS) sch[tid] = row[tid];
  for (int t = tid; t < 3 * l; t += T) st[t] = 0.f;
  // ---- phase 1: t_k = sum_j Q_k(j) F(j) ----
  for (u32 j0 = 0; j0 < n; j0 += JT) {
    const u32 nt = min((u32)JT, n - j0), ntp = pad8f(nt);
    __syncthreads();
    for (u32 t = tid; t < 3 * ntp; t += T) {
      u32 j = t / 3, c = t - 3 * j;
      sF[c][j] = j < nt ? Fs[3 * (size_t)(slo + j0) + t] : 0.f;
    }
    __syncthreads();
    const u32 nsub = (ntp + FAR_SUB - 1) / FAR_SUB;
    for (u32 u = warp; u < (u32)l * nsub; u += NW) {
      const u32 k = u / nsub, sb = u - k * nsub;
      const u32 c0 = sb * FAR_SUB, cn = min((u32)FAR_SUB, ntp - c0);          // multiple of 8
      const float* Qk = arena + (size_t)sch[k / HH_RC] * HH_UNIT_FLOATS + (size_t)HH_RC * 9 * mp + (size_t)(k % HH_RC) * 9 * np + j0 + c0;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f;
      for (u32 j4 = lane; j4 < cn / 4; j4 += 32) {
        float4 q[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) q[e] = ldg_stream(reinterpret_cast<const float4*>(Qk + (size_t)e * np) + j4);
        const float4 fx = *reinterpret_cast<const float4*>(&sF[0][c0 + 4 * j4]);
        const float4 fy = *reinterpret_cast<const float4*>(&sF[1][c0 + 4 * j4]);
        const float4 fz = *reinterpret_cast<const float4*>(&sF[2][c0 + 4 * j4]);
#define DOT4(a, b) ((a).x * (b).x + (a).y * (b).y + (a).z * (b).z + (a).w * (b).w)
        a0 += DOT4(q[0], fx) + DOT4(q[1], fy) + DOT4(q[2], fz);
        a1 += DOT4(q[3], fx) + DOT4(q[4], fy) + DOT4(q[5], fz);
        a2 += DOT4(q[6], fx) + DOT4(q[7], fy) + DOT4(q[8], fz);
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o);
      }
      if (lane == 0) { atomicAdd(&st[3 * k], a0); atomicAdd(&st[3 * k + 1], a1); atomicAdd(&st[3 * k + 2], a2); }
    }
  }
  __syncthreads();
  // ---- phase 2: U(i) += sum_k C_k(i) t_k ----
  for (u32 i = tid; i < m; i += T) {
    float u0 = 0.f, u1 = 0.f, u2 = 0.f;
    for (int k = 0; k < l; ++k) {
      const float* Ck = arena + (size_t)sch[k / HH_RC] * HH_UNIT_FLOATS + (size_t)(k % HH_RC) * 9 * mp + i;
      float c[9];
#pragma unroll
      for (int e = 0; e < 9; ++e) c[e] = ldg_stream1(Ck + (size_t)e * mp);
      const float t0 = st[3 * k], t1 = st[3 * k + 1], t2 = st[3 * k + 2];
      u0 += c[0] * t0 + c[1] * t1 + c[2] * t2;
      u1 += c[3] * t0 + c[4] * t1 + c[5] * t2;
      u2 += c[6] * t0 + c[7] * t1 + c[8] * t2;
    }
    atomicAdd(&Us[3 * (size_t)(tlo + i)], u0);
    atomicAdd(&Us[3 * (size_t)(tlo + i) + 1], u1);
    atomicAdd(&Us[3 * (size_t)(tlo + i) + 2], u2);
  }
}

// CTA sizes per size class (max(m,n) > 256, <= 256, <= 128, <= 64) and the 64-register cap (32 warps per SM) are measured,
// not derived: the kernel is bound by per-CTA start-up latency and load concurrency.  512 threads / 70 registers for the
// first class gave 4.28 TB/s at c3, 256 threads / 64 registers 5.03 TB/s (c4: 4.52 -> 5.06 TB/s); halving the threads of
// every class again helps c3's ragged 64-particle leaves slightly but costs 15 % at c4's 128-particle leaves.  Round 2: one work
// item per (rank, float4 of columns) flattened over the CTA for the classes whose sigma fits one tile (every lane loading, no
// serialisation of the ranks over the warps): 144.8 -> 149.5 ms at c3, 4.4 -> 4.8 ms at c2 (three shared-memory atomics per item).
int hh_far_apply(hh_ctx* ctx) {
  if (ctx->res_next <= ctx->res_first) return HH_OK;
  cudaStream_t s = ctx->stream;
  const u32 first = (u32)ctx->res_first, end = (u32)ctx->res_next;
  for (int c = 0; c < 4; ++c) {
    u32 b = ctx->class_bound[c] > first ? ctx->class_bound[c] : first;
    u32 e = ctx->class_bound[c + 1] < end ? ctx->class_bound[c + 1] : end;
    if (b >= e) continue;
    switch (c) {
      case 0: k_far<256, 2048><<<HH_N + e - b, 256, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, ctx->arena, ctx->Fs, ctx->Us, first, b); break;
      case 1: k_far<256, 256><<<HH_N + e - b, 256, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, ctx->arena, ctx->Fs, ctx->Us, first, b); break;
      case 2: k_far<128, 128><<<HH_N + e - b, 128, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, ctx->arena, ctx->Fs, ctx->Us, first, b); break;
      default: k_far<64, 64><<<HH_N + e - b, 64, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, ctx->arena, ctx->Fs, ctx->Us, first, b); break;
    }
  }
  HH_LAUNCH_CHECK();
  return HH_OK;
}
