// hh_far.cu -- SURVEY 8(a) row 9, the roofline-graded kernel: far-field apply over the factors resident in
// the arena, U^tau += C (Q F^sigma) per admissible block.  Bandwidth-bound: every
// factor byte is read exactly once from plane-major storage; t = Q F^sigma (3 floats per rank) never leaves the SM.
// Three kernels by block size (P^G is sorted by max(m,n), so each takes a contiguous range of a batch):
//   k_far_ring  max(m,n) <= 256    persistent CTAs, arena chunks through a shared-memory ring filled by TMA bulk copies
//   k_far_mid   257 .. 1024        the same ring, whole blocks per CTA, one bulk copy per rank's nine planes
//   k_far       larger             one CTA per block, coalesced float4 (Q) / 128-B warp rows (C), F^sigma staged per tile
// (hh_set_far_impl selects k_far for everything, or the ring only up to 256, for comparison.)
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

// =====================================================================================================================
// Ring form for the leaf-size classes (max(m,n) <= 256), the B200 way: persistent CTAs, one producer warp that streams
// the factor chunks of ITS share of the batch into a shared-memory byte ring with TMA bulk copies
// (cp.async.bulk + mbarrier complete_tx), and G consumer threads that reduce a chunk while the next ones are in
// flight.  A one-CTA-per-block kernel pays the metadata chain (PG -> nlo/nhi -> table row -> first factor byte) and a
// cold start of its loads once per 13-40 KB block (63-80 % of the copy peak, profiles/r02_far_traffic_c3.md); here the
// copies of up to NS items per CTA are always in flight and nothing waits for a block boundary.
//   item  = one arena chunk of one block (<= HH_RC ranks): C part [kk][9][mp] and Q part [kk][9][np], two bulk copies
//   list  = built per batch by k_far_count / scan / k_far_fill from ranks[], flags[], the table rows (16 B per item)
//   share = groups of 32 consecutive items dealt round-robin to the CTAs (P^G is sorted by size: this balances bytes)
// Consumer, per item:  t_k = sum_j Q_k(j) F(j)  (thread = (rank, column lane), shuffle reduction over the rank's lanes),
// named barrier, U(i) += sum_k C_k(i) t_k accumulated in registers over the items of a block, three atomics per row
// when the block (or the group of 32 items) ends.  The consumers issue no global load at all: the force slice and the
// item descriptor travel through the ring with the factors.
// Measured at c3 (ncu, dram bytes / kernel time, classes 129..256 | 65..128 | <= 64; one CTA per block: 5.18 | 4.61 | 4.05 TB/s):
//   v1  descriptors and F prefetched into registers by the consumers, one row / column per thread   6.35 | 4.99 | 5.63
//       (under full streaming load the L2 round trip of the prefetches takes longer than an item)
//   v2  + F and descriptors through the ring                                                          6.35 | 4.99 | 5.84
//   v3  + 4 rows / columns per lane (LDS.128), shares of U summed over the rank slots at the flush    6.98 | 7.04 | 6.87
//       (and the ring pointer derived without an integer round trip: before that every access was a generic LD.E)
// =====================================================================================================================
#define FAR_NS 8               /* barrier slots = most items in flight per CTA */
/* ring bytes and CTAs per SM of the three ring classes (129..256, 65..128, <= 64 rows / columns) */
#ifndef FAR_RING1
#define FAR_RING1 (98 * 1024)
#define FAR_CTAS1 2
#endif
#ifndef FAR_RING2
#define FAR_RING2 (66 * 1024)
#define FAR_CTAS2 3
#endif
#ifndef FAR_RING3
#define FAR_RING3 (50 * 1024)
#define FAR_CTAS3 4
#endif

__device__ __forceinline__ u32 far_smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ bool far_mbar_wait(u32 bar, u32 parity) {
  for (int it = 0; it < (1 << 22); ++it) {
    u32 ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return true;
  }
  return false;
}
__device__ __forceinline__ void far_decode(const uint4 d, u32& m, u32& n, u32& kk, u32& last) {
  m = d.w & 1023u; n = (d.w >> 10) & 1023u; kk = (d.w >> 20) & 7u; last = (d.w >> 23) & 1u;
}

// G consumer threads (+ 32 producer) = 4 rank slots x LPR lanes; a lane takes NQ quads of 4 consecutive columns resp.
// rows (4 * NQ * LPR >= the largest m, n of the size class); RING bytes of staging per CTA.
template <int G, int NQ, int RING>
__global__ void __launch_bounds__(G + 32) k_far_ring(const uint4* __restrict__ items, const u32* __restrict__ pre, u32 ib, u32 ie,
                                                    const float* __restrict__ arena, const float* __restrict__ Fs, float* __restrict__ Us,
                                                    u32* __restrict__ err) {
  constexpr int LPR = G / 4;
  extern __shared__ __align__(128) unsigned char far_raw[];
  // 128-byte alignment by pointer arithmetic on the shared array itself (a round trip through an integer would make every
  // access below a generic load)
  unsigned char* ringb = far_raw + ((128u - (far_smem_u32(far_raw) & 127u)) & 127u);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(ringb + RING);     // full[NS], empty[NS]
  uint4* sdesc = reinterpret_cast<uint4*>(bars + 2 * FAR_NS);                        // the item in each barrier slot
  u32* soff = reinterpret_cast<u32*>(sdesc + FAR_NS);                                // and where it sits in the ring
  float* st = reinterpret_cast<float*>(soff + FAR_NS);                               // [2][HH_RC][4]
  float* su = st + 2 * HH_RC * 4;                                                    // [HH_RC][4 * NQ * LPR][3]: the rank slots' shares of U at a flush
  const u32 tid = threadIdx.x, lane = tid & 31;
  const u32 it0 = pre[ib], it1 = pre[ie];
  const u32 bar_full = far_smem_u32(bars), bar_empty = far_smem_u32(bars + FAR_NS);
  if (tid == 0) {
    for (int s = 0; s < FAR_NS; ++s) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_full + 8 * s) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar_empty + 8 * s), "r"(G) : "memory");
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // q-th item of this CTA (groups of 32 items, round-robin over the grid); >= it1: no more items
  auto item_index = [&](u32 q) -> unsigned long long {
    return (unsigned long long)it0 + ((unsigned long long)blockIdx.x + (unsigned long long)(q >> 5) * gridDim.x) * 32ull + (q & 31u);
  };
  if (tid >= G) {
    // ------------------------------------------------ producer warp ------------------------------------------------
    // Everything a consumer touches arrives through the ring: factors, the force slice (an aligned superset of
    // F^sigma: bulk copies move multiples of 16 bytes from 16-byte-aligned addresses) and the item descriptor.
    u32 head = 0, released = 0, myoff = 0;               // lane s < NS keeps the ring offset of barrier slot s
    uint4 dl = make_uint4(0, 0, 0, 0);
    unsigned long long pol;                              // factors are read once: first in line for eviction from L2
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    for (u32 q = 0;; ++q) {
      const unsigned long long idx = item_index(q);
      if (idx >= it1) break;
      if ((q & 31u) == 0) { const unsigned long long ii = idx + lane; dl = ii < it1 ? items[ii] : make_uint4(0, 0, 0, 0); }
      uint4 d;
      d.x = __shfl_sync(0xffffffffu, dl.x, q & 31); d.y = __shfl_sync(0xffffffffu, dl.y, q & 31);
      d.z = __shfl_sync(0xffffffffu, dl.z, q & 31); d.w = __shfl_sync(0xffffffffu, dl.w, q & 31);
      u32 m, n, kk, last;
      far_decode(d, m, n, kk, last);
      const u32 mp = pad8f(m), np = pad8f(n);
      const u32 foff = (3u * d.z) & 3u;                  // floats between the aligned start and F(slo)
      const u32 bytesC = 36u * kk * mp, bytesQ = 36u * kk * np, bytesF = ((3u * n + foff) * 4u + 15u) & ~15u;
      const u32 B = bytesC + bytesQ + bytesF;
      u32 off = 0;
      bool alive = true;
      for (;;) {                                         // space in the byte ring: items are released in order
        const u32 outst = q - released;
        if (outst == 0) { off = 0; break; }
        if (outst < FAR_NS) {
          const u32 tail = __shfl_sync(0xffffffffu, myoff, released % FAR_NS);
          bool ok = false;
          if (head > tail) {
            if (head + B <= (u32)RING) { off = head; ok = true; }
            else if (B < tail) { off = 0; ok = true; }
          } else if (head + B < tail) { off = head; ok = true; }
          if (ok) break;
        }
        alive = far_mbar_wait(bar_empty + 8 * (released % FAR_NS), (released / FAR_NS) & 1u);
        if (!alive) break;
        ++released;
      }
      if (!alive) { if (lane == 0) atomicExch(err, 1u); break; }
      head = off + B;
      const u32 slot = q % FAR_NS;
      if (lane == slot) myoff = off;
      if (lane == 0) {
        soff[slot] = off;
        sdesc[slot] = d;
        const u32 fb = bar_full + 8 * slot, dst = far_smem_u32(ringb + off);
        const float* src = arena + (size_t)d.x * HH_UNIT_FLOATS;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fb), "r"(B) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst), "l"(src),
                     "r"(bytesC), "r"(fb), "l"(pol) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst + bytesC),
                     "l"(src + (size_t)HH_RC * 9 * mp), "r"(bytesQ), "r"(fb), "l"(pol) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst + bytesC + bytesQ),
                     "l"(Fs + (3 * (size_t)d.z - foff)), "r"(bytesF), "r"(fb) : "memory");
      }
    }
    return;
  }
  // -------------------------------------------------- consumers --------------------------------------------------
  // thread = (rank slot rk of the chunk, lane ql of the slot's LPR lanes); a lane takes 4 consecutive columns (phase 1)
  // resp. rows (phase 2) at a time, so every factor load is a conflict-free LDS.128
  const u32 rk = tid / LPR, ql = tid % LPR;
  float u[NQ][4][3];                                      // this rank slot's share of U for the lane's rows, over the items of a block
#pragma unroll
  for (int r = 0; r < NQ; ++r)
#pragma unroll
    for (int c = 0; c < 4; ++c) u[r][c][0] = u[r][c][1] = u[r][c][2] = 0.f;
  for (u32 q = 0; item_index(q) < it1; ++q) {
    const u32 slot = q % FAR_NS;
    if (!far_mbar_wait(bar_full + 8 * slot, (q / FAR_NS) & 1u)) { atomicExch(err, 1u); return; }
    const uint4 d0 = sdesc[slot];
    u32 m, n, kk, last;
    far_decode(d0, m, n, kk, last);
    const u32 mp = pad8f(m), np = pad8f(n);
    const float* base = reinterpret_cast<const float*>(ringb + soff[slot]);
    const float* sfa = base + (size_t)9 * kk * (mp + np);  // 16-byte aligned; F(slo) starts foff floats in
    const u32 foff = (3u * d0.z) & 3u;
    // phase 1: t_k = sum_j Q_k(j) F(j)
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
    if (rk < kk) {
      const float* Qb = base + (size_t)kk * 9 * mp + (size_t)rk * 9 * np;
#pragma unroll
      for (int c = 0; c < NQ; ++c) {
        const u32 j = 4u * (ql + c * LPR);
        if (j < n) {
          float4 qv[9];
#pragma unroll
          for (int e = 0; e < 9; ++e) qv[e] = *reinterpret_cast<const float4*>(Qb + e * np + j);
          float w[16], f[12];
#pragma unroll
          for (int e = 0; e < 4; ++e) *reinterpret_cast<float4*>(&w[4 * e]) = *reinterpret_cast<const float4*>(sfa + 3 * j + 4 * e);
          switch (foff) {                                  // uniform over the item: static register indices in every case
            case 0:
#pragma unroll
              for (int e = 0; e < 12; ++e) f[e] = w[e];
              break;
            case 1:
#pragma unroll
              for (int e = 0; e < 12; ++e) f[e] = w[e + 1];
              break;
            case 2:
#pragma unroll
              for (int e = 0; e < 12; ++e) f[e] = w[e + 2];
              break;
            default:
#pragma unroll
              for (int e = 0; e < 12; ++e) f[e] = w[e + 3];
              break;
          }
#pragma unroll
          for (int e = 0; e < 12; ++e) if (j + e / 3 >= n) f[e] = 0.f;   // pad columns: Q is zero there, what lies beyond F^sigma is not
#define FAR_DOT(a, fc) ((a).x * f[(fc)] + (a).y * f[3 + (fc)] + (a).z * f[6 + (fc)] + (a).w * f[9 + (fc)])
          a0 += FAR_DOT(qv[0], 0) + FAR_DOT(qv[1], 1) + FAR_DOT(qv[2], 2);
          a1 += FAR_DOT(qv[3], 0) + FAR_DOT(qv[4], 1) + FAR_DOT(qv[5], 2);
          a2 += FAR_DOT(qv[6], 0) + FAR_DOT(qv[7], 1) + FAR_DOT(qv[8], 2);
        }
      }
    }
#pragma unroll
    for (int o = LPR / 2; o; o >>= 1) {
      a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o);
    }
    float* stq = st + (q & 1u) * (HH_RC * 4);
    if (ql == 0 && rk < kk) { stq[4 * rk] = a0; stq[4 * rk + 1] = a1; stq[4 * rk + 2] = a2; }
    asm volatile("bar.sync 1, %0;" ::"n"(G) : "memory");
    // phase 2: this slot's C_k(i) t_k for the lane's rows (rows >= m of a quad hold whatever the arena held: never flushed)
    if (rk < kk) {
      const float t0 = stq[4 * rk], t1 = stq[4 * rk + 1], t2 = stq[4 * rk + 2];
      const float* Cb = base + (size_t)rk * 9 * mp;
#pragma unroll
      for (int r = 0; r < NQ; ++r) {
        const u32 i = 4u * (ql + r * LPR);
        if (i < m) {
          float4 cv[9];
#pragma unroll
          for (int e = 0; e < 9; ++e) cv[e] = *reinterpret_cast<const float4*>(Cb + e * mp + i);
#define FAR_ROW(c, comp) \
          u[r][c][0] += cv[0].comp * t0 + cv[1].comp * t1 + cv[2].comp * t2; \
          u[r][c][1] += cv[3].comp * t0 + cv[4].comp * t1 + cv[5].comp * t2; \
          u[r][c][2] += cv[6].comp * t0 + cv[7].comp * t1 + cv[8].comp * t2;
          FAR_ROW(0, x) FAR_ROW(1, y) FAR_ROW(2, z) FAR_ROW(3, w)
        }
      }
    }
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar_empty + 8 * slot) : "memory");   // the slot may be refilled
    if (last || (q & 31u) == 31u || item_index(q + 1) >= it1) {
      // the block (or this CTA's share of it) ends: the four rank slots leave their shares in shared memory, then one thread
      // per component adds them up: three atomics per row.  (The barrier of the next item's phases separates two flushes.)
      constexpr u32 SU = 3u * 4u * NQ * LPR;
#pragma unroll
      for (int r = 0; r < NQ; ++r) {
        const u32 i = 4u * (ql + r * LPR);
        float* sp = su + rk * SU + 3 * i;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          sp[3 * c] = u[r][c][0]; sp[3 * c + 1] = u[r][c][1]; sp[3 * c + 2] = u[r][c][2];
          u[r][c][0] = u[r][c][1] = u[r][c][2] = 0.f;
        }
      }
      asm volatile("bar.sync 1, %0;" ::"n"(G) : "memory");
      for (u32 t = tid; t < 3 * m; t += G) atomicAdd(Us + 3 * (size_t)d0.y + t, (su[t] + su[SU + t]) + (su[2 * SU + t] + su[3 * SU + t]));
    }
  }
}

// ---- item list of the resident blocks [b, e) (all of them in the ring classes): count, scan (hh_scan_u32), fill ----
__global__ void __launch_bounds__(256) k_far_count(const int* __restrict__ ranks, const int* __restrict__ flags, u32 b, u32 e, u32* __restrict__ cnt) {
  const u32 g = b + blockIdx.x * blockDim.x + threadIdx.x;
  if (g > e) return;
  u32 c = 0;
  if (g < e) { const int l = ranks[g]; if (l > 0 && flags[g] != 2) c = (u32)(l + HH_RC - 1) / HH_RC; }
  cnt[g - b] = c;                                                           // cnt[e - b] = 0: the scan leaves the total there
}
__global__ void __launch_bounds__(256) k_far_fill(const uint2* __restrict__ PG, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                  const int* __restrict__ ranks, const int* __restrict__ flags, const u32* __restrict__ tab,
                                                  u32 first, u32 b, u32 e, const u32* __restrict__ pre, uint4* __restrict__ items,
                                                  unsigned long long cap, u32* __restrict__ err) {
  const u32 g = b + blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= e) return;
  const int l = ranks[g];
  if (l <= 0 || flags[g] == 2) return;
  const uint2 blk = PG[g];
  const u32 tlo = nlo[blk.x], m = nhi[blk.x] - tlo, slo = nlo[blk.y], n = nhi[blk.y] - slo;
  const u32* row = tab + (size_t)(g - first) * HH_TAB_STRIDE;
  const u32 nc = (u32)(l + HH_RC - 1) / HH_RC, p0 = pre[g - b];
  if ((unsigned long long)p0 + nc > cap || m > 1023u || n > 1023u) { atomicExch(err, 2u); return; }
  for (u32 c = 0; c < nc; ++c) {
    const u32 kk = c + 1 < nc ? (u32)HH_RC : (u32)l - c * HH_RC;
    items[p0 + c] = make_uint4(row[c], tlo, slo, m | (n << 10) | (kk << 20) | ((c + 1 == nc ? 1u : 0u) << 23));
  }
}


// =====================================================================================================================
// The same ring for MID-SIZE blocks (256 < max(m,n) <= HH_FAR_MID_MAX = 1024): a persistent CTA takes WHOLE blocks
// (round-robin over the grid: P^G is sorted by size) and streams each rank term as two items, each ONE contiguous bulk copy
// of 36 n_pad resp. 36 m_pad bytes (the nine planes of a rank lie back to back in an arena chunk):
//   Q items (rank k):  t_k = sum_j Q_k(j) F(j), all 128 consumers over the columns (F^sigma sits in registers for the whole
//                      block), per-warp partial sums to shared memory;
//   C items (rank k):  u(i) += C_k(i) t_k in registers, every thread owning its rows for all ranks; U(i) += u(i) once per block
// in that order (all t of the block, then the C items).  The producer makes up the item descriptors on the fly from the
// block's table row (no item list in memory) and ends with a sentinel.  One CTA per block (k_far<256,2048>) streams these
// blocks at 5.3-5.8 TB/s at c3 (profiles/r02b_far_ring_c3.md).
// A first version cut the blocks into slices of 256 (128) rows: 36 plane segments of 1 KB (512 B) per item, one bulk copy
// each -- 4.2 TB/s (3.4): bulk copies are issued one at a time from uniform registers, and 36 small ones per item cost the
// producer warp more than the item's share of the bandwidth allows.
// =====================================================================================================================
/* Ring bytes and CTAs per SM are measured (c3, ms_far of the step; 123.5 ms with one CTA per block for this class):
 *   200 KB x 1 CTA: 131.6 (one group of consumers per SM: every item's wait - load - reduce chain is exposed);
 *   100 KB x 2 CTAs: 115.0;  60 KB x 3 CTAs with blocks up to 512 only: 117.1;  100 KB x 2 with blocks up to 512 only: 118.6 */
#ifndef FAR_MID_RING
#define FAR_MID_RING (100 * 1024)
#define FAR_MID_CTAS 2
#endif
#define FAR_MID_NQ ((HH_FAR_MID_MAX + 511) / 512)      /* quads of 4 rows / columns per consumer thread */

struct FarMidDesc {            /* 32 bytes, written by the producer into the barrier slot of the item */
  u32 pbase;                   /* first particle (tree order) of the side: slo (Q item) resp. tlo (C item) */
  u32 len;                     /* columns resp. rows */
  u32 lenp;                    /* padded to 8: the plane stride */
  u32 k;                       /* rank term */
  u32 type;                    /* 0 Q item, 1 C item, 2 end */
  u32 flags;                   /* bit 0: first item of its kind in the block (Q: load F^sigma; C: all t are there), bit 1: last C item (flush U), bit 2: parity of the block */
  u32 pad[2];
};

__global__ void __launch_bounds__(128 + 32, FAR_MID_CTAS) k_far_mid(const uint2* __restrict__ PG, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                          const int* __restrict__ ranks, const int* __restrict__ flags, const u32* __restrict__ tab,
                                                          u32 first, u32 begin, u32 end, const float* __restrict__ arena,
                                                          const float* __restrict__ Fs, float* __restrict__ Us, u32* __restrict__ err) {
  constexpr int G = 128, NQ = FAR_MID_NQ, RING = FAR_MID_RING;
  extern __shared__ __align__(128) unsigned char far_raw[];
  unsigned char* ringb = far_raw + ((128u - (far_smem_u32(far_raw) & 127u)) & 127u);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(ringb + RING);     // full[NS], empty[NS]
  FarMidDesc* sdesc = reinterpret_cast<FarMidDesc*>(bars + 2 * FAR_NS);
  u32* soff = reinterpret_cast<u32*>(sdesc + FAR_NS);
  float* stt = reinterpret_cast<float*>(soff + FAR_NS);                              // [2][HH_MAX_RANK][4 warps][4]: partial t_k, by block parity
  const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const u32 bar_full = far_smem_u32(bars), bar_empty = far_smem_u32(bars + FAR_NS);
  if (tid == 0) {
    for (int s = 0; s < FAR_NS; ++s) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_full + 8 * s) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar_empty + 8 * s), "r"(G) : "memory");
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid >= G) {
    // ------------------------------------------------ producer warp ------------------------------------------------
    u32 head = 0, released = 0, myoff = 0, q = 0, par = 0;
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    bool alive = true;
    // reserve B bytes of the ring for item q (items are released in order); false = a wait timed out
    auto reserve = [&](u32 B, u32& off) -> bool {
      for (;;) {
        const u32 outst = q - released;
        if (outst == 0) { off = 0; return true; }
        if (outst < FAR_NS) {
          const u32 tail = __shfl_sync(0xffffffffu, myoff, released % FAR_NS);
          if (head > tail) {
            if (head + B <= (u32)RING) { off = head; return true; }
            if (B < tail) { off = 0; return true; }
          } else if (head + B < tail) { off = head; return true; }
        }
        if (!far_mbar_wait(bar_empty + 8 * (released % FAR_NS), (released / FAR_NS) & 1u)) return false;
        ++released;
      }
    };
    for (u32 g = begin + blockIdx.x; g < end && alive; g += gridDim.x) {
      const int l = ranks[g];
      if (l <= 0 || flags[g] == 2) continue;
      const uint2 blk = PG[g];
      const u32 tlo = nlo[blk.x], m = nhi[blk.x] - tlo, slo = nlo[blk.y], n = nhi[blk.y] - slo;
      const u32 mp = pad8f(m), np = pad8f(n);
      const u32 mych = lane < HH_MAX_CHUNKS ? tab[(size_t)(g - first) * HH_TAB_STRIDE + lane] : 0u;   // lane c: offset of chunk c
      for (u32 it = 0; it < 2u * (u32)l; ++it) {
        const u32 type = it >= (u32)l ? 1u : 0u, k = type ? it - (u32)l : it;
        const u32 lenp = type ? mp : np, B = 36u * lenp;
        u32 off;
        if (!reserve(B, off)) { alive = false; break; }
        head = off + B;
        const u32 slot = q % FAR_NS;
        if (lane == slot) myoff = off;
        const u32 choff = __shfl_sync(0xffffffffu, mych, k / HH_RC);
        if (lane == 0) {
          soff[slot] = off;
          FarMidDesc d;
          d.pbase = type ? tlo : slo; d.len = type ? m : n; d.lenp = lenp; d.k = k; d.type = type;
          d.flags = (k == 0 ? 1u : 0u) | ((type && k + 1 == (u32)l) ? 2u : 0u) | (par << 2); d.pad[0] = d.pad[1] = 0;
          sdesc[slot] = d;
          const u32 fb = bar_full + 8 * slot;
          const float* src = arena + (size_t)choff * HH_UNIT_FLOATS + (type ? (size_t)0 : (size_t)HH_RC * 9 * mp) + (size_t)(k % HH_RC) * 9 * lenp;
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fb), "r"(B) : "memory");
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(far_smem_u32(ringb + off)),
                       "l"(src), "r"(B), "r"(fb), "l"(pol) : "memory");
        }
        ++q;
      }
      par ^= 1u;
    }
    if (!alive) { if (lane == 0) atomicExch(err, 1u); return; }
    u32 off;                                                  // sentinel: the consumers leave
    if (!reserve(16u, off)) { if (lane == 0) atomicExch(err, 1u); return; }
    if (lane == 0) {
      const u32 slot = q % FAR_NS;
      soff[slot] = off;
      FarMidDesc d;
      d.pbase = d.len = d.lenp = d.k = d.flags = d.pad[0] = d.pad[1] = 0; d.type = 2;
      sdesc[slot] = d;
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar_full + 8 * slot) : "memory");
    }
    return;
  }
  // -------------------------------------------------- consumers --------------------------------------------------
  // thread tid owns the quads tid, tid + 128, ... of 4 consecutive columns (Q items) resp. rows (C items)
  float u[NQ][4][3], f[NQ][12];
#pragma unroll
  for (int r = 0; r < NQ; ++r)
#pragma unroll
    for (int c = 0; c < 4; ++c) u[r][c][0] = u[r][c][1] = u[r][c][2] = 0.f;
  for (u32 q = 0;; ++q) {
    const u32 slot = q % FAR_NS;
    if (!far_mbar_wait(bar_full + 8 * slot, (q / FAR_NS) & 1u)) { atomicExch(err, 1u); return; }
    const FarMidDesc d = sdesc[slot];
    if (d.type == 2u) return;
    const u32 len = d.len, lenp = d.lenp;
    const float* base = reinterpret_cast<const float*>(ringb + soff[slot]);
    float* st = stt + (((d.flags >> 2) & 1u) * HH_MAX_RANK + d.k) * 16;
    if (d.type == 0u) {
      if (d.flags & 1u) {                                     // a new block: its F^sigma into registers (zero beyond n)
#pragma unroll
        for (int c = 0; c < NQ; ++c) {
          const u32 j = 4u * (tid + c * G);
#pragma unroll
          for (int e = 0; e < 12; ++e) f[c][e] = j + e / 3 < len ? Fs[3 * (size_t)(d.pbase + j) + e] : 0.f;
        }
      }
      float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
      for (int c = 0; c < NQ; ++c) {
        const u32 j = 4u * (tid + c * G);
        if (j < len) {
          float4 qv[9];
#pragma unroll
          for (int e = 0; e < 9; ++e) qv[e] = *reinterpret_cast<const float4*>(base + e * lenp + j);
#define FAR_DOTM(a, fc) ((a).x * f[c][(fc)] + (a).y * f[c][3 + (fc)] + (a).z * f[c][6 + (fc)] + (a).w * f[c][9 + (fc)])
          a0 += FAR_DOTM(qv[0], 0) + FAR_DOTM(qv[1], 1) + FAR_DOTM(qv[2], 2);
          a1 += FAR_DOTM(qv[3], 0) + FAR_DOTM(qv[4], 1) + FAR_DOTM(qv[5], 2);
          a2 += FAR_DOTM(qv[6], 0) + FAR_DOTM(qv[7], 1) + FAR_DOTM(qv[8], 2);
        }
      }
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar_empty + 8 * slot) : "memory");
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o);
      }
      if (lane == 0) { st[4 * warp] = a0; st[4 * warp + 1] = a1; st[4 * warp + 2] = a2; }
    } else {
      if (d.flags & 1u) asm volatile("bar.sync 1, %0;" ::"n"(G) : "memory");     // every t_k of the block is in shared memory
      const float t0 = (st[0] + st[4]) + (st[8] + st[12]), t1 = (st[1] + st[5]) + (st[9] + st[13]), t2 = (st[2] + st[6]) + (st[10] + st[14]);
#pragma unroll
      for (int r = 0; r < NQ; ++r) {
        const u32 i = 4u * (tid + r * G);
        if (i < len) {
          float4 cv[9];
#pragma unroll
          for (int e = 0; e < 9; ++e) cv[e] = *reinterpret_cast<const float4*>(base + e * lenp + i);
          FAR_ROW(0, x) FAR_ROW(1, y) FAR_ROW(2, z) FAR_ROW(3, w)
        }
      }
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar_empty + 8 * slot) : "memory");
      if (d.flags & 2u) {                                     // the block ends: three atomics per row
#pragma unroll
        for (int r = 0; r < NQ; ++r) {
          const u32 i = 4u * (tid + r * G);
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            if (i + c < len) {
              float* up = Us + 3 * (size_t)(d.pbase + i + c);
              atomicAdd(up, u[r][c][0]); atomicAdd(up + 1, u[r][c][1]); atomicAdd(up + 2, u[r][c][2]);
            }
            u[r][c][0] = u[r][c][1] = u[r][c][2] = 0.f;
          }
        }
      }
    }
  }
}

// CTA sizes per size class (max(m,n) > 256, <= 256, <= 128, <= 64) and the 64-register cap (32 warps per SM) are measured,
// not derived: the kernel is bound by per-CTA start-up latency and load concurrency.  512 threads / 70 registers for the
// first class gave 4.28 TB/s at c3, 256 threads / 64 registers 5.03 TB/s (c4: 4.52 -> 5.06 TB/s); halving the threads of
// every class again helps c3's ragged 64-particle leaves slightly but costs 15 % at c4's 128-particle leaves.  Round 2: one work
// item per (rank, float4 of columns) flattened over the CTA for the classes whose sigma fits one tile (every lane loading, no
// serialisation of the ranks over the warps): 144.8 -> 149.5 ms at c3, 4.4 -> 4.8 ms at c2 (three shared-memory atomics per item).
template <int G, int NQ, int RING>
static int far_ring_launch(hh_ctx* ctx, int cls, u32 ib, u32 ie, int ctas_per_sm) {
  const size_t smem = (size_t)RING + 128 + 2 * FAR_NS * 8 + FAR_NS * 16 + FAR_NS * 4 + 2 * HH_RC * 4 * 4 + (size_t)HH_RC * 3 * 4 * NQ * G;
  if (!(ctx->far_smem_set & (1 << cls))) {
    HH_CUDA(cudaFuncSetAttribute(k_far_ring<G, NQ, RING>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ctx->far_smem_set |= 1 << cls;
  }
  k_far_ring<G, NQ, RING><<<HH_N + (unsigned)(ctx->n_sm * ctas_per_sm), G + 32, smem, ctx->stream>>>(
      ctx->far_items, ctx->far_cnt, ib, ie, ctx->arena, ctx->Fs, ctx->Us, &ctx->d_sc->far_err);
  return HH_OK;
}

int hh_far_apply(hh_ctx* ctx) {
  if (ctx->res_next <= ctx->res_first) return HH_OK;
  cudaStream_t s = ctx->stream;
  const u32 first = (u32)ctx->res_first, end = (u32)ctx->res_next;
  // ring classes (max(m,n) <= 256): item list of the resident blocks, once per batch (it lives in the dead lock-step
  // accumulators of the batch, hh_aca2.cu)
  const u32 rb = ctx->class_bound[1] > first ? ctx->class_bound[1] : first;
  const bool ring = ctx->far_impl != 1 && ctx->far_items != nullptr && rb < end;
  if (ring && !ctx->far_built) {
    k_far_count<<<HH_N + cdiv((int64_t)(end - rb) + 1, 256), 256, 0, s>>>(ctx->ranks, ctx->flags, rb, end, ctx->far_cnt);
    HH_TRY(hh_scan_u32(ctx, ctx->far_cnt, ctx->far_cnt, (int64_t)(end - rb) + 1, nullptr));
    k_far_fill<<<HH_N + cdiv(end - rb, 256), 256, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, first, rb, end, ctx->far_cnt,
                                                           ctx->far_items, (unsigned long long)ctx->far_items_cap, &ctx->d_sc->far_err);
    ctx->far_built = 1;
  }
  for (int c = 0; c < 4; ++c) {
    u32 b = ctx->class_bound[c] > first ? ctx->class_bound[c] : first;
    u32 e = ctx->class_bound[c + 1] < end ? ctx->class_bound[c + 1] : end;
    if (b >= e) continue;
    if (ring && c >= 1) {
      switch (c) {
        case 1: HH_TRY((far_ring_launch<128, 2, FAR_RING1>(ctx, 1, b - rb, e - rb, FAR_CTAS1))); break;
        case 2: HH_TRY((far_ring_launch<128, 1, FAR_RING2>(ctx, 2, b - rb, e - rb, FAR_CTAS2))); break;
        default: HH_TRY((far_ring_launch<64, 1, FAR_RING3>(ctx, 3, b - rb, e - rb, FAR_CTAS3))); break;
      }
      continue;
    }
    if (c == 0 && ctx->far_impl == 0 && ctx->mid_bound < e) {
      // mid-size blocks [max(b, mid_bound), e): whole blocks per persistent CTA, rank by rank through the ring
      const u32 mb = ctx->mid_bound > b ? ctx->mid_bound : b;
      const size_t smem = (size_t)FAR_MID_RING + 128 + 2 * FAR_NS * 8 + FAR_NS * sizeof(FarMidDesc) + FAR_NS * 4 + 2 * HH_MAX_RANK * 16 * 4;
      if (!(ctx->far_smem_set & 1)) {
        HH_CUDA(cudaFuncSetAttribute(k_far_mid, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->far_smem_set |= 1;
      }
      const u32 nblk = e - mb, cap = (u32)ctx->n_sm * FAR_MID_CTAS;
      k_far_mid<<<HH_N + (nblk < cap ? nblk : cap), 128 + 32, smem, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, first, mb, e, ctx->arena,
                                                                          ctx->Fs, ctx->Us, &ctx->d_sc->far_err);
      e = mb;
      if (b >= e) continue;
    }
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
