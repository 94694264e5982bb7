// hh_near_tc.cu -- SURVEY 8(a) rows 6 and 8 on the 5th-generation tensor cores (near_path = 1 / 2; north_star: "near-field
// pair MLP evaluation as a dense contraction on tcgen05 tensor cores (TMA-staged weights, fp32 accumulate) only if it stays
// inside the stated tolerance").  Same work decomposition as k_near (hh_near.cu): one CTA per target leaf walks that leaf's
// source leaves (P^H sorted by tau), the (target, source) pairs of a tile of sources are flattened over the threads.  What
// changes is the MLP (Eq. (4)): a CTA of 128 threads evaluates 128 entries at a time, one per thread, and
// the 32 x 32 hidden layer (71 % of the multiply-adds) is ONE tensor-core contraction per 128 entries:
//
//   layer 1 (4 -> 32)    FFMA + tanh in registers, h1 written to shared memory as the A operand (128 x 32, K-major,
//                        no-swizzle core-matrix layout), as tf32 (hi) and, with SPLIT, its tf32 remainder (lo)
//   layer 2 (32 -> 32)   tcgen05.mma.cta_group::1.kind::tf32, M = 128, N = 32, K = 8 per instruction, issued by one thread;
//                        B = W2 (tf32 hi / lo parts), pre-arranged in the core-matrix layout by hh_create and staged once
//                        per CTA by a TMA bulk copy (cp.async.bulk ... mbarrier::complete_tx); accumulator D in TENSOR
//                        MEMORY (128 lanes x 32 columns fp32).  SPLIT: D = Ahi Bhi + Alo Bhi + Ahi Blo ("3xTF32": the
//                        dropped Alo Blo term is 2^-22 relative), 12 instructions instead of 4
//   epilogue             tcgen05.ld (32 lanes x 32 columns per warp: thread t gets row t, i.e. its own entry back), + b2,
//                        tanh, layer 3 (32 -> 9) and the 1/r scaling on FFMA, apply to F_j, shared-memory atomics into U_i
//
// near_path = 1: tf32 operands as they are (10-bit mantissa) and MUFU tanh.approx -- the 2e-3 path of north_star.
// near_path = 2: SPLIT + the accurate tanhf -- fp32-class entries with the contraction still on the tensor pipe.
// The tensor pipe is nearly idle either way (128 x 32 x 32 MACs per 128 entries); what the variant buys is the ~1,000
// FFMA per entry that no longer issue from the ALUs.
#include "hh_mlp.cuh"

#define NT_T 128               /* threads per CTA = rows of one MMA tile                                  */
#ifndef NT_TANH2
#define NT_TANH2(x) tanh_ex2(x) /* activation of near_path = 2 (-DNT_TANH2=tanhf for the library tanh)     */
#endif
#define NT_TILE 256            /* source particles staged per tile                                        */
#define NT_SPIN_MAX (1u << 24) /* bounded mbarrier spins: a wrong descriptor must not hang the GPU         */

template <int NP>              /* NP = 1: tf32 operands as they are, NP = 2: hi + lo parts (split operands) */
struct NtSmem {
  float A[NP][128 * 32];       /* h1 tile, hi / lo: element (row r, k) at (r/8)*256 + (k/4)*32 + (r%8)*4 + (k%4) */
  float B[NP][32 * 32];        /* W2 hi / lo in the same layout with n (output unit) as the row             */
  float w1[32 * 4], b1[32], b2[32], w3t[32 * 12], b3[12];
  float tX[HH_MAX_LEAF * 3], sU[HH_MAX_LEAF * 3];
  float sXj[NT_TILE * 3], sFj[NT_TILE * 3];
  u32 sJ[NT_TILE];
  u32 segStart[33], segLo[32];
  u32 s_nb, tmem_base;
  unsigned long long mbar_mma, mbar_tma;
};

__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ u32 to_tf32(float x) { u32 r; asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x)); return r; }
__device__ __forceinline__ float tanh_mufu(float x) { float y; asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// tanh x = 1 - 2 / (1 + 2^(2 x log2 e)) with MUFU ex2 and rcp (2 ulp each): ABSOLUTE error ~2e-7 everywhere (the subtraction cancels
// for small |x|, so the relative error of tiny values is not kept).  Five instructions instead of tanhf's ~20.  Good for the
// near-field, where an activation feeds a dot product and only its absolute error matters; NOT used inside Alg. 2, where entry
// errors are amplified by the pivot conditioning.  Saturates correctly: ex2 -> inf gives 1, ex2 -> 0 gives -1.
__device__ __forceinline__ float tanh_ex2(float x) {
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(x * 2.8853900817779268f));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(e + 1.0f));
  return fmaf(r, -2.0f, 1.0f);
}

// K-major, no-swizzle shared-memory matrix descriptor: 8-row x 16-byte core matrices, the two K-halves of one instruction
// 128 B apart (leading byte offset), consecutive 8-row groups 1024 B apart (stride byte offset), descriptor version 1.
__device__ __forceinline__ unsigned long long umma_desc(u32 saddr) {
  return (unsigned long long)((saddr & 0x3ffffu) >> 4) | (8ull << 16) | (64ull << 32) | (1ull << 46);
}
// kind::tf32 instruction descriptor: D fp32, A and B tf32, both K-major, N = 32, M = 128
#define NT_IDESC ((1u << 4) | (2u << 7) | (2u << 10) | ((32u >> 3) << 17) | ((128u >> 4) << 24))

__device__ __forceinline__ void umma_tf32(u32 tmem_d, unsigned long long da, unsigned long long db, u32 accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t"
      "}\n" ::"r"(tmem_d), "l"(da), "l"(db), "r"(NT_IDESC), "r"(accumulate), "r"(0u)
      : "memory");
}
__device__ __forceinline__ bool mbar_wait(u32 bar, u32 parity) {
  for (u32 spin = 0; spin < NT_SPIN_MAX; ++spin) {
    u32 ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return true;
  }
  return false;
}

// Software pipeline over the 128-entry tiles of a CTA (two accumulators in tensor memory, one A buffer):
//   layer 1 of tile n in registers | wait MMA(n-1) | write A | sync | issue MMA(n) -> D[n & 1] | epilogue of tile n-1 from D[(n-1) & 1]
// so the tensor-core latency of a tile hides behind the epilogue of the one before and layer 1 of the one after.
template <bool SPLIT>
__global__ void __launch_bounds__(NT_T) k_near_tc(const float* __restrict__ gw, const float* __restrict__ gw2tc, float a,
                                                   const u32* __restrict__ leaf_nodes, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                   const uint2* __restrict__ PH, const u32* __restrict__ near_begin, const u32* __restrict__ near_end,
                                                   const float* __restrict__ Xs, const float* __restrict__ Fs, float* __restrict__ Us, u32* __restrict__ err_flag) {
  extern __shared__ __align__(1024) unsigned char nt_raw[];
  typedef NtSmem<SPLIT ? 2 : 1> Smem;
  Smem& S = *reinterpret_cast<Smem*>(nt_raw);
  typedef MlpOff<HH_MLP2_INP, HH_MLP2_H> O;
  const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const u32 node = leaf_nodes[blockIdx.x];
  const u32 tlo = nlo[node], m = nhi[node] - tlo;
  const u32 bar_mma = smem_u32(&S.mbar_mma), bar_tma = smem_u32(&S.mbar_tma);

  // ---- one-time setup: tensor memory (2 accumulators of 32 columns), barriers, W2 by TMA bulk copy, the small layers ----
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" ::"r"(smem_u32(&S.tmem_base)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_mma) : "memory");
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_tma) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const u32 bytes = (SPLIT ? 2u : 1u) * 32u * 32u * 4u;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_tma), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(&S.B[0][0])), "l"(gw2tc),
                 "r"(bytes), "r"(bar_tma)
                 : "memory");
  }
  for (u32 t = tid; t < 32 * 4; t += NT_T) S.w1[t] = gw[O::W1 + t];
  for (u32 t = tid; t < 32; t += NT_T) { S.b1[t] = gw[O::B1 + t]; S.b2[t] = gw[O::B2 + t]; }
  for (u32 t = tid; t < 32 * 12; t += NT_T) S.w3t[t] = gw[O::W3 + t];
  if (tid < 12) S.b3[tid] = gw[O::B3 + tid];
  for (u32 t = tid; t < 3 * m; t += NT_T) { S.tX[t] = Xs[3 * (size_t)tlo + t]; S.sU[t] = 0.f; }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const u32 tmem_d = S.tmem_base;
  bool alive = mbar_wait(bar_tma, 0);
  u32 phase = 0, ntile = 0;                        // ntile counts the MMAs issued by this CTA: accumulator ntile & 1

  // epilogue of one tile: accumulator -> registers, + b2, tanh, layer 3, 1/r, apply (S-3), shared-memory atomics into U_i
  auto epilogue = [&](u32 acc_idx, bool valid, u32 ii, u32 jj, float inv) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    u32 dr[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, "
        "%21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(dr[0]), "=r"(dr[1]), "=r"(dr[2]), "=r"(dr[3]), "=r"(dr[4]), "=r"(dr[5]), "=r"(dr[6]), "=r"(dr[7]), "=r"(dr[8]), "=r"(dr[9]),
          "=r"(dr[10]), "=r"(dr[11]), "=r"(dr[12]), "=r"(dr[13]), "=r"(dr[14]), "=r"(dr[15]), "=r"(dr[16]), "=r"(dr[17]), "=r"(dr[18]),
          "=r"(dr[19]), "=r"(dr[20]), "=r"(dr[21]), "=r"(dr[22]), "=r"(dr[23]), "=r"(dr[24]), "=r"(dr[25]), "=r"(dr[26]), "=r"(dr[27]),
          "=r"(dr[28]), "=r"(dr[29]), "=r"(dr[30]), "=r"(dr[31])
        : "r"(tmem_d + ((warp * 32u) << 16) + acc_idx * 32u)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    float out[9];
#pragma unroll
    for (int r = 0; r < 9; ++r) out[r] = S.b3[r];
#pragma unroll
    for (int o = 0; o < 32; ++o) {
      const float pre = __uint_as_float(dr[o]) + S.b2[o];
      const float t = SPLIT ? NT_TANH2(pre) : tanh_mufu(pre);
      const float4 wa = *reinterpret_cast<const float4*>(&S.w3t[12 * o]);
      const float4 wb = *reinterpret_cast<const float4*>(&S.w3t[12 * o + 4]);
      const float wc = S.w3t[12 * o + 8];
      out[0] = fmaf(wa.x, t, out[0]); out[1] = fmaf(wa.y, t, out[1]); out[2] = fmaf(wa.z, t, out[2]);
      out[3] = fmaf(wa.w, t, out[3]); out[4] = fmaf(wb.x, t, out[4]); out[5] = fmaf(wb.y, t, out[5]);
      out[6] = fmaf(wb.z, t, out[6]); out[7] = fmaf(wb.w, t, out[7]); out[8] = fmaf(wc, t, out[8]);
    }
    if (valid && tlo + ii != S.sJ[jj]) {                                   // S-5: the pair i == j is skipped
      const float f0 = S.sFj[3 * jj], f1 = S.sFj[3 * jj + 1], f2 = S.sFj[3 * jj + 2];
#pragma unroll
      for (int al = 0; al < 3; ++al)
        atomicAdd(&S.sU[3 * ii + al], inv * fmaf(out[3 * al], f0, fmaf(out[3 * al + 1], f1, out[3 * al + 2] * f2)));
    }
  };

  u32 b = near_begin[node];
  const u32 bend = near_end[node];
  while (b < bend) {
    if (warp == 0) {
      u32 blk = b + lane;
      u32 lo = 0, sz = 0;
      if (blk < bend) { u32 sg = PH[blk].y; lo = nlo[sg]; sz = nhi[sg] - lo; }
      u32 inc = sz;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { u32 t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (u32)o) inc += t; }
      bool fits = blk < bend && inc <= NT_TILE;
      u32 nb = __popc(__ballot_sync(0xffffffffu, fits));
      S.segStart[lane] = inc - sz;
      S.segLo[lane] = lo;
      if (lane == nb - 1) S.segStart[nb] = inc;
      if (lane == 0) S.s_nb = nb;
    }
    __syncthreads();
    const u32 nb = S.s_nb, nt = S.segStart[nb];
    for (u32 s = tid; s < nt; s += NT_T) {
      u32 g = 0;
      while (g + 1 < nb && S.segStart[g + 1] <= s) ++g;
      u32 j = S.segLo[g] + (s - S.segStart[g]);
      S.sJ[s] = j;
#pragma unroll
      for (int c = 0; c < 3; ++c) { S.sXj[3 * s + c] = Xs[3 * (size_t)j + c]; S.sFj[3 * s + c] = Fs[3 * (size_t)j + c]; }
    }
    __syncthreads();
    const u32 pairs = m * nt;
    bool pend = false, p_valid = false;                                  // the tile whose MMA is in flight
    u32 p_ii = 0, p_jj = 0;
    float p_inv = 0.f;
    for (u32 p0 = 0; p0 < pairs; p0 += NT_T) {
      const u32 p = p0 + tid;
      const bool valid = p < pairs;
      const u32 pc = valid ? p : 0u;
      const u32 jj = pc / m, ii = pc - jj * m;
      // ---- features and layer 1 (S-1, S-2, S-4), in registers: overlaps the MMA of the previous tile ----
      float x[4], inv;
      {
        const float rx = S.sXj[3 * jj] - S.tX[3 * ii], ry = S.sXj[3 * jj + 1] - S.tX[3 * ii + 1], rz = S.sXj[3 * jj + 2] - S.tX[3 * ii + 2];
        float d = sqrtf(fmaf(rx, rx, fmaf(ry, ry, rz * rz)));
        d = fmaxf(d, 1e-12f * a);
        inv = 1.0f / d;
        x[0] = rx * inv; x[1] = ry * inv; x[2] = rz * inv; x[3] = a * inv;
      }
      float h[32];
#pragma unroll
      for (int o = 0; o < 32; ++o) {
        const float4 w = *reinterpret_cast<const float4*>(&S.w1[4 * o]);
        const float pre = fmaf(w.x, x[0], fmaf(w.y, x[1], fmaf(w.z, x[2], fmaf(w.w, x[3], S.b1[o]))));
        h[o] = SPLIT ? NT_TANH2(pre) : tanh_mufu(pre);
      }
      // ---- the previous MMA has read A: wait for it, then publish this tile's A operand ----
      if (pend) { alive = alive && mbar_wait(bar_mma, phase); phase ^= 1u; }
      float* Ahi = &S.A[0][(tid >> 3) * 256 + (tid & 7) * 4];
      float* Alo = &S.A[SPLIT ? 1 : 0][(tid >> 3) * 256 + (tid & 7) * 4];
#pragma unroll
      for (int kc = 0; kc < 8; ++kc) {
        float4 hi, lo;
        hi.x = __uint_as_float(to_tf32(h[4 * kc])); hi.y = __uint_as_float(to_tf32(h[4 * kc + 1]));
        hi.z = __uint_as_float(to_tf32(h[4 * kc + 2])); hi.w = __uint_as_float(to_tf32(h[4 * kc + 3]));
        *reinterpret_cast<float4*>(Ahi + kc * 32) = hi;
        if (SPLIT) {
          lo.x = __uint_as_float(to_tf32(h[4 * kc] - hi.x)); lo.y = __uint_as_float(to_tf32(h[4 * kc + 1] - hi.y));
          lo.z = __uint_as_float(to_tf32(h[4 * kc + 2] - hi.z)); lo.w = __uint_as_float(to_tf32(h[4 * kc + 3] - hi.w));
          *reinterpret_cast<float4*>(Alo + kc * 32) = lo;
        }
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // generic-proxy writes of A -> visible to the MMA
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");       // orders earlier tcgen05.ld of this accumulator before the MMA
      __syncthreads();
      // ---- layer 2 on the tensor core: D[ntile & 1] = A W2^T ----
      if (tid == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const u32 d_addr = tmem_d + (ntile & 1u) * 32u;
        const u32 a_hi = smem_u32(&S.A[0][0]), a_lo = smem_u32(&S.A[SPLIT ? 1 : 0][0]), b_hi = smem_u32(&S.B[0][0]), b_lo = smem_u32(&S.B[SPLIT ? 1 : 0][0]);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) umma_tf32(d_addr, umma_desc(a_hi + kk * 256), umma_desc(b_hi + kk * 256), kk > 0);
        if (SPLIT) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) umma_tf32(d_addr, umma_desc(a_lo + kk * 256), umma_desc(b_hi + kk * 256), 1u);
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) umma_tf32(d_addr, umma_desc(a_hi + kk * 256), umma_desc(b_lo + kk * 256), 1u);
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar_mma) : "memory");
      }
      // ---- epilogue of the previous tile (its accumulator was complete at the wait above): overlaps this MMA ----
      if (pend) epilogue((ntile - 1u) & 1u, p_valid, p_ii, p_jj, p_inv);
      pend = true; p_valid = valid; p_ii = ii; p_jj = jj; p_inv = inv;
      ++ntile;
    }
    if (pend) {                                                            // drain: the staged sources are about to be replaced
      alive = alive && mbar_wait(bar_mma, phase);
      phase ^= 1u;
      epilogue((ntile - 1u) & 1u, p_valid, p_ii, p_jj, p_inv);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    b += nb;
  }
  for (u32 t = tid; t < 3 * m; t += NT_T) atomicAdd(&Us[3 * (size_t)tlo + t], S.sU[t]);
  if (!alive && tid == 0) atomicExch(err_flag, 1u);
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" ::"r"(tmem_d) : "memory");
}

// W2 as the B operand of the contraction: tf32 hi part and tf32 remainder, both in the K-major core-matrix layout of the
// header comment (n = output unit is the row).  Called by hh_create; `out` holds 2 x 1024 floats.
void hh_pack_w2_tc(const float* W2 /* [32][32] row-major [out][in] */, float* out) {
  auto rna = [](float v) {                                          // cvt.rna.tf32.f32: nearest, ties away from zero
    u32 bits;
    memcpy(&bits, &v, 4);
    bits = (bits + 0x1000u) & 0xffffe000u;
    float r;
    memcpy(&r, &bits, 4);
    return r;
  };
  for (int n = 0; n < 32; ++n)
    for (int k = 0; k < 32; ++k) {
      const float w = W2[n * 32 + k], hi = rna(w), lo = rna(w - hi);
      const int idx = (n / 8) * 256 + (k / 4) * 32 + (n % 8) * 4 + (k % 4);
      out[idx] = hi;
      out[1024 + idx] = lo;
    }
}

int hh_near_apply_tc(hh_ctx* ctx) {
  if (ctx->n_leaves <= 0 || ctx->nH <= 0) return HH_OK;
  const size_t smem = (ctx->p.near_path == 2 ? sizeof(NtSmem<2>) : sizeof(NtSmem<1>)) + 1024;
  cudaStream_t s = ctx->stream;
  HH_CUDA(cudaMemsetAsync(&ctx->d_sc->deg_overflow, 0, sizeof(u32), s));   // doubles as the kernel's error flag
  if (ctx->p.near_path == 2) {
    HH_CUDA(cudaFuncSetAttribute(k_near_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_near_tc<true><<<HH_N + ctx->n_leaves, NT_T, smem, s>>>(ctx->w2, ctx->w2tc, ctx->p.radius_a, ctx->leaf_nodes, ctx->nlo, ctx->nhi, ctx->PH, ctx->near_begin,
                                                             ctx->near_end, ctx->Xs, ctx->Fs, ctx->Us, &ctx->d_sc->deg_overflow);
  } else {
    HH_CUDA(cudaFuncSetAttribute(k_near_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_near_tc<false><<<HH_N + ctx->n_leaves, NT_T, smem, s>>>(ctx->w2, ctx->w2tc, ctx->p.radius_a, ctx->leaf_nodes, ctx->nlo, ctx->nhi, ctx->PH, ctx->near_begin,
                                                              ctx->near_end, ctx->Xs, ctx->Fs, ctx->Us, &ctx->d_sc->deg_overflow);
  }
  HH_LAUNCH_CHECK();
  HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->deg_overflow, &ctx->d_sc->deg_overflow, sizeof(u32), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  if (ctx->h_sc->deg_overflow) return hh_fail(ctx, HH_ERR_CUDA, "near-field tensor-core path: an mbarrier wait timed out (MMA or TMA never completed)");
  return HH_OK;
}
