// hh_aca.cu -- SURVEY 8(a) row 7: Alg. 2 (Eqs. (8)-(10), L196-L205) with 3x3 entries,
// one CTA per admissible block, entries evaluated on demand by the two-body MLP (L262 lines 4, 7).
//
// Storage is the listing's: rank term k keeps the normalised column c_k(i) = E_{k-1}(i, j_k) P^{-1} with
// P = E_{k-1}(i_k, j_k) (line 6, so c_k(i_k) = I) and the raw residual row q_k(j) = E_{k-1}(i_k, j).  The
// 3x3 inverse and the products c'(i) P^{-1} are taken in fp64 and rounded once: with an fp32 inverse the
// factor (and every later apply) loses cond(P) * 2^-24, which breaks the 1e-5 bar.
// nu^2 and the lambda^2 recursion (S-19):
//   nu^2   = tr(A_kk B_kk),  A_pk = sum_i C_p(i)^T c_k(i),  B_kp = sum_j q_k(j) Q_p(j)^T
//   cross  = sum_p tr(A_pk B_kp) = sum_j tr( [sum_p Q_p(j)^T A_pk] q_k(j) )        (one scalar reduction)
// Factors live in the arena in chunks of HH_RC ranks, plane-major: C part [r][e][m_pad], Q part [r][e][n_pad].
#include "hh_mlp.cuh"

struct AcaArgs {
  const float* w2; float a; float tol; int max_rank; int rule; double kappa_max, dense_cap;
  const uint2* PG; const u32 *nlo, *nhi; const float* Xs;
  float* arena; u64 arena_units; u32* tab; DevScalars* sc;
  int *ranks, *flags;
  u32 first;      // first block of the batch (table row 0)
  u32 begin;      // first block of this launch
};

__device__ __forceinline__ u32 pad8u(u32 v) { return (v + 7u) & ~7u; }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// arg-max with ties -> lowest index (S-18)
__device__ __forceinline__ void amax_merge(float& s, int& i, float s2, int i2) {
  if (i2 >= 0 && (i < 0 || s2 > s || (s2 == s && i2 < i))) { s = s2; i = i2; }
}
__device__ __forceinline__ void warp_amax(float& s, int& i) {
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    float s2 = __shfl_xor_sync(0xffffffffu, s, o);
    int i2 = __shfl_xor_sync(0xffffffffu, i, o);
    amax_merge(s, i, s2, i2);
  }
}

struct AcaSmem {
  float sw[HH_MLP2_FLOATS];
  double sPinvD[9];               // P^{-1} in fp64
  float sQj[HH_MAX_RANK * 9];     // Q_p(j_k),  p < k
  float sCi[HH_MAX_RANK * 9];     // C_p(i_k),  p < k
  float sA[HH_MAX_RANK * 9];      // A_pk,      p < k
  float sAkk[9], sP[9], sPinv[9];
  float red[4];                   // cross, nu2
  float wsc[2][8]; int wid[2][8]; // per-warp arg-max (det, fro)
  int piv_i[HH_MAX_RANK], piv_j[HH_MAX_RANK];
  u32 chunk[HH_MAX_CHUNKS];
  int ctl[4];                     // [0] pivot index, [1] status, [2] next column
};

template <int T>
__device__ __forceinline__ void block_amax2(AcaSmem& S, float& sd, int& id, float& sf, int& jf) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  warp_amax(sd, id);
  warp_amax(sf, jf);
  if (lane == 0) { S.wsc[0][w] = sd; S.wid[0][w] = id; S.wsc[1][w] = sf; S.wid[1][w] = jf; }
  __syncthreads();
  sd = S.wsc[0][0]; id = S.wid[0][0]; sf = S.wsc[1][0]; jf = S.wid[1][0];
#pragma unroll
  for (int q = 1; q < T / 32; ++q) { amax_merge(sd, id, S.wsc[0][q], S.wid[0][q]); amax_merge(sf, jf, S.wsc[1][q], S.wid[1][q]); }
  __syncthreads();
}

template <int T>
__global__ void __launch_bounds__(T, T >= 256 ? 1 : 384 / T) k_aca(AcaArgs A) {
  __shared__ __align__(16) AcaSmem S;
  const int tid = threadIdx.x, lane = tid & 31;
  const u32 g = A.begin + blockIdx.x;
  const uint2 blk = A.PG[g];
  const u32 tlo = A.nlo[blk.x], m = A.nhi[blk.x] - tlo;
  const u32 slo = A.nlo[blk.y], n = A.nhi[blk.y] - slo;
  const u32 mp = pad8u(m), np = pad8u(n);
  const u32 chunk_units = 9u * (mp + np) / 8u;                 // HH_RC * 9 * (mp + np) floats / 32
  const int kmax = min(min((int)m, (int)n), A.max_rank);
  u32* tabrow = A.tab + (size_t)(g - A.first) * HH_TAB_STRIDE;
  load_weights(S.sw, A.w2, HH_MLP2_FLOATS);
  if (tid < 4) S.ctl[tid] = 0;
  __syncthreads();

  float lam2 = 0.f;
  int rank = 0, flag = 0, jk = 0;                              // S-17: j_1 = 0
  bool met = false;
  for (int k = 0; k < kmax; ++k) {
    // ---- arena space for ranks k .. k+HH_RC-1 (plus the pivot record with the first chunk) ----
    if ((k % HH_RC) == 0) {
      if (tid == 0) {
        u32 need = chunk_units + (k == 0 ? 6u : 0u);
        u64 off = atomicAdd((unsigned long long*)&A.sc->arena_cursor, (unsigned long long)need);
        if (off + need > A.arena_units) {
          S.ctl[1] = -1;
        } else {
          if (k == 0) { tabrow[HH_TAB_PIV] = (u32)off; off += 6; }
          S.chunk[k / HH_RC] = (u32)off;
        }
      }
      __syncthreads();
      if (S.ctl[1] < 0) {                                       // arena full: this block is redone in the next batch
        if (tid == 0) atomicMin(&A.sc->fail_min, g);
        return;
      }
    }
    float* Ck = A.arena + (size_t)S.chunk[k / HH_RC] * HH_UNIT_FLOATS + (size_t)(k % HH_RC) * 9 * mp;
    float* Qk = A.arena + (size_t)S.chunk[k / HH_RC] * HH_UNIT_FLOATS + (size_t)HH_RC * 9 * mp + (size_t)(k % HH_RC) * 9 * np;
    if (tid == 0) S.piv_j[k] = jk;
    for (int t = tid; t < 9 * k; t += T) {
      int p = t / 9, e = t - 9 * p;
      const float* Qp = A.arena + (size_t)S.chunk[p / HH_RC] * HH_UNIT_FLOATS + (size_t)HH_RC * 9 * mp + (size_t)(p % HH_RC) * 9 * np;
      S.sQj[t] = Qp[(size_t)e * np + jk];
      S.sA[t] = 0.f;
    }
    if (tid < 9) S.sAkk[tid] = 0.f;
    if (tid < 4) S.red[tid] = 0.f;
    __syncthreads();

    // ---- line 4: column residual c'_k(i) = G(i, j_k) - sum_p C_p(i) Qt_p(j_k); line 5: row pivot ----
    float bd = -1.f, bf = -1.f;
    int bdi = -1, bfi = -1;
    float xs[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) xs[c] = A.Xs[3 * (size_t)(slo + jk) + c];
    for (u32 base = 0; base < m; base += 2 * T) {
      u32 ii[2] = {base + tid, base + tid + T};
      bool ok[2] = {ii[0] < m, ii[1] < m};
      float xi[2][3], xj[2][3], c[2][9];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        u32 ic = ok[e] ? ii[e] : m - 1;
#pragma unroll
        for (int d = 0; d < 3; ++d) { xi[e][d] = A.Xs[3 * (size_t)(tlo + ic) + d]; xj[e][d] = xs[d]; }
      }
      entry2_eval<2>(S.sw, A.a, xi, xj, c);
      for (int p = 0; p < k; ++p) {
        const float* Cp = A.arena + (size_t)S.chunk[p / HH_RC] * HH_UNIT_FLOATS + (size_t)(p % HH_RC) * 9 * mp;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          if (ok[e]) {
            float cp[9];
#pragma unroll
            for (int r = 0; r < 9; ++r) cp[r] = Cp[(size_t)r * mp + ii[e]];
            submul33(c[e], cp, &S.sQj[9 * p]);
          }
        }
      }
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (ok[e]) {
#pragma unroll
          for (int r = 0; r < 9; ++r) Ck[(size_t)r * mp + ii[e]] = c[e][r];      // raw residual; normalised in pass 2
          bool used = false;
          for (int q = 0; q < k; ++q) used |= (S.piv_i[q] == (int)ii[e]);
          if (!used) {
            amax_merge(bd, bdi, fabsf(det33(c[e])), (int)ii[e]);
            amax_merge(bf, bfi, fro2_33(c[e]), (int)ii[e]);
          }
        }
      }
    }
    block_amax2<T>(S, bd, bdi, bf, bfi);
    // S-18: |det| rule falls back to Frobenius when every remaining |det| is 0; rule 1 = Frobenius
    int ik;
    float best;
    if (A.rule == 0) { if (bd > 0.f || bf <= 0.f) { ik = bdi; best = bd; } else { ik = bfi; best = bf; } }
    else { ik = bfi; best = bf; }
    if (ik < 0 || !(best > 0.f)) { met = true; break; }         // S-21: zero residual column -> block reproduced
    // pivot block P = c'_k(i_k) and its inverse (adjugate / det)
    if (tid < 9) S.sP[tid] = Ck[(size_t)tid * mp + ik];
    for (int t = tid; t < 9 * k; t += T) {
      int p = t / 9, e = t - 9 * p;
      const float* Cp = A.arena + (size_t)S.chunk[p / HH_RC] * HH_UNIT_FLOATS + (size_t)(p % HH_RC) * 9 * mp;
      S.sCi[t] = Cp[(size_t)e * mp + ik];
    }
    __syncthreads();
    if (tid == 0) {
      double P[9];
#pragma unroll
      for (int r = 0; r < 9; ++r) P[r] = (double)S.sP[r];
      const double dP = P[0] * (P[4] * P[8] - P[5] * P[7]) - P[1] * (P[3] * P[8] - P[5] * P[6]) + P[2] * (P[3] * P[7] - P[4] * P[6]);
      if (fabs(dP) < 1e-30) {
        S.ctl[1] = 2;
      } else {
        const double iv = 1.0 / dP;
        S.sPinvD[0] = (P[4] * P[8] - P[5] * P[7]) * iv; S.sPinvD[1] = (P[2] * P[7] - P[1] * P[8]) * iv;
        S.sPinvD[2] = (P[1] * P[5] - P[2] * P[4]) * iv; S.sPinvD[3] = (P[5] * P[6] - P[3] * P[8]) * iv;
        S.sPinvD[4] = (P[0] * P[8] - P[2] * P[6]) * iv; S.sPinvD[5] = (P[2] * P[3] - P[0] * P[5]) * iv;
        S.sPinvD[6] = (P[3] * P[7] - P[4] * P[6]) * iv; S.sPinvD[7] = (P[1] * P[6] - P[0] * P[7]) * iv;
        S.sPinvD[8] = (P[0] * P[4] - P[1] * P[3]) * iv;
        double np2 = 0.0, ni2 = 0.0;
#pragma unroll
        for (int r = 0; r < 9; ++r) { np2 += P[r] * P[r]; ni2 += S.sPinvD[r] * S.sPinvD[r]; }
        if (sqrt(np2 * ni2) > A.kappa_max && (double)m * (double)n <= A.dense_cap * ((double)m + (double)n))
          S.ctl[1] = 2;                                           // S-18b: numerically singular at fp32 entry accuracy
      }
      S.piv_i[k] = ik;
    }
    __syncthreads();
    if (S.ctl[1] == 2) { flag = 2; break; }                     // S-18 / S-18b: breakdown -> the block is applied densely

    // ---- line 6: c_k(i) = c'_k(i) P^{-1} (fp64 products, rounded once); Gram matrices A_kk, A_pk (S-19) ----
    {
      double Pi[9];
#pragma unroll
      for (int r = 0; r < 9; ++r) Pi[r] = S.sPinvD[r];
      float akk[9];
#pragma unroll
      for (int e = 0; e < 9; ++e) akk[e] = 0.f;
      for (u32 base = 0; base < m; base += T) {
        const u32 i = base + tid;
        const bool ok = i < m;
        float c[9];
        if (ok) {
          float cr[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) cr[r] = Ck[(size_t)r * mp + i];              // written by this same thread in pass 1
#pragma unroll
          for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int s2 = 0; s2 < 3; ++s2)
              c[3 * r + s2] = (float)((double)cr[3 * r] * Pi[s2] + (double)cr[3 * r + 1] * Pi[3 + s2] + (double)cr[3 * r + 2] * Pi[6 + s2]);
#pragma unroll
          for (int r = 0; r < 9; ++r) Ck[(size_t)r * mp + i] = c[r];
#pragma unroll
          for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int s2 = 0; s2 < 3; ++s2) akk[3 * r + s2] += c[r] * c[s2] + c[3 + r] * c[3 + s2] + c[6 + r] * c[6 + s2];
        } else {
#pragma unroll
          for (int r = 0; r < 9; ++r) c[r] = 0.f;
        }
        for (int p = 0; p < k; ++p) {
          const float* Cp = A.arena + (size_t)S.chunk[p / HH_RC] * HH_UNIT_FLOATS + (size_t)(p % HH_RC) * 9 * mp;
          float acc[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) acc[r] = 0.f;
          if (ok) {
            float cp[9];
#pragma unroll
            for (int r = 0; r < 9; ++r) cp[r] = Cp[(size_t)r * mp + i];
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int s2 = 0; s2 < 3; ++s2) acc[3 * r + s2] = cp[r] * c[s2] + cp[3 + r] * c[3 + s2] + cp[6 + r] * c[6 + s2];
          }
#pragma unroll
          for (int r = 0; r < 9; ++r) {
            float v = warp_sum(acc[r]);
            if (lane == 0) atomicAdd(&S.sA[9 * p + r], v);
          }
        }
      }
#pragma unroll
      for (int r = 0; r < 9; ++r) {
        float v = warp_sum(akk[r]);
        if (lane == 0) atomicAdd(&S.sAkk[r], v);
      }
    }
    __syncthreads();

    // ---- line 7: row residual q_k(j) = G(i_k, j) - sum_p C_p(i_k) Q_p(j); line 8: next column; lines 9-10 ----
    bd = -1.f; bf = -1.f; bdi = -1; bfi = -1;
    float cross = 0.f, nu2 = 0.f;
    float xt[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) xt[c] = A.Xs[3 * (size_t)(tlo + ik) + c];
    for (u32 base = 0; base < n; base += 2 * T) {
      u32 jj[2] = {base + tid, base + tid + T};
      bool ok[2] = {jj[0] < n, jj[1] < n};
      float xi[2][3], xj[2][3], q[2][9];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        u32 jc = ok[e] ? jj[e] : n - 1;
#pragma unroll
        for (int d = 0; d < 3; ++d) { xi[e][d] = xt[d]; xj[e][d] = A.Xs[3 * (size_t)(slo + jc) + d]; }
      }
      entry2_eval<2>(S.sw, A.a, xi, xj, q);
      float Z[2][9];
#pragma unroll
      for (int e = 0; e < 2; ++e)
#pragma unroll
        for (int r = 0; r < 9; ++r) Z[e][r] = 0.f;
      for (int p = 0; p < k; ++p) {
        const float* Qp = A.arena + (size_t)S.chunk[p / HH_RC] * HH_UNIT_FLOATS + (size_t)HH_RC * 9 * mp + (size_t)(p % HH_RC) * 9 * np;
        const float* Ap = &S.sA[9 * p];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          if (ok[e]) {
            float qp[9];
#pragma unroll
            for (int r = 0; r < 9; ++r) qp[r] = Qp[(size_t)r * np + jj[e]];
            submul33(q[e], &S.sCi[9 * p], qp);
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int s = 0; s < 3; ++s)
                Z[e][3 * r + s] += qp[r] * Ap[s] + qp[3 + r] * Ap[3 + s] + qp[6 + r] * Ap[6 + s];
          }
        }
      }
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (ok[e]) {
          bool used = false;
          for (int t = 0; t <= k; ++t) used |= (S.piv_j[t] == (int)jj[e]);
          if (!used) {
            amax_merge(bd, bdi, fabsf(det33(q[e])), (int)jj[e]);
            amax_merge(bf, bfi, fro2_33(q[e]), (int)jj[e]);
          }
          float W[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) Qk[(size_t)r * np + jj[e]] = q[e][r];    // raw residual row (listing line 7)
          mul33(S.sAkk, q[e], W);
#pragma unroll
          for (int r = 0; r < 9; ++r) nu2 = fmaf(W[r], q[e][r], nu2);          // tr(A_kk q q^T)
#pragma unroll
          for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int s = 0; s < 3; ++s) cross = fmaf(Z[e][3 * r + s], q[e][3 * s + r], cross);   // tr(Z q)
        }
      }
    }
    for (u32 t = tid; t < 9 * (np - n); t += T) Qk[(size_t)(t / (np - n)) * np + n + t % (np - n)] = 0.f;   // zero the pad columns
    cross = warp_sum(cross);
    nu2 = warp_sum(nu2);
    if (lane == 0) { atomicAdd(&S.red[0], cross); atomicAdd(&S.red[1], nu2); }
    block_amax2<T>(S, bd, bdi, bf, bfi);
    cross = S.red[0];
    nu2 = S.red[1];
    lam2 += nu2 + 2.f * cross;
    rank = k + 1;
    // line 12 / Eq. (10): stop when nu <= zeta * lambda (S-20)
    const float nu = sqrtf(fmaxf(nu2, 0.f)), lam = sqrtf(fmaxf(lam2, 0.f));
    if (nu <= A.tol * lam) { met = true; break; }
    int jn;
    if (A.rule == 0) jn = (bd > 0.f || bf <= 0.f) ? bdi : bfi; else jn = bfi;
    if (jn < 0) { met = true; break; }
    jk = jn;
    __syncthreads();
  }
  if (!met && flag == 0 && rank == kmax && kmax < min((int)m, (int)n)) flag = 1;   // S-21: hit N_ite_max
  __syncthreads();
  // ---- record: rank, flag, chunk table, pivots ----
  if (tid == 0) { A.ranks[g] = rank; A.flags[g] = flag; }
  for (int t = tid; t < HH_MAX_CHUNKS; t += T) tabrow[t] = (t * HH_RC < rank) ? S.chunk[t] : 0xffffffffu;
  int* piv = (int*)(A.arena + (size_t)tabrow[HH_TAB_PIV] * HH_UNIT_FLOATS);
  // a breakdown (flag 2) also lists the attempted pivot after the accepted ones
  for (int t = tid; t < rank + (flag == 2 ? 1 : 0); t += T) { piv[t] = S.piv_i[t]; piv[HH_MAX_RANK + t] = S.piv_j[t]; }
}

// ------------------------------------------------------------------------------ batching (L246, L260)
// largest `end` such that blocks [first, end) fit the arena at the predicted number of chunks per block
__global__ void k_batch_range(const u64* __restrict__ unit_prefix, u32 first, u32 nG, u64 total_units, u32 chunks_pred,
                              DevScalars* sc) {
  u32 lo = first, hi = nG;                                       // invariant: [first, lo) fits
  const u64 s0 = unit_prefix[first];
  while (lo < hi) {
    u32 mid = lo + (hi - lo + 1) / 2;
    u64 need = (unit_prefix[mid] - s0) * 9ull / 8ull * chunks_pred + (u64)(mid - first) * 7ull;
    if (need <= total_units) lo = mid; else hi = mid - 1;
  }
  sc->batch_end = lo;
  sc->arena_cursor = 0;
  sc->fail_min = 0xffffffffu;
  sc->sum_rank = sc->aca_entries = sc->factor_bytes = 0;
  sc->not_conv = sc->singular = sc->max_rank_seen = 0;
  sc->n_dense = 0;
  sc->fallback_entries = 0;
}

__global__ void __launch_bounds__(256) k_batch_stats(const uint2* __restrict__ PG, const u32* __restrict__ nlo,
                                                      const u32* __restrict__ nhi, int* __restrict__ ranks,
                                                      const int* __restrict__ flags, u32 first, u32 next, u32 end,
                                                      u32* __restrict__ dense_list, DevScalars* sc) {
  u32 g = first + blockIdx.x * blockDim.x + threadIdx.x;
  u64 sr = 0, en = 0, fu = 0;
  u32 nc = 0, sg = 0, mr = 0;
  if (g < next) {
    uint2 p = PG[g];
    u64 mn = (u64)(nhi[p.x] - nlo[p.x]) + (nhi[p.y] - nlo[p.y]);
    int r = ranks[g];
    sr = (u64)r; en = (u64)r * mn; mr = (u32)r;
    nc = flags[g] == 1; sg = flags[g] == 2;
    fu = sg ? 0 : en;                                            // factor entries the far-field apply reads
    if (sg) {                                                    // S-18b: applied densely by hh_dense_apply
      dense_list[atomicAdd(&sc->n_dense, 1u)] = g;
      atomicAdd((unsigned long long*)&sc->fallback_entries, (unsigned long long)(nhi[p.x] - nlo[p.x]) * (nhi[p.y] - nlo[p.y]));
    }
  } else if (g < end) {
    ranks[g] = -1;                                               // factorised past the failure point: discarded
  }
  for (int o = 16; o; o >>= 1) {
    sr += __shfl_xor_sync(0xffffffffu, sr, o); en += __shfl_xor_sync(0xffffffffu, en, o);
    fu += __shfl_xor_sync(0xffffffffu, fu, o);
    nc += __shfl_xor_sync(0xffffffffu, nc, o); sg += __shfl_xor_sync(0xffffffffu, sg, o);
    mr = max(mr, __shfl_xor_sync(0xffffffffu, mr, o));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd((unsigned long long*)&sc->sum_rank, (unsigned long long)sr);
    atomicAdd((unsigned long long*)&sc->aca_entries, (unsigned long long)en);
    atomicAdd((unsigned long long*)&sc->factor_bytes, (unsigned long long)fu * 36ull);
    atomicAdd(&sc->not_conv, nc); atomicAdd(&sc->singular, sg); atomicMax(&sc->max_rank_seen, mr);
  }
}

int hh_aca_batch(hh_ctx* ctx, int64_t first, int64_t* next) {
  cudaStream_t s = ctx->stream;
  const u32 nG = (u32)ctx->nG;
  // the table (one 128-B row per resident block) sits at the start of the scratch region, the arena after it
  if (first == 0) ctx->l_pred = ctx->l_pred_first;
  u32 chunks_pred = (u32)((ctx->l_pred + HH_RC - 1) / HH_RC);
  if (chunks_pred < 1) chunks_pred = 1;
  if (chunks_pred > HH_MAX_CHUNKS) chunks_pred = HH_MAX_CHUNKS;
  const u64 total_units = ctx->scratch_bytes / 128;
  k_batch_range<<<HH_N + 1, 1, 0, s>>>(ctx->unit_prefix, (u32)first, nG, total_units > 8 ? total_units - 8 : 0, chunks_pred, ctx->d_sc);
  HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->batch_end, &ctx->d_sc->batch_end, sizeof(u32), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  u32 end = ctx->h_sc->batch_end;
  if (end <= first) end = (u32)first + 1;                        // try a single block; it fails below if it cannot fit
  const u32 nb = end - (u32)first;
  ctx->tab = (u32*)ctx->scratch;
  ctx->far_items = nullptr; ctx->far_cnt = nullptr; ctx->far_items_cap = 0;   // no room for an item list in this layout: k_far, one CTA per block
  size_t tab_bytes = ((size_t)nb * HH_TAB_STRIDE * sizeof(u32) + 127) / 128 * 128;
  if (tab_bytes + 4096 > ctx->scratch_bytes) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "factor arena too small");
  ctx->arena = (float*)(ctx->scratch + tab_bytes);
  ctx->arena_units = (ctx->scratch_bytes - tab_bytes) / 128;
  AcaArgs A;
  A.w2 = ctx->w2; A.a = ctx->p.radius_a; A.tol = ctx->p.aca_tol; A.max_rank = ctx->p.aca_max_rank; A.rule = ctx->p.pivot_rule;
  A.kappa_max = ctx->p.kappa_max > 0.f ? (double)ctx->p.kappa_max : (double)INFINITY;   // 0 = the plain listing (L221)
  A.dense_cap = ctx->p.dense_cap > 0.f ? (double)ctx->p.dense_cap : 128.0;
  A.PG = ctx->PG; A.nlo = ctx->nlo; A.nhi = ctx->nhi; A.Xs = ctx->Xs;
  A.arena = ctx->arena; A.arena_units = ctx->arena_units; A.tab = ctx->tab; A.sc = ctx->d_sc;
  A.ranks = ctx->ranks; A.flags = ctx->flags; A.first = (u32)first;
  for (int c = 0; c < 4; ++c) {                                  // size classes: max(m,n) > 256, <= 256, <= 128, <= 64
    u32 b = ctx->class_bound[c] > (u32)first ? ctx->class_bound[c] : (u32)first;
    u32 e = ctx->class_bound[c + 1] < end ? ctx->class_bound[c + 1] : end;
    if (b >= e) continue;
    A.begin = b;
    switch (c) {
      case 0: k_aca<256><<<HH_N + e - b, 256, 0, s>>>(A); break;
      case 1: k_aca<128><<<HH_N + e - b, 128, 0, s>>>(A); break;
      case 2: k_aca<64><<<HH_N + e - b, 64, 0, s>>>(A); break;
      default: k_aca<32><<<HH_N + e - b, 32, 0, s>>>(A); break;
    }
  }
  HH_LAUNCH_CHECK();
  return hh_aca_batch_finish(ctx, first, end, next);
}

// hh_set_capture: pivot records of the just-factorised blocks [first, next) whose target range holds a flagged row
__global__ void __launch_bounds__(128) k_capture(const uint2* __restrict__ PG, const u32* __restrict__ nlo, const u32* __restrict__ nhi,
                                                  const int* __restrict__ ranks, const int* __restrict__ flags, const u32* __restrict__ tab,
                                                  const float* __restrict__ arena, u32 first, u32 next, const int32_t* __restrict__ prefix,
                                                  int32_t* __restrict__ rec, unsigned long long cap, DevScalars* sc) {
  const u32 g = first + blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (g >= next) return;
  const u32 t = PG[g].x;
  if (prefix[nhi[t]] - prefix[nlo[t]] <= 0) return;
  unsigned long long slot = 0;
  if (lane == 0) slot = atomicAdd((unsigned long long*)&sc->cap_count, 1ull);
  slot = __shfl_sync(0xffffffffu, slot, 0);
  if (slot >= cap) return;
  const int r = ranks[g], f = flags[g];
  const int np = r + (f == 2 ? 1 : 0);                            // a breakdown also lists its attempted pivot
  int32_t* out = rec + (size_t)slot * HH_CAP_STRIDE;
  const int* piv = (const int*)(arena + (size_t)tab[(size_t)(g - first) * HH_TAB_STRIDE + HH_TAB_PIV] * HH_UNIT_FLOATS);
  if (lane == 0) { out[0] = (int32_t)g; out[1] = r; out[2] = f; out[3] = np; }
  for (int k = lane; k < HH_MAX_RANK; k += 32) {
    out[4 + k] = k < np ? piv[k] : -1;
    out[4 + HH_MAX_RANK + k] = k < np ? piv[HH_MAX_RANK + k] : -1;
  }
}

// shared by both ACA forms: batch boundary, counters, dense list (S-18b), rank prediction for the next batch
int hh_aca_batch_finish(hh_ctx* ctx, int64_t first, u32 end, int64_t* next) {
  cudaStream_t s = ctx->stream;
  const u32 nb = end - (u32)first;
  HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->fail_min, &ctx->d_sc->fail_min, sizeof(u32), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  u32 nx = ctx->h_sc->fail_min < end ? ctx->h_sc->fail_min : end;
  k_batch_stats<<<HH_N + cdiv(nb, 256), 256, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, (u32)first, nx, end,
                                                             ctx->dense_list, ctx->d_sc);
  if (ctx->cap_rec && nx > (u32)first)
    k_capture<<<HH_N + cdiv(nx - (u32)first, 4), 128, 0, s>>>(ctx->PG, ctx->nlo, ctx->nhi, ctx->ranks, ctx->flags, ctx->tab, ctx->arena, (u32)first, nx,
                                                              ctx->cap_prefix, ctx->cap_rec, (unsigned long long)ctx->cap_max, ctx->d_sc);
  HH_CUDA(cudaMemcpyAsync(ctx->h_sc, ctx->d_sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  const DevScalars& h = *ctx->h_sc;
  ctx->far_built = 0;
  if (h.aca_err) return hh_fail(ctx, HH_ERR_CUDA, "lock-step ACA (staged tiles): an mbarrier wait timed out");
  if (h.far_err) return hh_fail(ctx, HH_ERR_CUDA, h.far_err == 2 ? "far-field ring kernel: item list overflow (internal)" : "far-field ring kernel: an mbarrier wait timed out");
  if (ctx->mlp2_wide && h.deg_overflow) return hh_fail(ctx, HH_ERR_CUDA, "paper-size MLP entries (ACA): an mbarrier wait timed out");
  ctx->res_first = first;
  ctx->res_next = nx;
  *next = nx;
  if (nx <= first) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "factor arena cannot hold a single admissible block");
  ctx->st.sum_rank += (int64_t)h.sum_rank;
  ctx->st.aca_entries += (int64_t)h.aca_entries;
  ctx->st.factor_bytes += (int64_t)h.factor_bytes;
  ctx->st.aca_not_converged += h.not_conv;
  ctx->st.aca_singular += h.singular;
  ctx->st.fallback_entries += (int64_t)h.fallback_entries;
  ctx->n_dense = h.n_dense;
  ctx->st.aca_batches += 1;
  // next prediction: what this batch really used per predicted chunk, plus 10 %
  if (nx > first) {
    double mean_rank = (double)h.sum_rank / (double)(nx - first);
    double pred = (mean_rank + HH_RC) * 1.10;
    if (h.fail_min < end) pred = ctx->l_pred * 1.25 > pred ? ctx->l_pred * 1.25 : pred;
    ctx->l_pred = pred < HH_RC ? HH_RC : (pred > HH_MAX_RANK ? HH_MAX_RANK : pred);
    if (first == 0) ctx->l_pred_first = ctx->l_pred;
  }
  return HH_OK;
}

// ------------------------------------------------------------------------------ introspection
// Copies the factors of a resident block to the host, entry-major: C [rank][m][9], Q [rank][n][9] as stored
// (the listing's: C_k = normalised residual column with C_k(i_k) = I, Q_k = residual row).
int hh_factors_fetch(hh_ctx* ctx, int64_t block, int32_t* rank, int32_t* flag, int32_t cap_rank, int32_t* piv_i,
                     int32_t* piv_j, float* C, float* Q) {
  cudaStream_t s = ctx->stream;
  u32 row[HH_TAB_STRIDE];
  uint2 blk;
  int r = 0, f = 0;
  HH_CUDA(cudaMemcpyAsync(row, ctx->tab + (size_t)(block - ctx->res_first) * HH_TAB_STRIDE, sizeof row, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaMemcpyAsync(&blk, ctx->PG + block, sizeof blk, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaMemcpyAsync(&r, ctx->ranks + block, sizeof r, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaMemcpyAsync(&f, ctx->flags + block, sizeof f, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  u32 lohi[4];
  HH_CUDA(cudaMemcpyAsync(&lohi[0], ctx->nlo + blk.x, 4, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaMemcpyAsync(&lohi[1], ctx->nhi + blk.x, 4, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaMemcpyAsync(&lohi[2], ctx->nlo + blk.y, 4, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaMemcpyAsync(&lohi[3], ctx->nhi + blk.y, 4, cudaMemcpyDeviceToHost, s));
  HH_CUDA(cudaStreamSynchronize(s));
  const u32 m = lohi[1] - lohi[0], n = lohi[3] - lohi[2], mp = (m + 7) & ~7u, np = (n + 7) & ~7u;
  if (rank) *rank = r;
  if (flag) *flag = f;
  if (r < 0) return hh_fail(ctx, HH_ERR_INVALID_ARG, "block has not been factorised");
  int rr = r < cap_rank ? r : cap_rank;
  int np_ = r + (f == 2 ? 1 : 0);                                // a breakdown also lists its attempted pivot
  if (np_ > cap_rank) np_ = cap_rank;
  if (np_ > HH_MAX_RANK) np_ = HH_MAX_RANK;
  if ((piv_i || piv_j) && np_ > 0) {
    int piv[2 * HH_MAX_RANK];
    HH_CUDA(cudaMemcpyAsync(piv, ctx->arena + (size_t)row[HH_TAB_PIV] * HH_UNIT_FLOATS, sizeof piv, cudaMemcpyDeviceToHost, s));
    HH_CUDA(cudaStreamSynchronize(s));
    for (int k = 0; k < np_; ++k) { if (piv_i) piv_i[k] = piv[k]; if (piv_j) piv_j[k] = piv[HH_MAX_RANK + k]; }
  }
  if (C || Q) {
    float* tmp = (float*)malloc(sizeof(float) * 9 * (size_t)(mp > np ? mp : np));
    if (!tmp) return hh_fail(ctx, HH_ERR_INVALID_ARG, "host allocation failed");
    cudaError_t ce = cudaSuccess;
    for (int k = 0; k < rr && ce == cudaSuccess; ++k) {
      const float* base = ctx->arena + (size_t)row[k / HH_RC] * HH_UNIT_FLOATS;
      if (C) {
        ce = cudaMemcpyAsync(tmp, base + (size_t)(k % HH_RC) * 9 * mp, sizeof(float) * 9 * mp, cudaMemcpyDeviceToHost, s);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(s);
        if (ce != cudaSuccess) break;
        for (u32 i = 0; i < m; ++i) for (int e = 0; e < 9; ++e) C[((size_t)k * m + i) * 9 + e] = tmp[(size_t)e * mp + i];
      }
      if (Q) {
        ce = cudaMemcpyAsync(tmp, base + (size_t)HH_RC * 9 * mp + (size_t)(k % HH_RC) * 9 * np, sizeof(float) * 9 * np, cudaMemcpyDeviceToHost, s);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(s);
        if (ce != cudaSuccess) break;
        for (u32 j = 0; j < n; ++j) for (int e = 0; e < 9; ++e) Q[((size_t)k * n + j) * 9 + e] = tmp[(size_t)e * np + j];
      }
    }
    free(tmp);
    HH_CUDA(ce);
  }
  return HH_OK;
}
