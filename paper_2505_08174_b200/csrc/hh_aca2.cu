// hh_aca2.cu -- SURVEY 8(a) row 7, lock-step form: Alg. 2 (Eqs. (8)-(10)) run on ALL admissible
// blocks of an arena batch at once, one listing line per kernel, the way the paper's own implementation does it
// (L262: "lines 2-12 each a parallel_for over the selected blocks; lines 4, 7 = gather coords -> NN inference ->
// scatter into C / Q") -- done the B200 way: no coordinate matrices Y, Z and no separate inference call; the rows
// (line 4) resp. columns (line 7) of all active blocks are cut into 16-entry granules, the granules of one
// iteration form one flat, load-balanced work list, and the MLP is evaluated in registers exactly as in the
// near-field kernel (hh_mlp.cuh).  A 2^19-row top-level block and a 20-row leaf block cost the same per entry.
//
// One iteration k (all blocks in lock step; blocks drop out as they stop), the default form (hh_set_aca_impl 0):
//   k2_eval<rows>    line 4    raw entries G(i, j_k) into the slot of rank k (the MLP, two entries per thread)
//   k2_upd<rows>     line 4-5  c'(i) = G(i,j_k) - sum_p C_p(i) Q_p(j_k) (4 rows per thread, vector loads); arg-max scores
//                              (Eq. (9), S-18) by atomicMax; A'_pk = sum_i C_p(i)^T c'(i)
//   k2_piv           line 5-6  pivot row i_k, P = c'(i_k), P^-1 and cond_F(P) in fp64; zero column -> done (S-21); singular or
//                              cond_F > kappa_max -> breakdown, block goes dense (S-18, S-18b); A_pk = A'_pk P^-1
//   k2_eval<columns> line 7    raw entries G(i_k, j); and line 6 rides along: c_k(i) = c'(i) P^-1 (fp64 products, rounded
//                              once), A_kk = sum_i c_k(i)^T c_k(i) (S-19) -- memory-bound, hidden by this kernel's arithmetic
//   k2_upd<columns>  line 7-8  q_k(j) = G(i_k,j) - sum_p C_p(i_k) Q_p(j) (2 columns per thread); arg-max for j_{k+1};
//                              B_kk = sum_j q(j) q(j)^T, cross = sum_j tr([sum_p Q_p(j)^T A_pk] q(j))  (= sum_p tr(A_pk B_kp), S-19)
//   k2_fin           line 9-12 nu^2 = tr(A_kk B_kk); lambda^2 += nu^2 + 2 cross; stop test Eq. (10) (S-20);
//                              next column; arena space for the next HH_RC ranks
// k2_step is the fused form (entries and update in one kernel; hh_set_aca_impl 3, and the fp64 parity mode), k2_step_t the
// fused form with TMA-staged rank terms (2), a2_two_halves form 0 on two half-batches one listing line apart (4).
// Storage, arena chunks, table rows and the pivot record are those of hh_aca.cu (the far-field kernel reads both).
#include "hh_mlp.cuh"
#include "hh_wide.cuh"
#ifdef HH_PROF
#include <chrono>
#endif

#define GR 16                    /* entries per granule = half a warp                                   */
#define A2_T 256                 /* threads of the entry-evaluating kernels                              */
// One entry per thread at 80 registers (24 warps per SM) instead of two at 128 (16 warps): the weight loads from shared
// memory are no longer shared by two entries, but a third more warps are in flight to cover the loads of the stored rank
// terms.  Measured at c3 (ms_aca): 2 entries / 2 CTAs 5,485; 1 / 3: 5,067; 1 / 4 (64 registers, spills): 5,313.
#ifndef A2_E
#define A2_E 1                   /* entries per thread of k2_step (granules per warp = 2 * A2_E)          */
#endif
#ifndef A2_OCC
#define A2_OCC 3                 /* CTAs of k2_step per SM the register budget is cut for                 */
#endif

struct BlkState {                /* 64 bytes per block of the batch                                      */
  u32 tlo, slo, m, n;
  int k;                         /* step = number of accepted rank terms                                 */
  int jk, ik;                    /* current column / pivot row                                           */
  int status;                    /* 0 active, 1 done, 2 breakdown (dense), -1 arena space failed         */
  float lam2;
  int flag;
  int kmax;
  u32 pad[5];
};

struct A2Args {
  const float* w2; const double* w2d; float a; float tol; int rule; double kappa_max, dense_cap;
  const uint2* PG; const u32 *nlo, *nhi; const float* Xs;
  float* arena; u64 arena_units; u32* tab; DevScalars* sc;
  int *ranks, *flags;
  u32 first, nb;
  int R;                         /* rank cap of the context: accumulators hold R + 1 Gram slots          */
  BlkState* st; unsigned long long* amax; double* pinv; float* acc;
  u32 *cm, *cn; uint2 *gm, *gn;
  u32* nact;                     /* counter of the active blocks (k2_gran_count)                          */
};

__device__ __forceinline__ u32 a2_pad8(u32 v) { return (v + 7u) & ~7u; }
#define ACC_AKK 0                /* accumulators of a block: [0,9) A_kk, [9,18) B_kk, [18] cross term, 27 + 9p: A_pk    */
#define ACC_BKK 9
#define ACC_CROSS 18
#define ACC_APK 27
__device__ __forceinline__ int acc_stride(int R) { return ACC_APK + 9 * (R + 1); }
__device__ __forceinline__ float* chunk_ptr(const A2Args& A, const u32* tabrow, int p) {
  return A.arena + (size_t)tabrow[p / HH_RC] * HH_UNIT_FLOATS;
}
__device__ __forceinline__ unsigned long long amax_key(float score, u32 idx) {   // larger score wins, ties -> lowest index
  return ((unsigned long long)__float_as_uint(score) << 32) | (unsigned long long)(0xffffffffu - idx);
}
__device__ __forceinline__ float half_sum(float v) {                             // sum over the 16 lanes of a half-warp
#pragma unroll
  for (int o = 8; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// Sum 9 values over the 16 lanes of a half-warp with 15 shuffles (halving butterfly): on return lane l (l < 9) of the
// half-warp holds the total of v[l] in v[0].
__device__ __forceinline__ float half_sum9(const float (&in)[9], u32 l16) {
  float v[16];
#pragma unroll
  for (int r = 0; r < 9; ++r) v[r] = in[r];
#pragma unroll
  for (int r = 9; r < 16; ++r) v[r] = 0.f;
#pragma unroll
  for (int w = 8; w; w >>= 1) {
    const bool up = (l16 & w) != 0;
#pragma unroll
    for (int r = 0; r < w; ++r) {
      const float send = up ? v[r] : v[r + w], keep = up ? v[r + w] : v[r];
      v[r] = keep + __shfl_xor_sync(0xffffffffu, send, w);
    }
  }
  return v[0];
}
__device__ __forceinline__ unsigned long long half_max(unsigned long long v) {
#pragma unroll
  for (int o = 8; o; o >>= 1) { unsigned long long t = __shfl_xor_sync(0xffffffffu, v, o); v = t > v ? t : v; }
  return v;
}

// ---- arena space for ranks k .. k+HH_RC-1 of one block (plus the pivot record with the first chunk) ----
__device__ __forceinline__ bool a2_alloc(const A2Args& A, u32 b, const BlkState& s, int k) {
  const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
  const u32 chunk_units = 9u * (mp + np) / 8u;
  u32* tabrow = A.tab + (size_t)b * HH_TAB_STRIDE;
  const u32 need = chunk_units + (k == 0 ? 6u : 0u);
  u64 off = atomicAdd((unsigned long long*)&A.sc->arena_cursor, (unsigned long long)need);
  if (off + need > A.arena_units) { atomicMin(&A.sc->fail_min, A.first + b); return false; }
  if (k == 0) { tabrow[HH_TAB_PIV] = (u32)off; off += 6; }
  tabrow[k / HH_RC] = (u32)off;
  return true;
}
__device__ __forceinline__ int* a2_piv(const A2Args& A, u32 b) {
  return (int*)(A.arena + (size_t)A.tab[(size_t)b * HH_TAB_STRIDE + HH_TAB_PIV] * HH_UNIT_FLOATS);
}
__device__ __forceinline__ void a2_zero_acc(const A2Args& A, u32 b, int k) {      // slots used by step k
  float* acc = A.acc + (size_t)b * acc_stride(A.R);
  for (int t = 0; t < ACC_APK + 9 * k; ++t) acc[t] = 0.f;
  for (int t = 0; t < 4; ++t) A.amax[(size_t)b * 4 + t] = 0ull;
}
__device__ __forceinline__ void a2_finish(const A2Args& A, u32 b, BlkState& s, int status, int flag) {
  s.status = status; s.flag = flag;
  A.ranks[A.first + b] = s.k;
  A.flags[A.first + b] = flag;
  u32* tabrow = A.tab + (size_t)b * HH_TAB_STRIDE;
  for (int t = (s.k + HH_RC - 1) / HH_RC; t < HH_MAX_CHUNKS; ++t) tabrow[t] = 0xffffffffu;
}

__global__ void __launch_bounds__(256) k2_init(A2Args A) {
  const u32 b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= A.nb) return;
  const uint2 blk = A.PG[A.first + b];
  BlkState s;
  s.tlo = A.nlo[blk.x]; s.m = A.nhi[blk.x] - s.tlo;
  s.slo = A.nlo[blk.y]; s.n = A.nhi[blk.y] - s.slo;
  s.k = 0; s.jk = 0; s.ik = -1;                                   // S-17: j_1 = 0
  s.lam2 = 0.f; s.flag = 0; s.status = 0;
  s.kmax = min(min((int)s.m, (int)s.n), A.R);
  for (int t = 0; t < 5; ++t) s.pad[t] = 0;
  A.ranks[A.first + b] = -1; A.flags[A.first + b] = 0;
  if (!a2_alloc(A, b, s, 0)) s.status = -1;
  else { a2_piv(A, b)[HH_MAX_RANK] = 0; a2_zero_acc(A, b, 0); }
  A.st[b] = s;
}

// ---- granule lists of the iteration: one (block, first entry) pair per 16 rows resp. columns of every active block ----
__global__ void __launch_bounds__(256) k2_gran_count(A2Args A) {
  const u32 b = blockIdx.x * blockDim.x + threadIdx.x;
  u32 act = 0;
  if (b < A.nb) {
    const BlkState& s = A.st[b];
    act = s.status == 0;
    A.cm[b] = act ? (s.m + GR - 1) / GR : 0u;
    A.cn[b] = act ? (s.n + GR - 1) / GR : 0u;
  }
  act = __popc(__ballot_sync(0xffffffffu, act));
  if ((threadIdx.x & 31) == 0 && act) atomicAdd(A.nact, act);
}
__global__ void __launch_bounds__(256) k2_gran_fill(A2Args A) {                // one warp per block
  const u32 b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (b >= A.nb) return;
  const BlkState& s = A.st[b];
  if (s.status != 0) return;
  const u32 nm = (s.m + GR - 1) / GR, nn = (s.n + GR - 1) / GR, pm = A.cm[b], pn = A.cn[b];
  for (u32 t = lane; t < nm; t += 32) A.gm[pm + t] = make_uint2(b, t * GR);
  for (u32 t = lane; t < nn; t += 32) A.gn[pn + t] = make_uint2(b, t * GR);
}

// ---- line 6: c_k(i) = c'(i) P^-1 (fp64 products, rounded once); A_kk = sum_i c_k(i)^T c_k(i) (S-19).
// Half a warp per granule of rows; called by all 32 lanes (shuffles inside).  It is memory-bound and independent of
// the entry evaluation of the row side (line 7), so k2_step<true> interleaves it with its MLP tiles: the loads of one
// hide behind the arithmetic of the other.
__device__ __forceinline__ void a2_norm_granule(const A2Args& A, u32 gi, u32 count, u32 lane) {
  const u32 l16 = lane & 15;
  const bool gv = gi < count;
  const uint2 g = A.gm[gv ? gi : count - 1];
  const BlkState& s = A.st[g.x];
  const u32 i = g.y + l16, mp = a2_pad8(s.m);
  const bool ok = gv && s.status == 0 && i < s.m;
  const int k = s.k;
  const u32* tabrow = A.tab + (size_t)g.x * HH_TAB_STRIDE;
  float* acc = A.acc + (size_t)g.x * acc_stride(A.R);
  float c[9], akk[9];
#pragma unroll
  for (int r = 0; r < 9; ++r) { c[r] = 0.f; akk[r] = 0.f; }
  if (ok) {
    float* Ck = chunk_ptr(A, tabrow, k) + (size_t)(k % HH_RC) * 9 * mp;
    double Pi[9];
    float cr[9];
#pragma unroll
    for (int r = 0; r < 9; ++r) { Pi[r] = A.pinv[(size_t)g.x * 9 + r]; cr[r] = Ck[(size_t)r * mp + i]; }
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int q = 0; q < 3; ++q)
        c[3 * r + q] = (float)((double)cr[3 * r] * Pi[q] + (double)cr[3 * r + 1] * Pi[3 + q] + (double)cr[3 * r + 2] * Pi[6 + q]);
#pragma unroll
    for (int r = 0; r < 9; ++r) Ck[(size_t)r * mp + i] = c[r];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int q = 0; q < 3; ++q) akk[3 * r + q] = c[r] * c[q] + c[3 + r] * c[3 + q] + c[6 + r] * c[6 + q];
  }
  {
    const float t = half_sum9(akk, l16);
    const bool okh = __shfl_sync(0xffffffffu, ok, lane & 16);       // validity of the granule (its first row)
    if (l16 < 9 && okh) atomicAdd(&acc[l16], t);
  }
}


// ---- lines 4-5 (COLS = false: over the rows of tau, entries G(i, j_k)) resp. lines 7-8 (COLS = true: over the columns of
// sigma, entries G(i_k, j)) of all active blocks in ONE launch: entry evaluation by the MLP, residual against the stored
// rank terms, pivot scores, Gram sums.  A warp takes 4 granules: slot (e, half) -> granule 4*tile + 2*e + half; every thread
// evaluates two entries (the in-register MLP of hh_mlp.cuh) and keeps them in registers for the update, so a raw entry
// never travels through memory (round 1 ran entry evaluation and update as two launches with a 72-byte round trip per entry
// between them; same speed).  The update re-reads the k stored rank terms of its rows, 36 k bytes per
// row: the l^2 term of Alg. 2's cost.  An arena batch is far larger than L2, so these reads come from HBM:
// about 7 TB per mat-vec at c3, ten times the factors themselves, and the reason the ACA build is the longest stage.
// Measured and dropped: prefetching those lines into L2 before the MLP arithmetic (+5 %), staging them
// through shared memory with cp.async (+29 %), one loop over both slots (+22 %, spills).
// F64 (aca_precision = 1, parity mode): the entry and the residual subtraction in fp64, rounded once when stored.
// PRE (paper-size MLP, hh_wide.cuh): the raw entries were written into the rank-k slot by k2_eval_wide; they are loaded here.
template <bool COLS, bool F64, bool PRE = false>
__global__ void __launch_bounds__(A2_T, F64 ? 2 : A2_OCC) k2_step(A2Args A, u32 count, u32 ncount) {
  constexpr int E = A2_E, GPW = 2 * A2_E;                           // entries per thread, granules per warp
  __shared__ __align__(16) float sw[PRE ? 4 : (F64 ? 2 * HH_MLP2_FLOATS : HH_MLP2_FLOATS)];
  if (!PRE) {
    if (F64) load_weights(sw, reinterpret_cast<const float*>(A.w2d), 2 * HH_MLP2_FLOATS);
    else load_weights(sw, A.w2, HH_MLP2_FLOATS);
  }
  __syncthreads();
  const u32 lane = threadIdx.x & 31, half = lane >> 4, l16 = lane & 15, warp = threadIdx.x >> 5;
  const uint2* gl = COLS ? A.gn : A.gm;
  const u32 ntiles = (count + GPW - 1) / GPW;
  u32 tile = blockIdx.x * (A2_T / 32) + warp;
  for (; tile < ntiles; tile += gridDim.x * (A2_T / 32)) {
    // (a) line 6 for the row granules with the same indices (memory-bound, independent of line 7)
    if (COLS && GPW * tile < ncount) {
#pragma unroll
      for (int e = 0; e < E; ++e) a2_norm_granule(A, GPW * tile + 2 * e + half, ncount, lane);
    }
    // (b) the entries
    float v[E][9];
    double vd[F64 ? E : 1][9];
    if (PRE) {
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const u32 gi = GPW * tile + 2 * e + half;
        const bool gv = gi < count;
        const uint2 g = gl[gv ? gi : count - 1];
        const BlkState& s = A.st[g.x];
        const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
        const u32 len = COLS ? s.n : s.m, lenp = COLS ? np : mp, idx = g.y + l16;
        const bool ok = gv && s.status == 0 && idx < len;
        const float* src = chunk_ptr(A, A.tab + (size_t)g.x * HH_TAB_STRIDE, s.k) +
                           (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(s.k % HH_RC) * 9 * np : (size_t)(s.k % HH_RC) * 9 * mp);
#pragma unroll
        for (int r = 0; r < 9; ++r) v[e][r] = ok ? src[(size_t)r * lenp + idx] : 0.f;
      }
    } else {
      float xi[E][3], xj[E][3];
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const u32 gi = GPW * tile + 2 * e + half;
        const uint2 g = gl[gi < count ? gi : count - 1];
        const BlkState& s = A.st[g.x];
        const u32 len = COLS ? s.n : s.m, idx = g.y + l16;
        const u32 ic = idx < len ? idx : len - 1;
        const u32 ti = COLS ? s.tlo + (u32)(s.ik < 0 ? 0 : s.ik) : s.tlo + ic;   // target (row) particle (ik unset on blocks that just stopped)
        const u32 sj = COLS ? s.slo + ic : s.slo + (u32)s.jk;                    // source (column) particle
#pragma unroll
        for (int d = 0; d < 3; ++d) { xi[e][d] = A.Xs[3 * (size_t)ti + d]; xj[e][d] = A.Xs[3 * (size_t)sj + d]; }
      }
      if (F64) {
#pragma unroll 1
        for (int e = 0; e < E; ++e) {
          float a3[3], b3[3];
          double m9[9];
#pragma unroll
          for (int d = 0; d < 3; ++d) { a3[d] = xi[0][d]; b3[d] = xj[0][d]; }
#pragma unroll
          for (int e2 = 1; e2 < E; ++e2)
            if (e == e2) {
#pragma unroll
              for (int d = 0; d < 3; ++d) { a3[d] = xi[e2][d]; b3[d] = xj[e2][d]; }
            }
          entry2_eval_d(reinterpret_cast<const double*>(sw), (double)A.a, a3, b3, m9);
#pragma unroll
          for (int e2 = 0; e2 < E; ++e2)
            if (e == e2) {
#pragma unroll
              for (int r = 0; r < 9; ++r) vd[F64 ? e2 : 0][r] = m9[r];
            }
        }
      } else {
        entry2_eval<E>(sw, A.a, xi, xj, v);
      }
    }
    // (c) residual, pivot scores, Gram sums: one granule per half-warp and slot
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const u32 gi = GPW * tile + 2 * e + half;
      const bool gv = gi < count;
      const uint2 g = gl[gv ? gi : count - 1];
      const BlkState& s = A.st[g.x];
      const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
      const u32 len = COLS ? s.n : s.m, lenp = COLS ? np : mp, idx = g.y + l16;
      const int k = s.k;
      const bool live = gv && s.status == 0, ok = live && idx < len;
      const u32* tabrow = A.tab + (size_t)g.x * HH_TAB_STRIDE;
      float* acc = A.acc + (size_t)g.x * acc_stride(A.R);
      float* dst = chunk_ptr(A, tabrow, k) + (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(k % HH_RC) * 9 * np : (size_t)(k % HH_RC) * 9 * mp);
      float Z[9];
#pragma unroll
      for (int r = 0; r < 9; ++r) { Z[r] = 0.f; if (!ok || F64) v[e][r] = 0.f; }
      // subtract sum_p C_p(row) Q_p(col); the fixed operand is a broadcast load.  On the row side the same pass over the
      // stored rows Q_p(j) also builds Z(j) = sum_p Q_p(j)^T A_pk for the cross term (S-19).
      if (ok) {
        const u32 fix = COLS ? (u32)s.ik : (u32)s.jk;
#pragma unroll 2
        for (int p = 0; p < k; ++p) {
          const float* base = chunk_ptr(A, tabrow, p);
          const float* Cp = base + (size_t)(p % HH_RC) * 9 * mp;
          const float* Qp = base + (size_t)HH_RC * 9 * mp + (size_t)(p % HH_RC) * 9 * np;
          float cp[9], qp[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) {
            cp[r] = Cp[(size_t)r * mp + (COLS ? fix : idx)];
            qp[r] = Qp[(size_t)r * np + (COLS ? idx : fix)];
          }
          if (F64) {
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int c = 0; c < 3; ++c)
                vd[F64 ? e : 0][3 * r + c] -= (double)cp[3 * r] * (double)qp[c] + (double)cp[3 * r + 1] * (double)qp[3 + c] + (double)cp[3 * r + 2] * (double)qp[6 + c];
          } else {
            submul33(v[e], cp, qp);
          }
          if (COLS) {
            const float* Ap = acc + ACC_APK + 9 * p;
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int c = 0; c < 3; ++c) Z[3 * r + c] += qp[r] * Ap[c] + qp[3 + r] * Ap[3 + c] + qp[6 + r] * Ap[6 + c];
          }
        }
        if (F64) {
#pragma unroll
          for (int r = 0; r < 9; ++r) v[e][r] = (float)vd[F64 ? e : 0][r];      // rounded once
        }
#pragma unroll
        for (int r = 0; r < 9; ++r) dst[(size_t)r * lenp + idx] = v[e][r];   // the residual (column: normalised by line 6 later; row: kept raw)
      } else if (COLS && live && idx < lenp) {
#pragma unroll
        for (int r = 0; r < 9; ++r) dst[(size_t)r * lenp + idx] = 0.f;      // zero the pad columns (the far-field kernel reads float4)
      }
      // arg-max scores over unused rows / columns (Eq. (9); S-18)
      unsigned long long kd = 0ull, kf = 0ull;
      if (ok) {
        const int* piv = a2_piv(A, g.x) + (COLS ? HH_MAX_RANK : 0);
        bool used = false;
        for (int q = 0; q < k + (COLS ? 1 : 0); ++q) used |= (piv[q] == (int)idx);
        if (!used) { kd = amax_key(fabsf(det33(v[e])), idx); kf = amax_key(fro2_33(v[e]), idx); }
      }
      kd = half_max(kd); kf = half_max(kf);
      if (l16 == 0 && (kd | kf)) {
        atomicMax(&A.amax[(size_t)g.x * 4 + (COLS ? 2 : 0)], kd);
        atomicMax(&A.amax[(size_t)g.x * 4 + (COLS ? 3 : 1)], kf);
      }
      if (COLS) {
        // norm recursion (S-19): B_kk = sum_j q(j) q(j)^T (nu^2 = tr(A_kk B_kk) is formed in k2_fin, once line 6 has summed
        // A_kk over all rows), cross = sum_p tr(A_pk B_kp) = sum_j tr(Z(j) q(j))
        float bkk[9], cross = 0.f;
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            bkk[3 * r + c] = v[e][3 * r] * v[e][3 * c] + v[e][3 * r + 1] * v[e][3 * c + 1] + v[e][3 * r + 2] * v[e][3 * c + 2];
            cross = fmaf(Z[3 * r + c], v[e][3 * c + r], cross);
          }
        const float t = half_sum9(bkk, l16);
        cross = half_sum(cross);
        const bool okh = __shfl_sync(0xffffffffu, ok, lane & 16);       // validity of the granule (its first column)
        if (okh && l16 < 9) atomicAdd(&acc[ACC_BKK + l16], t);
        if (okh && l16 == 9) atomicAdd(&acc[ACC_CROSS], cross);
      } else {
        // Gram matrices of the raw column, A'_pk = sum_i C_p(i)^T c'(i); k2_piv turns them into A_pk = A'_pk P^-1.
        // The stored columns were read a moment ago by this same thread (L1 / L2 hits, no second trip to HBM).
        int kw = ok ? k : 0;
#pragma unroll
        for (int o = 16; o; o >>= 1) kw = max(kw, __shfl_xor_sync(0xffffffffu, kw, o));
        const int kh = __shfl_sync(0xffffffffu, ok ? k : 0, lane & 16);
        for (int p = 0; p < kw; ++p) {
          float ap[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) ap[r] = 0.f;
          if (ok && p < k) {
            const float* Cp = chunk_ptr(A, tabrow, p) + (size_t)(p % HH_RC) * 9 * mp;
            float cp[9];
#pragma unroll
            for (int r = 0; r < 9; ++r) cp[r] = Cp[(size_t)r * mp + idx];
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int c = 0; c < 3; ++c) ap[3 * r + c] = cp[r] * v[e][c] + cp[3 + r] * v[e][3 + c] + cp[6 + r] * v[e][6 + c];
          }
          const float t = half_sum9(ap, l16);
          if (l16 < 9 && p < kh) atomicAdd(&acc[ACC_APK + 9 * p + l16], t);
        }
      }
    }
  }
  if (COLS)                                                         // more row granules than column granules: finish line 6
    for (; GPW * tile < ncount; tile += gridDim.x * (A2_T / 32)) {
#pragma unroll
      for (int e = 0; e < E; ++e) a2_norm_granule(A, GPW * tile + 2 * e + half, ncount, lane);
    }
}

// ---- the default form, first half: the entries of lines 4 / 7 alone, two per thread at the register budget of the MLP
// (the near-field kernel's), stored raw in the slot of rank k; k2_upd then does the update ----
// NORM (with COLS): line 6 for the row granules with the same indices rides along -- it is memory-bound and independent of
// these entries, and this kernel's arithmetic hides its loads (k2_upd is memory-bound itself and would only be delayed by it).
template <bool COLS, bool NORM = false>
__global__ void __launch_bounds__(A2_T, 2) k2_eval(A2Args A, u32 count, u32 ncount) {
  __shared__ __align__(16) float sw[HH_MLP2_FLOATS];
  load_weights(sw, A.w2, HH_MLP2_FLOATS);
  __syncthreads();
  const u32 lane = threadIdx.x & 31, half = lane >> 4, l16 = lane & 15, warp = threadIdx.x >> 5;
  const uint2* gl = COLS ? A.gn : A.gm;
  const u32 ntiles = (count + 3) / 4;
  u32 tile = blockIdx.x * (A2_T / 32) + warp;
  for (; tile < ntiles; tile += gridDim.x * (A2_T / 32)) {
    if (NORM && 4 * tile < ncount) {
      a2_norm_granule(A, 4 * tile + half, ncount, lane);
      a2_norm_granule(A, 4 * tile + 2 + half, ncount, lane);
    }
    float xi[2][3], xj[2][3], v[2][9];
    float* dst[2];
    u32 lenp2[2];
    bool ok[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const u32 gi = 4 * tile + 2 * e + half;
      const bool gv = gi < count;
      const uint2 g = gl[gv ? gi : count - 1];
      const BlkState& s = A.st[g.x];
      const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
      const u32 len = COLS ? s.n : s.m, idx = g.y + l16;
      const u32 ic = idx < len ? idx : len - 1;
      const u32 ti = COLS ? s.tlo + (u32)(s.ik < 0 ? 0 : s.ik) : s.tlo + ic;
      const u32 sj = COLS ? s.slo + ic : s.slo + (u32)s.jk;
#pragma unroll
      for (int d = 0; d < 3; ++d) { xi[e][d] = A.Xs[3 * (size_t)ti + d]; xj[e][d] = A.Xs[3 * (size_t)sj + d]; }
      ok[e] = gv && s.status == 0 && idx < len;
      lenp2[e] = COLS ? np : mp;
      dst[e] = chunk_ptr(A, A.tab + (size_t)g.x * HH_TAB_STRIDE, s.k) +
               (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(s.k % HH_RC) * 9 * np : (size_t)(s.k % HH_RC) * 9 * mp) + idx;
    }
    entry2_eval<2>(sw, A.a, xi, xj, v);
#pragma unroll
    for (int e = 0; e < 2; ++e)
      if (ok[e]) {
#pragma unroll
        for (int r = 0; r < 9; ++r) dst[e][(size_t)r * lenp2[e]] = v[e][r];
      }
  }
  if (NORM)                                                         // more row granules than column granules: finish line 6
    for (; 4 * tile < ncount; tile += gridDim.x * (A2_T / 32)) {
      a2_norm_granule(A, 4 * tile + half, ncount, lane);
      a2_norm_granule(A, 4 * tile + 2 + half, ncount, lane);
    }
}

// ---- the update alone, vectorised (the default with k2_eval in front): a thread takes RPT consecutive rows (4) resp. columns
// (2) of a granule, so the stored rank terms are read as 16- / 8-byte loads, the 27 multiply-adds per rank term are done for RPT
// entries per fixed-operand fetch, and the 3x3 Gram sums of a granule are reduced over 4 resp. 8 lanes instead of 16.  Per
// (entry, rank term) that is about 80 instructions instead of 200 in k2_step.  Arithmetic per entry is k2_step's, in its order.
#ifndef K2U_UNROLL
#define K2U_UNROLL 2             /* rank terms in flight per thread in k2_upd's update loop                */
#endif
#ifndef K2U_CTAS_COLS
#define K2U_CTAS_COLS 2          /* CTAs of k2_upd<false> per SM (the grid cap): fewer rows in flight = the Gram pass finds more of its terms in L2 */
#endif
template <int TPG>                                                  // sum 9 values over the TPG lanes of a granule group;
__device__ __forceinline__ void group_sum9(const float (&in)[9], u32 lig, float (&out)[TPG == 4 ? 3 : 2]) {   // lane lig gets slots [VPL lig, VPL lig + VPL)
  constexpr int VPL = TPG == 4 ? 3 : 2, NS = TPG * VPL;
  float v[NS];
#pragma unroll
  for (int r = 0; r < NS; ++r) v[r] = r < 9 ? in[r] : 0.f;
  int cnt = NS;
#pragma unroll
  for (int w = TPG / 2; w; w >>= 1) {
    const bool up = (lig & w) != 0;
    cnt >>= 1;
#pragma unroll
    for (int r = 0; r < cnt; ++r) {
      const float send = up ? v[r] : v[r + cnt], keep = up ? v[r + cnt] : v[r];
      v[r] = keep + __shfl_xor_sync(0xffffffffu, send, w);
    }
  }
#pragma unroll
  for (int r = 0; r < VPL; ++r) out[r] = v[r];
}
template <int RPT> struct VecT;
template <> struct VecT<4> { typedef float4 T; };
template <> struct VecT<2> { typedef float2 T; };
template <int RPT>
__device__ __forceinline__ void vec_load(const float* p, float (&o)[RPT]) {
  const typename VecT<RPT>::T t = *reinterpret_cast<const typename VecT<RPT>::T*>(p);
  o[0] = t.x; o[1] = t.y;
  if constexpr (RPT == 4) { o[2] = t.z; o[3] = t.w; }
}
// the same load with an L2 eviction-priority policy (createpolicy): the column side reads every stored term twice (update,
// then the Gram sums against the finished residual); the first read asks L2 to keep the line, the second lets it go
template <int RPT>
__device__ __forceinline__ void vec_load_pol(const float* p, float (&o)[RPT], unsigned long long pol) {
  if constexpr (RPT == 4)
    asm volatile("ld.global.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;" : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]) : "l"(p), "l"(pol));
  else
    asm volatile("ld.global.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(o[0]), "=f"(o[1]) : "l"(p), "l"(pol));
}
template <int RPT>
__device__ __forceinline__ void vec_store(float* p, const float (&o)[RPT]) {
  typename VecT<RPT>::T t;
  t.x = o[0]; t.y = o[1];
  if constexpr (RPT == 4) { t.z = o[2]; t.w = o[3]; }
  *reinterpret_cast<typename VecT<RPT>::T*>(p) = t;
}

template <bool COLS, bool NORM = false>
__global__ void __launch_bounds__(A2_T, 2) k2_upd(A2Args A, u32 count, u32 ncount) {
  constexpr int RPT = COLS ? 2 : 4, TPG = GR / RPT, GPW = 32 / TPG, VPL = TPG == 4 ? 3 : 2;
  const u32 lane = threadIdx.x & 31, half = lane >> 4, warp = threadIdx.x >> 5, grp = lane / TPG, lig = lane % TPG;
  const uint2* gl = COLS ? A.gn : A.gm;
  const u32 ntiles = (count + GPW - 1) / GPW;
  unsigned long long pol_keep, pol_drop;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_drop));
  u32 tile = blockIdx.x * (A2_T / 32) + warp;
  for (; tile < ntiles; tile += gridDim.x * (A2_T / 32)) {
    if (NORM && GPW * tile < ncount) {                               // line 6 for the row granules with the same indices
#pragma unroll
      for (int e = 0; e < GPW / 2; ++e) a2_norm_granule(A, GPW * tile + 2 * e + half, ncount, lane);
    }
    const u32 gi = GPW * tile + grp;
    const bool gv = gi < count;
    const uint2 g = gl[gv ? gi : count - 1];
    const BlkState& s = A.st[g.x];
    const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
    const u32 len = COLS ? s.n : s.m, lenp = COLS ? np : mp, idx0 = g.y + RPT * lig;
    const int k = s.k;
    const bool live = gv && s.status == 0, any = live && idx0 < len;   // this thread has at least one real row / column
    const u32* tabrow = A.tab + (size_t)g.x * HH_TAB_STRIDE;
    float* acc = A.acc + (size_t)g.x * acc_stride(A.R);
    float* dst = chunk_ptr(A, tabrow, k) + (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(k % HH_RC) * 9 * np : (size_t)(k % HH_RC) * 9 * mp);
    float v[9][RPT], Z[COLS ? 9 : 1][RPT];
#pragma unroll
    for (int r = 0; r < 9; ++r)
#pragma unroll
      for (int c = 0; c < RPT; ++c) { v[r][c] = 0.f; if (COLS) Z[COLS ? r : 0][c] = 0.f; }
    if (any) {
#pragma unroll
      for (int r = 0; r < 9; ++r) vec_load<RPT>(dst + (size_t)r * lenp + idx0, v[r]);   // the raw entries (k2_eval)
#pragma unroll
      for (int r = 0; r < 9; ++r)
#pragma unroll
        for (int c = 0; c < RPT; ++c) if (idx0 + c >= len) v[r][c] = 0.f;                  // pad rows / columns
      const u32 fix = COLS ? (u32)s.ik : (u32)s.jk;
      constexpr int UNR = K2U_UNROLL;
#pragma unroll UNR
      for (int p = 0; p < k; ++p) {
        const float* base = chunk_ptr(A, tabrow, p);
        const float* Cp = base + (size_t)(p % HH_RC) * 9 * mp;
        const float* Qp = base + (size_t)HH_RC * 9 * mp + (size_t)(p % HH_RC) * 9 * np;
        float sp[9][RPT], fx[9];
#pragma unroll
        for (int r = 0; r < 9; ++r) {
          if (COLS) vec_load_pol<RPT>(Qp + (size_t)r * lenp + idx0, sp[r], pol_drop);      // read once per iteration
          else vec_load_pol<RPT>(Cp + (size_t)r * lenp + idx0, sp[r], pol_keep);          // read again by the Gram pass below
          fx[r] = COLS ? Cp[(size_t)r * mp + fix] : Qp[(size_t)r * np + fix];
        }
#pragma unroll
        for (int c = 0; c < RPT; ++c) {
          float a9[9], b9[9], r9[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) { a9[r] = COLS ? fx[r] : sp[r][c]; b9[r] = COLS ? sp[r][c] : fx[r]; r9[r] = v[r][c]; }
          submul33(r9, a9, b9);                                      // R -= C_p(row) Q_p(col), the expression of k2_step
#pragma unroll
          for (int r = 0; r < 9; ++r) v[r][c] = r9[r];
        }
        if (COLS) {
          const float* Ap = acc + ACC_APK + 9 * p;
          float ap[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) ap[r] = Ap[r];
#pragma unroll
          for (int c = 0; c < RPT; ++c)
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int q = 0; q < 3; ++q)
                Z[COLS ? 3 * r + q : 0][c] += sp[r][c] * ap[q] + sp[3 + r][c] * ap[3 + q] + sp[6 + r][c] * ap[6 + q];
        }
      }
#pragma unroll
      for (int r = 0; r < 9; ++r)
#pragma unroll
        for (int c = 0; c < RPT; ++c) if (idx0 + c >= len) v[r][c] = 0.f;                  // pads stay zero (the far-field kernels read them)
#pragma unroll
      for (int r = 0; r < 9; ++r) vec_store<RPT>(dst + (size_t)r * lenp + idx0, v[r]);
    } else if (COLS && live && idx0 < lenp) {
#pragma unroll
      for (int r = 0; r < 9; ++r) vec_store<RPT>(dst + (size_t)r * lenp + idx0, v[r]);      // all-pad group: zeros
    }
    // arg-max scores over unused rows / columns (Eq. (9); S-18)
    unsigned long long kd = 0ull, kf = 0ull;
    if (any) {
      const int* piv = a2_piv(A, g.x) + (COLS ? HH_MAX_RANK : 0);
      u32 used = 0;
      for (int q = 0; q < k + (COLS ? 1 : 0); ++q) {
        const u32 d = (u32)piv[q] - idx0;
        if (d < (u32)RPT) used |= 1u << d;
      }
#pragma unroll
      for (int c = 0; c < RPT; ++c) {
        if (idx0 + c < len && !((used >> c) & 1u)) {
          float m9[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) m9[r] = v[r][c];
          const unsigned long long d1 = amax_key(fabsf(det33(m9)), idx0 + c), f1 = amax_key(fro2_33(m9), idx0 + c);
          kd = d1 > kd ? d1 : kd; kf = f1 > kf ? f1 : kf;
        }
      }
    }
#pragma unroll
    for (int o = TPG / 2; o; o >>= 1) {
      unsigned long long t = __shfl_xor_sync(0xffffffffu, kd, o); kd = t > kd ? t : kd;
      t = __shfl_xor_sync(0xffffffffu, kf, o); kf = t > kf ? t : kf;
    }
    if (lig == 0 && (kd | kf)) {
      atomicMax(&A.amax[(size_t)g.x * 4 + (COLS ? 2 : 0)], kd);
      atomicMax(&A.amax[(size_t)g.x * 4 + (COLS ? 3 : 1)], kf);
    }
    const bool okg = __shfl_sync(0xffffffffu, any, lane - lig);      // the granule is real (its first thread has a real row)
    if (COLS) {
      // norm recursion (S-19): B_kk = sum_j q(j) q(j)^T, cross = sum_j tr(Z(j) q(j))
      float bkk[9], cross = 0.f, o2[VPL];
#pragma unroll
      for (int r = 0; r < 9; ++r) bkk[r] = 0.f;
#pragma unroll
      for (int c = 0; c < RPT; ++c)
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            bkk[3 * r + q] += v[3 * r][c] * v[3 * q][c] + v[3 * r + 1][c] * v[3 * q + 1][c] + v[3 * r + 2][c] * v[3 * q + 2][c];
            cross = fmaf(Z[COLS ? 3 * r + q : 0][c], v[3 * q + r][c], cross);
          }
      group_sum9<TPG>(bkk, lig, o2);
#pragma unroll
      for (int o = TPG / 2; o; o >>= 1) cross += __shfl_xor_sync(0xffffffffu, cross, o);
      if (okg) {
#pragma unroll
        for (int r = 0; r < VPL; ++r) if (VPL * lig + r < 9) atomicAdd(&acc[ACC_BKK + VPL * lig + r], o2[r]);
        if (lig == TPG - 1) atomicAdd(&acc[ACC_CROSS], cross);
      }
    } else {
      // Gram matrices of the raw column, A'_pk = sum_i C_p(i)^T c'(i) (k2_piv turns them into A_pk); the stored columns were
      // read a moment ago by this same thread (L1 / L2 hits)
      int kw = any ? k : 0;
#pragma unroll
      for (int o = 16; o; o >>= 1) kw = max(kw, __shfl_xor_sync(0xffffffffu, kw, o));
      const int kg = __shfl_sync(0xffffffffu, any ? k : 0, lane - lig);
      for (int p = 0; p < kw; ++p) {
        float ap[9], o3[VPL];
#pragma unroll
        for (int r = 0; r < 9; ++r) ap[r] = 0.f;
        if (any && p < k) {
          const float* Cp = chunk_ptr(A, tabrow, p) + (size_t)(p % HH_RC) * 9 * mp;
          float cp[9][RPT];
#pragma unroll
          for (int r = 0; r < 9; ++r) vec_load_pol<RPT>(Cp + (size_t)r * mp + idx0, cp[r], pol_drop);
#pragma unroll
          for (int c = 0; c < RPT; ++c)
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int q = 0; q < 3; ++q) ap[3 * r + q] += cp[r][c] * v[q][c] + cp[3 + r][c] * v[3 + q][c] + cp[6 + r][c] * v[6 + q][c];
        }
        group_sum9<TPG>(ap, lig, o3);
        if (p < kg) {
#pragma unroll
          for (int r = 0; r < VPL; ++r) if (VPL * lig + r < 9) atomicAdd(&acc[ACC_APK + 9 * p + VPL * lig + r], o3[r]);
        }
      }
    }
  }
  if (NORM)                                                         // more row granules than column granules: finish line 6
    for (; GPW * tile < ncount; tile += gridDim.x * (A2_T / 32)) {
#pragma unroll
      for (int e = 0; e < GPW / 2; ++e) a2_norm_granule(A, GPW * tile + 2 * e + half, ncount, lane);
    }
}

// ---- the same listing lines with the stored rank terms STAGED: a CTA takes a tile of 16 consecutive granules (256 rows
// resp. columns), and before the entries of the tile are evaluated warp 0 issues TMA bulk copies (cp.async.bulk, one mbarrier
// per CTA) of the first min(k, TS_KS) stored terms of those rows into shared memory -- a whole plane-major part of an arena
// chunk in one copy where the tile covers a block completely, one copy per (rank, component plane) where it covers a slice
// of a larger block.  The copies land while the MLP arithmetic runs (microseconds per tile), the update then reads shared
// memory, and the Gram pass of the column side reads the same staged terms again.  Ranks beyond TS_KS (360 bytes of staging
// per row) are read from global memory as in k2_step.  Arithmetic and its order are those of k2_step<COLS, false>: same bits.
// MEASURED (c3, B200): correct (ranks identical to k2_step, U within 3e-7) but SLOWER, ms_aca 6,456 vs 5,066, so it is opt-in
// (hh_set_aca_impl 2), not the default.  ncu (profiles/r02_k2_step_t.md): 16 warps per SM instead of 24, issue slots 54-58 %
// busy, fma pipe 32 %, 1.6-1.8 warps per scheduler still waiting on global loads (the fixed operand, positions, table rows, the
// A_pk accumulators, the used-pivot list), 0.5-1.2 at the tile barrier.  The staged operand was half of the loads, not the half
// that stalls: the update is bound by the latency of MANY small dependent loads per thread, not by HBM bytes.
#define TS_GR 16                 /* granules per tile                                                    */
#define TS_ROWS (TS_GR * GR)     /* 256 threads, one entry each                                          */
#define TS_KS 10                 /* stored rank terms staged per row                                     */
#define TS_W_FLOATS ((HH_MLP2_FLOATS + 31) / 32 * 32)
#define TS_SMEM (TS_W_FLOATS * 4 + TS_KS * 9 * TS_ROWS * 4 + 2 * TS_GR * 4 + 16 + 128)

__device__ __forceinline__ u32 ts_smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }

template <bool COLS>
__global__ void __launch_bounds__(TS_ROWS, 2) k2_step_t(A2Args A, u32 count, u32 ncount, u32* __restrict__ err) {
  extern __shared__ __align__(128) unsigned char ts_raw[];
  unsigned char* ts0 = ts_raw + ((128u - (ts_smem_u32(ts_raw) & 127u)) & 127u);
  float* sw = reinterpret_cast<float*>(ts0);
  float* buf = sw + TS_W_FLOATS;                                   // staged terms: per segment [rank][9][plane stride]
  u32* gbase = reinterpret_cast<u32*>(buf + TS_KS * 9 * TS_ROWS);  // per granule of the tile: offset of its first row (rank 0, plane 0)
  u32* gps = gbase + TS_GR;                                        //                      plane stride of its segment
  unsigned long long* barp = reinterpret_cast<unsigned long long*>(gps + TS_GR);
  const u32 bar = ts_smem_u32(barp);
  load_weights(sw, A.w2, HH_MLP2_FLOATS);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const u32 lane = threadIdx.x & 31, half = lane >> 4, l16 = lane & 15, warp = threadIdx.x >> 5, gslot = threadIdx.x >> 4;
  const uint2* gl = COLS ? A.gn : A.gm;
  const u32 ntiles = (count + TS_GR - 1) / TS_GR;
  u32 phase = 0;
  u32 tile = blockIdx.x;
  for (; tile < ntiles; tile += gridDim.x) {
    // (0) warp 0: cut the tile into segments (runs of consecutive granules of one block) and start the copies
    if (warp == 0) {
      const u32 gi = TS_GR * tile + l16;
      const bool gv = gi < count && half == 0;
      const uint2 g = gl[gi < count ? gi : count - 1];
      const BlkState& s = A.st[g.x];
      const bool live = gv && s.status == 0;
      const u32 pb = __shfl_up_sync(0xffffffffu, g.x, 1), pr = __shfl_up_sync(0xffffffffu, g.y, 1);
      const bool pl = __shfl_up_sync(0xffffffffu, live, 1);
      const bool head = live && (lane == 0 || !pl || pb != g.x || pr + GR != g.y);
      const u32 hm = __ballot_sync(0xffffffffu, head), lm = __ballot_sync(0xffffffffu, live);
      // the head lane of my segment, and the number of granules of the segment
      const u32 below = hm & (0xffffffffu >> (31 - lane));           // heads at or below my lane
      const int hl = below ? 31 - __clz(below) : 0;
      const u32 above = hm & ~(0xffffffffu >> (31 - lane));          // heads above my lane
      const u32 dead_above = ~lm & ~(0xffffffffu >> (31 - lane));    // first lane above that is not live ends the run as well
      const u32 stop = above | dead_above;
      const int endl = stop ? __ffs(stop) - 1 : 32;                  // one past the last granule of a segment whose head I am
      const u32 len = COLS ? s.n : s.m, lenp = a2_pad8(len), mp = a2_pad8(s.m), np = a2_pad8(s.n);
      const u32 ngr = (u32)(endl - (int)lane);
      const bool whole = g.y == 0 && g.y + GR * ngr >= len;
      const u32 rows_here = GR * ngr < lenp - g.y ? GR * ngr : lenp - g.y;   // multiple of 8
      const u32 ps_h = whole ? lenp : rows_here;
      const u32 ks_h = (u32)(s.k < TS_KS ? s.k : TS_KS);
      const u32 fl_h = head ? ks_h * 9u * ps_h : 0u;                 // floats of staging of the segment
      u32 inc = fl_h;                                                // exclusive prefix over the lanes
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const u32 t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (u32)o) inc += t; }
      const u32 total = __shfl_sync(0xffffffffu, inc, 31);
      const u32 off_h = inc - fl_h;
      const u32 seg_off = __shfl_sync(0xffffffffu, off_h, hl), seg_ps = __shfl_sync(0xffffffffu, ps_h, hl), seg_r0 = __shfl_sync(0xffffffffu, g.y, hl);
      if (lane < TS_GR) { gbase[lane] = live ? seg_off + (g.y - seg_r0) : 0u; gps[lane] = live ? seg_ps : 0u; }
      if (head && ks_h) {
        const u32* tabrow = A.tab + (size_t)g.x * HH_TAB_STRIDE;
        const u32 dst0 = ts_smem_u32(buf + off_h);
        if (whole) {
          for (u32 c = 0; 4 * c < ks_h; ++c) {
            const u32 nr = ks_h - 4 * c < 4 ? ks_h - 4 * c : 4;
            const float* src = chunk_ptr(A, tabrow, 4 * c) + (COLS ? (size_t)HH_RC * 9 * mp : 0);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst0 + 4u * c * 9u * ps_h * 4u),
                         "l"(src), "r"(nr * 9u * ps_h * 4u), "r"(bar) : "memory");
          }
        } else {
          for (u32 p = 0; p < ks_h; ++p) {
            const float* src = chunk_ptr(A, tabrow, p) + (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(p % HH_RC) * 9 * np : (size_t)(p % HH_RC) * 9 * mp) + g.y;
#pragma unroll
            for (u32 r = 0; r < 9; ++r)
              asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst0 + (p * 9u + r) * ps_h * 4u),
                           "l"(src + (size_t)r * lenp), "r"(ps_h * 4u), "r"(bar) : "memory");
          }
        }
      }
      __syncwarp();
      if (lane == 0) {
        if (total) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(total * 4u) : "memory");
        else asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
      }
    }
    // (a) line 6 for the row granules with the same indices (memory-bound, independent of line 7)
    if (COLS && TS_GR * tile < ncount) a2_norm_granule(A, TS_GR * tile + 2 * warp + half, ncount, lane);
    // (b) the entry of this thread
    const u32 gi = TS_GR * tile + gslot;
    const bool gv = gi < count;
    const uint2 g = gl[gv ? gi : count - 1];
    const BlkState& s = A.st[g.x];
    const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
    const u32 len = COLS ? s.n : s.m, lenp = COLS ? np : mp, idx = g.y + l16;
    const int k = s.k;
    const bool live = gv && s.status == 0, ok = live && idx < len;
    float v[1][9];
    {
      float xi[1][3], xj[1][3];
      const u32 ic = idx < len ? idx : len - 1;
      const u32 ti = COLS ? s.tlo + (u32)(s.ik < 0 ? 0 : s.ik) : s.tlo + ic;
      const u32 sj = COLS ? s.slo + ic : s.slo + (u32)s.jk;
#pragma unroll
      for (int d = 0; d < 3; ++d) { xi[0][d] = A.Xs[3 * (size_t)ti + d]; xj[0][d] = A.Xs[3 * (size_t)sj + d]; }
      entry2_eval<1>(sw, A.a, xi, xj, v);
    }
    // the staged terms have landed (they had the whole MLP evaluation to do so)
    {
      bool done = false;
      for (int it = 0; it < (1 << 22) && !done; ++it) {
        u32 okw;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n" : "=r"(okw) : "r"(bar), "r"(phase) : "memory");
        done = okw != 0;
      }
      if (!done) { atomicExch(err, 1u); return; }
      phase ^= 1u;
    }
    // (c) residual, pivot scores, Gram sums
    {
      const u32* tabrow = A.tab + (size_t)g.x * HH_TAB_STRIDE;
      float* acc = A.acc + (size_t)g.x * acc_stride(A.R);
      float* dst = chunk_ptr(A, tabrow, k) + (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(k % HH_RC) * 9 * np : (size_t)(k % HH_RC) * 9 * mp);
      const int ks = k < TS_KS ? k : TS_KS;
      const u32 ps = gps[gslot];
      const float* sb = buf + gbase[gslot] + l16;                   // staged: term p, plane r at sb[(9 p + r) ps]
      float Z[9];
#pragma unroll
      for (int r = 0; r < 9; ++r) { Z[r] = 0.f; if (!ok) v[0][r] = 0.f; }
      if (ok) {
        const u32 fix = COLS ? (u32)s.ik : (u32)s.jk;
#pragma unroll 2
        for (int p = 0; p < k; ++p) {
          const float* base = chunk_ptr(A, tabrow, p);
          const float* Cp = base + (size_t)(p % HH_RC) * 9 * mp;
          const float* Qp = base + (size_t)HH_RC * 9 * mp + (size_t)(p % HH_RC) * 9 * np;
          float cp[9], qp[9];
          if (p < ks) {
#pragma unroll
            for (int r = 0; r < 9; ++r) {
              const float sv = sb[(size_t)(9 * p + r) * ps];
              if (COLS) { cp[r] = Cp[(size_t)r * mp + fix]; qp[r] = sv; } else { cp[r] = sv; qp[r] = Qp[(size_t)r * np + fix]; }
            }
          } else {
#pragma unroll
            for (int r = 0; r < 9; ++r) {
              cp[r] = Cp[(size_t)r * mp + (COLS ? fix : idx)];
              qp[r] = Qp[(size_t)r * np + (COLS ? idx : fix)];
            }
          }
          submul33(v[0], cp, qp);
          if (COLS) {
            const float* Ap = acc + ACC_APK + 9 * p;
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int c = 0; c < 3; ++c) Z[3 * r + c] += qp[r] * Ap[c] + qp[3 + r] * Ap[3 + c] + qp[6 + r] * Ap[6 + c];
          }
        }
#pragma unroll
        for (int r = 0; r < 9; ++r) dst[(size_t)r * lenp + idx] = v[0][r];
      } else if (COLS && live && idx < lenp) {
#pragma unroll
        for (int r = 0; r < 9; ++r) dst[(size_t)r * lenp + idx] = 0.f;      // zero the pad columns (the far-field kernels read float4)
      }
      unsigned long long kd = 0ull, kf = 0ull;
      if (ok) {
        const int* piv = a2_piv(A, g.x) + (COLS ? HH_MAX_RANK : 0);
        bool used = false;
        for (int q = 0; q < k + (COLS ? 1 : 0); ++q) used |= (piv[q] == (int)idx);
        if (!used) { kd = amax_key(fabsf(det33(v[0])), idx); kf = amax_key(fro2_33(v[0]), idx); }
      }
      kd = half_max(kd); kf = half_max(kf);
      if (l16 == 0 && (kd | kf)) {
        atomicMax(&A.amax[(size_t)g.x * 4 + (COLS ? 2 : 0)], kd);
        atomicMax(&A.amax[(size_t)g.x * 4 + (COLS ? 3 : 1)], kf);
      }
      if (COLS) {
        float bkk[9], cross = 0.f;
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            bkk[3 * r + c] = v[0][3 * r] * v[0][3 * c] + v[0][3 * r + 1] * v[0][3 * c + 1] + v[0][3 * r + 2] * v[0][3 * c + 2];
            cross = fmaf(Z[3 * r + c], v[0][3 * c + r], cross);
          }
        const float t = half_sum9(bkk, l16);
        cross = half_sum(cross);
        const bool okh = __shfl_sync(0xffffffffu, ok, lane & 16);
        if (okh && l16 < 9) atomicAdd(&acc[ACC_BKK + l16], t);
        if (okh && l16 == 9) atomicAdd(&acc[ACC_CROSS], cross);
      } else {
        int kw = ok ? k : 0;
#pragma unroll
        for (int o = 16; o; o >>= 1) kw = max(kw, __shfl_xor_sync(0xffffffffu, kw, o));
        const int kh = __shfl_sync(0xffffffffu, ok ? k : 0, lane & 16);
        for (int p = 0; p < kw; ++p) {
          float ap[9];
#pragma unroll
          for (int r = 0; r < 9; ++r) ap[r] = 0.f;
          if (ok && p < k) {
            float cp[9];
            if (p < ks) {
#pragma unroll
              for (int r = 0; r < 9; ++r) cp[r] = sb[(size_t)(9 * p + r) * ps];
            } else {
              const float* Cp = chunk_ptr(A, tabrow, p) + (size_t)(p % HH_RC) * 9 * mp;
#pragma unroll
              for (int r = 0; r < 9; ++r) cp[r] = Cp[(size_t)r * mp + idx];
            }
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
              for (int c = 0; c < 3; ++c) ap[3 * r + c] = cp[r] * v[0][c] + cp[3 + r] * v[0][3 + c] + cp[6 + r] * v[0][6 + c];
          }
          const float t = half_sum9(ap, l16);
          if (l16 < 9 && p < kh) atomicAdd(&acc[ACC_APK + 9 * p + l16], t);
        }
      }
    }
    __syncthreads();                                                // the staging buffer and the granule table are free again
  }
  if (COLS)                                                         // more row granules than column granules: finish line 6
    for (; TS_GR * tile < ncount; tile += gridDim.x) a2_norm_granule(A, TS_GR * tile + 2 * warp + half, ncount, lane);
}

// ---- paper-size MLP: the entries of lines 4 / 7 for all active blocks, 128 per tensor-core tile (8 granules), stored raw
// in the slot of rank k (gather coordinates -> network inference -> scatter into C / Q) ----
template <bool COLS>
__global__ void __launch_bounds__(WD_T) k2_eval_wide(A2Args A, const float* __restrict__ gw, u32 count, u32* __restrict__ err_flag) {
  extern __shared__ __align__(1024) unsigned char we_raw[];
  WideSmem& S = *reinterpret_cast<WideSmem*>(we_raw);
  wide_setup(S, gw);
  const u32 tid = threadIdx.x, row = tid & 127u, l16 = row & 15;
  const uint2* gl = COLS ? A.gn : A.gm;
  const u32 ntiles = (count + 7) / 8;
  bool alive = true;
  for (u32 tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const u32 gi = 8 * tile + (row >> 4);
    const bool gv = gi < count;
    const uint2 g = gl[gv ? gi : count - 1];
    const BlkState& s = A.st[g.x];
    const u32 mp = a2_pad8(s.m), np = a2_pad8(s.n);
    const u32 len = COLS ? s.n : s.m, lenp = COLS ? np : mp, idx = g.y + l16;
    const u32 ic = idx < len ? idx : len - 1;
    const u32 ti = COLS ? s.tlo + (u32)(s.ik < 0 ? 0 : s.ik) : s.tlo + ic;
    const u32 sj = COLS ? s.slo + ic : s.slo + (u32)s.jk;
    float xi[3], xj[3], x[4], inv, out[9];
#pragma unroll
    for (int d = 0; d < 3; ++d) { xi[d] = A.Xs[3 * (size_t)ti + d]; xj[d] = A.Xs[3 * (size_t)sj + d]; }
    {
      const float rx = xj[0] - xi[0], ry = xj[1] - xi[1], rz = xj[2] - xi[2];
      float d = sqrtf(fmaf(rx, rx, fmaf(ry, ry, rz * rz)));
      d = fmaxf(d, 1e-12f * A.a);
      inv = 1.0f / d;
      x[0] = rx * inv; x[1] = ry * inv; x[2] = rz * inv; x[3] = A.a * inv;
    }
    alive = wide_tile(S, gw, x, out) && alive;
    if (tid < 128u && gv && s.status == 0 && idx < len) {                  // the result lives in the first warpgroup
      float* dst = chunk_ptr(A, A.tab + (size_t)g.x * HH_TAB_STRIDE, s.k) +
                   (COLS ? (size_t)HH_RC * 9 * mp + (size_t)(s.k % HH_RC) * 9 * np : (size_t)(s.k % HH_RC) * 9 * mp);
#pragma unroll
      for (int r = 0; r < 9; ++r) dst[(size_t)r * lenp + idx] = out[r] * inv;
    }
  }
  if (!alive && tid == 0) atomicExch(err_flag, 1u);
  wide_teardown(S);
}

__device__ __forceinline__ void a2_decode(unsigned long long key, float& score, int& idx) {
  score = key ? __uint_as_float((u32)(key >> 32)) : -1.f;
  idx = key ? (int)(0xffffffffu - (u32)key) : -1;
}
// S-18: |det| rule falls back to Frobenius when every remaining |det| is 0; rule 1 = Frobenius
__device__ __forceinline__ void a2_choose(int rule, unsigned long long kd, unsigned long long kf, int& idx, float& best) {
  float bd, bf; int bdi, bfi;
  a2_decode(kd, bd, bdi); a2_decode(kf, bf, bfi);
  if (rule == 0 && (bd > 0.f || bf <= 0.f)) { idx = bdi; best = bd; } else { idx = bfi; best = bf; }
}

// ---- lines 5-6: pivot row, P^-1 and cond_F(P) in fp64 ----
__global__ void __launch_bounds__(256) k2_piv(A2Args A) {
  const u32 b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= A.nb) return;
  BlkState s = A.st[b];
  if (s.status != 0) return;
  int ik; float best;
  a2_choose(A.rule, A.amax[(size_t)b * 4], A.amax[(size_t)b * 4 + 1], ik, best);
  if (ik < 0 || !(best > 0.f)) { a2_finish(A, b, s, 1, 0); A.st[b] = s; return; }   // S-21: zero residual column -> block reproduced
  const u32 mp = a2_pad8(s.m);
  const u32* tabrow = A.tab + (size_t)b * HH_TAB_STRIDE;
  const float* Ck = chunk_ptr(A, tabrow, s.k) + (size_t)(s.k % HH_RC) * 9 * mp;
  double P[9], Pi[9];
#pragma unroll
  for (int r = 0; r < 9; ++r) P[r] = (double)Ck[(size_t)r * mp + ik];
  a2_piv(A, b)[s.k] = ik;
  const double dP = P[0] * (P[4] * P[8] - P[5] * P[7]) - P[1] * (P[3] * P[8] - P[5] * P[6]) + P[2] * (P[3] * P[7] - P[4] * P[6]);
  bool sing = fabs(dP) < 1e-30;
  if (!sing) {
    const double iv = 1.0 / dP;
    Pi[0] = (P[4] * P[8] - P[5] * P[7]) * iv; Pi[1] = (P[2] * P[7] - P[1] * P[8]) * iv; Pi[2] = (P[1] * P[5] - P[2] * P[4]) * iv;
    Pi[3] = (P[5] * P[6] - P[3] * P[8]) * iv; Pi[4] = (P[0] * P[8] - P[2] * P[6]) * iv; Pi[5] = (P[2] * P[3] - P[0] * P[5]) * iv;
    Pi[6] = (P[3] * P[7] - P[4] * P[6]) * iv; Pi[7] = (P[1] * P[6] - P[0] * P[7]) * iv; Pi[8] = (P[0] * P[4] - P[1] * P[3]) * iv;
    double np2 = 0.0, ni2 = 0.0;
#pragma unroll
    for (int r = 0; r < 9; ++r) { np2 += P[r] * P[r]; ni2 += Pi[r] * Pi[r]; }
    sing = sqrt(np2 * ni2) > A.kappa_max &&                        // S-18b, where the dense evaluation is affordable
           (double)s.m * (double)s.n <= A.dense_cap * ((double)s.m + (double)s.n);
  }
  if (sing) { a2_finish(A, b, s, 2, 2); A.st[b] = s; return; }     // S-18 / S-18b: breakdown -> the block is applied densely
#pragma unroll
  for (int r = 0; r < 9; ++r) A.pinv[(size_t)b * 9 + r] = Pi[r];
  // c_k = c' P^-1  =>  A_pk = sum_i C_p(i)^T c_k(i) = A'_pk P^-1
  float* acc = A.acc + (size_t)b * acc_stride(A.R);
  for (int p = 0; p < s.k; ++p) {
    float* Ap = acc + ACC_APK + 9 * p;
    double a[9];
#pragma unroll
    for (int r = 0; r < 9; ++r) a[r] = (double)Ap[r];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int q = 0; q < 3; ++q) Ap[3 * r + q] = (float)(a[3 * r] * Pi[q] + a[3 * r + 1] * Pi[3 + q] + a[3 * r + 2] * Pi[6 + q]);
  }
  s.ik = ik;
  A.st[b] = s;
}

// ---- lines 9-12: norm recursion (S-19), stop test Eq. (10) (S-20), next column (line 8), arena space ----
__global__ void __launch_bounds__(256) k2_fin(A2Args A) {
  const u32 b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= A.nb) return;
  BlkState s = A.st[b];
  if (s.status != 0) return;
  const float* acc = A.acc + (size_t)b * acc_stride(A.R);
  const int k = s.k;
  float nu2 = 0.f;                                                  // nu^2 = tr(A_kk B_kk)  (S-19)
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) nu2 = fmaf(acc[ACC_AKK + 3 * r + c], acc[ACC_BKK + 3 * c + r], nu2);
  const float cross = acc[ACC_CROSS];
  s.lam2 += nu2 + 2.f * cross;
  s.k = k + 1;
  const float nu = sqrtf(fmaxf(nu2, 0.f)), lam = sqrtf(fmaxf(s.lam2, 0.f));
  if (nu <= A.tol * lam) { a2_finish(A, b, s, 1, 0); A.st[b] = s; return; }                        // Eq. (10)
  int jn; float best;
  a2_choose(A.rule, A.amax[(size_t)b * 4 + 2], A.amax[(size_t)b * 4 + 3], jn, best);
  if (jn < 0) { a2_finish(A, b, s, 1, 0); A.st[b] = s; return; }
  if (s.k >= s.kmax) {                                                                             // S-21: N_ite_max reached (flag 1) or min(c,q): exact
    a2_finish(A, b, s, 1, s.kmax < min((int)s.m, (int)s.n) ? 1 : 0);
    A.st[b] = s;
    return;
  }
  s.jk = jn;
  a2_piv(A, b)[HH_MAX_RANK + s.k] = jn;
  if ((s.k % HH_RC) == 0 && !a2_alloc(A, b, s, s.k)) s.status = -1;     // arena full: this block is redone in the next batch
  else a2_zero_acc(A, b, s.k);
  A.st[b] = s;
}

// largest `end` such that blocks [first, end) fit the scratch region at the predicted number of chunks per block,
// including the lock-step state (table row, block state, accumulators, granule lists)
__global__ void k2_batch_range(const u64* __restrict__ unit_prefix, u32 first, u32 nG, u64 total_units, u32 chunks_pred,
                               u32 per_block_units, DevScalars* sc) {
  u32 lo = first, hi = nG;
  const u64 s0 = unit_prefix[first];
  while (lo < hi) {
    u32 mid = lo + (hi - lo + 1) / 2;
    const u64 rows = unit_prefix[mid] - s0;
    u64 need = rows * 9ull / 8ull * chunks_pred + (u64)(mid - first) * (7ull + per_block_units) + rows / 8ull + 64ull;
    if (need <= total_units) lo = mid; else hi = mid - 1;
  }
  sc->batch_end = lo;
  sc->batch_units = unit_prefix[lo] - s0;
  {                                                      // first block of the second half: half of the rows + columns on either side
    const u64 target = s0 + (unit_prefix[lo] - s0) / 2;
    u32 a = first, b = lo;
    while (a < b) { const u32 mid = a + (b - a) / 2; if (unit_prefix[mid] < target) a = mid + 1; else b = mid; }
    sc->batch_mid = a;
  }
  sc->batch_units1 = unit_prefix[first + 1 <= nG ? first + 1 : first] - s0;
  sc->arena_cursor = 0;
  sc->fail_min = 0xffffffffu;
  sc->sum_rank = sc->aca_entries = sc->factor_bytes = 0;
  sc->not_conv = sc->singular = sc->max_rank_seen = 0;
  sc->n_dense = 0;
  sc->fallback_entries = 0;
}

// ---- hh_set_aca_impl 4: the batch as TWO half-batches (half of the rows + columns each), one listing line apart ----
// Entry evaluation (k2_eval) is bound by the ALUs, the update (k2_upd) by memory, and inside one block they cannot overlap
// (the next pivot needs the finished residual).  Two half-batches can: while half A evaluates entries on the caller's stream,
// half B runs its update on a side stream, both kernels launched with one CTA per SM so that an SM holds one of each.
// Per half the four stages are  0: k2_eval<rows of tau>, 1: k2_upd + k2_piv, 2: k2_eval<columns of sigma> (+ line 6),
// 3: k2_upd + k2_fin + granule lists of the next iteration.  The halves share the arena, its cursor and fail_min.
static int a2_two_halves(hh_ctx* ctx, const A2Args& A0, u32 mid, u32* cm2, u32* cn2, uint2* gm2, uint2* gn2, size_t ngran) {
  cudaStream_t s = ctx->stream, s2 = ctx->stream2;
  const int R = A0.R;
  const size_t accs = ACC_APK + 9 * (size_t)(R + 1);
  if (mid <= A0.first) mid = A0.first + 1;
  if (mid >= A0.first + A0.nb) mid = A0.first + A0.nb - 1;
  struct Half { A2Args A; u32 gmc, gnc; int stage; bool active; } H[2];
  for (int h = 0; h < 2; ++h) {
    const u32 o = h ? mid - A0.first : 0u, n = h ? A0.first + A0.nb - mid : mid - A0.first;
    A2Args& A = H[h].A;
    A = A0;
    A.first = A0.first + o; A.nb = n;
    A.tab = A0.tab + (size_t)o * HH_TAB_STRIDE; A.st = A0.st + o; A.amax = A0.amax + (size_t)o * 4; A.pinv = A0.pinv + (size_t)o * 9;
    A.acc = A0.acc + (size_t)o * accs;
    if (h) { A.cm = cm2; A.cn = cn2; A.gm = gm2; A.gn = gn2; }
    A.nact = &ctx->d_sc->ab[h];
    H[h].stage = 0; H[h].active = true; H[h].gmc = H[h].gnc = 0;
  }
  // granule lists of a half for its next iteration; the counts come back with the next read-back
  auto lists = [&](int h) -> int {
    const A2Args& A = H[h].A;
    HH_CUDA(cudaMemsetAsync(&ctx->d_sc->ab[h], 0, sizeof(u32), s));
    k2_gran_count<<<HH_N + cdiv(A.nb, 256), 256, 0, s>>>(A);
    HH_TRY(hh_scan_u32(ctx, A.cm, A.cm, A.nb, &ctx->d_sc->ab[2 + h]));
    HH_TRY(hh_scan_u32(ctx, A.cn, A.cn, A.nb, &ctx->d_sc->ab[4 + h]));
    return HH_OK;
  };
  auto readback = [&](int h) -> int {
    HH_CUDA(cudaMemcpyAsync(ctx->h_sc->ab, ctx->d_sc->ab, sizeof ctx->h_sc->ab, cudaMemcpyDeviceToHost, s));
    HH_CUDA(cudaStreamSynchronize(s));
    H[h].active = ctx->h_sc->ab[h] != 0;
    H[h].gmc = ctx->h_sc->ab[2 + h]; H[h].gnc = ctx->h_sc->ab[4 + h];
    if (H[h].gmc > ngran || H[h].gnc > ngran) return hh_fail(ctx, HH_ERR_CUDA, "lock-step ACA: granule list overflow (internal)");
    if (H[h].active) k2_gran_fill<<<HH_N + cdiv((int64_t)H[h].A.nb * 32, 256), 256, 0, s>>>(H[h].A);
    return HH_OK;
  };
  HH_TRY(lists(0)); HH_TRY(readback(0));
  HH_TRY(lists(1)); HH_TRY(readback(1));
  const unsigned nsm = (unsigned)ctx->n_sm;
  for (int tick = 0; tick < 4 * (R + 2) + 2 && (H[0].active || H[1].active); ++tick) {
    const bool run[2] = {H[0].active, H[1].active && tick > 0};                  // the second half starts one listing line later
    const bool both = run[0] && run[1];
    // with both halves in flight one does entries and the other an update (stages of opposite parity): one CTA of each per SM
    const unsigned cap = both ? nsm : nsm * 2 * 4, ucap = both ? nsm : nsm * K2U_CTAS_COLS, ucap2 = both ? nsm : nsm * 2 * 4;
    int on_side = -1;
    if (both) {
      on_side = (H[0].stage & 1) ? 0 : 1;                                       // the half whose stage is an update goes to the side stream
      if (!(H[on_side].stage & 1) || (H[1 - on_side].stage & 1)) on_side = -1;  // (both of one kind can only happen after a half has idled: run them in turn)
    }
    if (on_side >= 0) { HH_CUDA(cudaEventRecord(ctx->ev_ab[0], s)); HH_CUDA(cudaStreamWaitEvent(s2, ctx->ev_ab[0], 0)); }
    for (int pass = 0; pass < 2; ++pass) {                                       // side-stream half first, so that both kernels are queued back to back
      const int h = on_side >= 0 ? (pass == 0 ? on_side : 1 - on_side) : pass;
      if (!run[h]) continue;
      const A2Args& A = H[h].A;
      cudaStream_t st = h == on_side ? s2 : s;
      const u32 gmc = H[h].gmc, gnc = H[h].gnc;
      switch (H[h].stage) {
        case 0: { const unsigned g = cdiv(cdiv(gmc, 4), A2_T / 32); k2_eval<false><<<HH_N + (g < cap ? g : cap), A2_T, 0, st>>>(A, gmc, 0u); break; }
        case 1: { const unsigned g = cdiv(cdiv(gmc, 8), A2_T / 32); k2_upd<false><<<HH_N + (g < ucap ? g : ucap), A2_T, 0, st>>>(A, gmc, 0u); break; }
        case 2: { const unsigned g = cdiv(cdiv(gnc > gmc ? gnc : gmc, 4), A2_T / 32); k2_eval<true, true><<<HH_N + (g < cap ? g : cap), A2_T, 0, st>>>(A, gnc, gmc); break; }
        default: { const unsigned g = cdiv(cdiv(gnc, 4), A2_T / 32); k2_upd<true><<<HH_N + (g < ucap2 ? g : ucap2), A2_T, 0, st>>>(A, gnc, 0u); break; }
      }
    }
    if (on_side >= 0) { HH_CUDA(cudaEventRecord(ctx->ev_ab[1], s2)); HH_CUDA(cudaStreamWaitEvent(s, ctx->ev_ab[1], 0)); }
    HH_LAUNCH_CHECK();
    for (int h = 0; h < 2; ++h) {
      if (!run[h]) continue;
      const A2Args& A = H[h].A;
      if (H[h].stage == 1) k2_piv<<<HH_N + cdiv(A.nb, 256), 256, 0, s>>>(A);
      if (H[h].stage == 3) {
        k2_fin<<<HH_N + cdiv(A.nb, 256), 256, 0, s>>>(A);
        HH_TRY(lists(h));
        HH_TRY(readback(h));
      }
      H[h].stage = (H[h].stage + 1) & 3;
    }
    HH_LAUNCH_CHECK();
  }
  return HH_OK;
}

static size_t a2_align(size_t v) { return (v + 255) / 256 * 256; }

int hh_aca2_batch(hh_ctx* ctx, int64_t first, int64_t* next) {
  cudaStream_t s = ctx->stream;
  const u32 nG = (u32)ctx->nG;
  const int R = ctx->p.aca_max_rank;
  if (first == 0) ctx->l_pred = ctx->l_pred_first;
  u32 chunks_pred = (u32)((ctx->l_pred + HH_RC - 1) / HH_RC);
  if (chunks_pred < 1) chunks_pred = 1;
  if (chunks_pred > HH_MAX_CHUNKS) chunks_pred = HH_MAX_CHUNKS;
  // per block: table row 128 B, state 64 B, arg-max keys 32 B, P^-1 72 B, accumulators, 2 counters, 2 granules of slack
  const size_t acc_floats = ACC_APK + 9 * (size_t)(R + 1);
  const size_t per_block_bytes = 128 + 64 + 32 + 72 + 4 * acc_floats + 8 + 32 + 16;
  const u32 per_block_units = (u32)((per_block_bytes + 127) / 128);
  const u64 total_units = ctx->scratch_bytes / 128;
  u32 end_cap = nG;
  const size_t wsm = sizeof(WideSmem) + 1024;
  if (ctx->mlp2_wide) {
    HH_CUDA(cudaFuncSetAttribute(k2_eval_wide<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wsm));
    HH_CUDA(cudaFuncSetAttribute(k2_eval_wide<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)wsm));
    HH_CUDA(cudaMemsetAsync(&ctx->d_sc->deg_overflow, 0, sizeof(u32), s));   // doubles as the tensor-core kernels' error flag
  }
  for (int attempt = 0; attempt < 24; ++attempt) {
    k2_batch_range<<<HH_N + 1, 1, 0, s>>>(ctx->unit_prefix, (u32)first, end_cap, total_units > 64 ? total_units - 64 : 0, chunks_pred,
                                          per_block_units, ctx->d_sc);
    HH_CUDA(cudaMemcpyAsync(ctx->h_sc, ctx->d_sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
    HH_CUDA(cudaStreamSynchronize(s));
    u32 end = ctx->h_sc->batch_end;
    u64 rows = ctx->h_sc->batch_units;
    if (end <= first) { end = (u32)first + 1; rows = ctx->h_sc->batch_units1; }   // try a single block; it fails below if it cannot fit
    const u32 nb = end - (u32)first;
    const size_t ngran = (size_t)(rows / GR) + nb + 8;                           // bound on the granules of either list
    // carve the scratch region: lock-step state first, the arena after it
    char* p = ctx->scratch;
    size_t off = 0;
    auto take = [&](size_t bytes) { char* r = p + off; off = a2_align(off + bytes); return r; };
    ctx->tab = (u32*)take((size_t)nb * HH_TAB_STRIDE * sizeof(u32));
    A2Args A;
    A.st = (BlkState*)take((size_t)nb * sizeof(BlkState));
    A.amax = (unsigned long long*)take((size_t)nb * 4 * sizeof(unsigned long long));
    A.pinv = (double*)take((size_t)nb * 9 * sizeof(double));
    A.acc = (float*)take((size_t)nb * acc_floats * sizeof(float));
    A.cm = (u32*)take((size_t)(nb + 1) * sizeof(u32));
    A.cn = (u32*)take((size_t)(nb + 1) * sizeof(u32));
    A.gm = (uint2*)take(ngran * sizeof(uint2));
    A.gn = (uint2*)take(ngran * sizeof(uint2));
    const bool two_halves = ctx->aca_impl == 4 && !ctx->mlp2_wide && !ctx->p.aca_precision && nb >= 2;
    u32 *cm2 = nullptr, *cn2 = nullptr; uint2 *gm2 = nullptr, *gn2 = nullptr;
    if (two_halves) {                                                            // the second half's own counters and granule lists
      cm2 = (u32*)take((size_t)(nb + 1) * sizeof(u32)); cn2 = (u32*)take((size_t)(nb + 1) * sizeof(u32));
      gm2 = (uint2*)take(ngran * sizeof(uint2)); gn2 = (uint2*)take(ngran * sizeof(uint2));
    }
    if (off + 4096 > ctx->scratch_bytes) return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "factor arena too small");
    ctx->arena = (float*)(ctx->scratch + off);
    ctx->arena_units = (ctx->scratch_bytes - off) / 128;
    // once Alg. 2 is through, the accumulators and the row-granule counters are dead: the far-field item list lives there
    ctx->far_cnt = A.cm; ctx->far_items = (uint4*)A.acc; ctx->far_items_cap = (size_t)nb * acc_floats * sizeof(float) / sizeof(uint4);
    A.w2 = ctx->w2; A.w2d = ctx->w2d; A.a = ctx->p.radius_a; A.tol = ctx->p.aca_tol; A.rule = ctx->p.pivot_rule;
    A.kappa_max = ctx->p.kappa_max > 0.f ? (double)ctx->p.kappa_max : (double)INFINITY;   // 0 = the plain listing (L221)
    A.dense_cap = ctx->p.dense_cap > 0.f ? (double)ctx->p.dense_cap : 128.0;
    A.PG = ctx->PG; A.nlo = ctx->nlo; A.nhi = ctx->nhi; A.Xs = ctx->Xs;
    A.arena = ctx->arena; A.arena_units = ctx->arena_units; A.tab = ctx->tab; A.sc = ctx->d_sc;
    A.ranks = ctx->ranks; A.flags = ctx->flags; A.first = (u32)first; A.nb = nb; A.R = R;
    A.nact = &ctx->d_sc->n_split;                                                // n_split doubles as the active-block count here
    const unsigned gb = cdiv(nb, 256);
    k2_init<<<HH_N + gb, 256, 0, s>>>(A);
    HH_LAUNCH_CHECK();
#ifdef HH_PROF
    double prof_sync = 0, prof_launch = 0; int prof_it = 0; auto prof_last = std::chrono::steady_clock::now(); const auto prof_t0 = prof_last;
#endif
    if (two_halves) HH_TRY(a2_two_halves(ctx, A, ctx->h_sc->batch_mid, cm2, cn2, gm2, gn2, ngran));
    else
    for (int it = 0; it <= R; ++it) {
      HH_CUDA(cudaMemsetAsync(&ctx->d_sc->n_split, 0, sizeof(u32), s));
      k2_gran_count<<<HH_N + gb, 256, 0, s>>>(A);
      HH_TRY(hh_scan_u32(ctx, A.cm, A.cm, nb, &ctx->d_sc->lvl.g));
      HH_TRY(hh_scan_u32(ctx, A.cn, A.cn, nb, &ctx->d_sc->lvl.h));
      HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->n_split, &ctx->d_sc->n_split, sizeof(u32), cudaMemcpyDeviceToHost, s));
      HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->lvl, &ctx->d_sc->lvl, sizeof(Cnt3), cudaMemcpyDeviceToHost, s));
#ifdef HH_PROF
      const auto tp0 = std::chrono::steady_clock::now();
#endif
      HH_CUDA(cudaStreamSynchronize(s));
#ifdef HH_PROF
      { const auto tp1 = std::chrono::steady_clock::now(); prof_sync += std::chrono::duration<double, std::milli>(tp1 - tp0).count();
        prof_launch += std::chrono::duration<double, std::milli>(tp0 - prof_last).count(); prof_last = tp1; ++prof_it; }
#endif
      const u32 nact = ctx->h_sc->n_split, gmc = ctx->h_sc->lvl.g, gnc = ctx->h_sc->lvl.h;
      if (nact == 0) break;
      if (gmc > ngran || gnc > ngran) return hh_fail(ctx, HH_ERR_CUDA, "lock-step ACA: granule list overflow (internal)");
      k2_gran_fill<<<HH_N + cdiv((int64_t)nb * 32, 256), 256, 0, s>>>(A);
      const unsigned cap = (unsigned)ctx->n_sm * A2_OCC * 4;
      unsigned g1 = cdiv(cdiv(gmc, 2 * A2_E), A2_T / 32), g2 = cdiv(cdiv(gnc, 2 * A2_E), A2_T / 32);
      const unsigned gr = (g1 < cap ? g1 : cap), gc = (g1 > g2 ? g1 : g2) < cap ? (g1 > g2 ? g1 : g2) : cap;
      const unsigned ecap = (unsigned)ctx->n_sm * 2 * 4, ucap = (unsigned)ctx->n_sm * K2U_CTAS_COLS;
      const unsigned u1 = cdiv(cdiv(gmc, 8), A2_T / 32), u2 = cdiv(cdiv(gnc, 4), A2_T / 32), u2n = cdiv(cdiv(gnc > gmc ? gnc : gmc, 4), A2_T / 32);
      if (ctx->mlp2_wide) {
        // paper-size MLP: entries on the tensor cores (hh_wide.cuh), then the vectorised update (line 6 rides with the row side)
        const unsigned t1 = cdiv(gmc, 8), t2 = cdiv(gnc, 8), nsm = (unsigned)ctx->n_sm;
        k2_eval_wide<false><<<HH_N + (t1 < nsm ? t1 : nsm), WD_T, wsm, s>>>(A, ctx->w2w, gmc, &ctx->d_sc->deg_overflow);
        k2_upd<false><<<HH_N + (u1 < ecap ? u1 : ecap), A2_T, 0, s>>>(A, gmc, 0u);
        k2_piv<<<HH_N + gb, 256, 0, s>>>(A);
        k2_eval_wide<true><<<HH_N + (t2 < nsm ? t2 : nsm), WD_T, wsm, s>>>(A, ctx->w2w, gnc, &ctx->d_sc->deg_overflow);
        k2_upd<true, true><<<HH_N + (u2n < ecap ? u2n : ecap), A2_T, 0, s>>>(A, gnc, gmc);
      } else if (ctx->aca_impl == 0 && !ctx->p.aca_precision) {
        // the default: entries (k2_eval, the MLP at its own register budget) and the vectorised update (k2_upd) as separate launches
        const unsigned e1 = cdiv(cdiv(gmc, 4), A2_T / 32), e2n = cdiv(cdiv(gnc > gmc ? gnc : gmc, 4), A2_T / 32);
        k2_eval<false><<<HH_N + (e1 < ecap ? e1 : ecap), A2_T, 0, s>>>(A, gmc, 0u);
        k2_upd<false><<<HH_N + (u1 < ucap ? u1 : ucap), A2_T, 0, s>>>(A, gmc, 0u);
        k2_piv<<<HH_N + gb, 256, 0, s>>>(A);
        k2_eval<true, true><<<HH_N + (e2n < ecap ? e2n : ecap), A2_T, 0, s>>>(A, gnc, gmc);            // + line 6 (normalisation)
        k2_upd<true><<<HH_N + (u2 < ecap ? u2 : ecap), A2_T, 0, s>>>(A, gnc, 0u);
      } else if (ctx->aca_impl == 2 && !ctx->p.aca_precision) {
        // opt-in (hh_set_aca_impl 2): tiles of 16 granules, stored terms staged through shared memory by TMA bulk copies.
        // Measured slower at c3 (ms_aca 6,456 vs 5,066 for the fused form): see the comment above k2_step_t and DESIGN.md section 6
        if (!ctx->aca_smem_set) {
          HH_CUDA(cudaFuncSetAttribute(k2_step_t<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TS_SMEM));
          HH_CUDA(cudaFuncSetAttribute(k2_step_t<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TS_SMEM));
          ctx->aca_smem_set = 1;
        }
        const unsigned tcap = (unsigned)ctx->n_sm * 2, t1 = cdiv(gmc, TS_GR), t2 = cdiv(gnc > gmc ? gnc : gmc, TS_GR);
        k2_step_t<false><<<HH_N + (t1 < tcap ? t1 : tcap), TS_ROWS, TS_SMEM, s>>>(A, gmc, 0u, &ctx->d_sc->aca_err);
        k2_piv<<<HH_N + gb, 256, 0, s>>>(A);
        k2_step_t<true><<<HH_N + (t2 < tcap ? t2 : tcap), TS_ROWS, TS_SMEM, s>>>(A, gnc, gmc, &ctx->d_sc->aca_err);   // + line 6 (normalisation)
      } else {
        // the fused form (hh_set_aca_impl 3; and the fp64 parity mode, aca_precision = 1): entries and update in one kernel
        if (ctx->p.aca_precision) k2_step<false, true><<<HH_N + gr, A2_T, 0, s>>>(A, gmc, 0u);
        else k2_step<false, false><<<HH_N + gr, A2_T, 0, s>>>(A, gmc, 0u);
        k2_piv<<<HH_N + gb, 256, 0, s>>>(A);
        if (ctx->p.aca_precision) k2_step<true, true><<<HH_N + gc, A2_T, 0, s>>>(A, gnc, gmc);   // + line 6 (normalisation)
        else k2_step<true, false><<<HH_N + gc, A2_T, 0, s>>>(A, gnc, gmc);
      }
      k2_fin<<<HH_N + gb, 256, 0, s>>>(A);
      HH_LAUNCH_CHECK();
    }
    // blocks drop out in rank order, not in list order: when the arena overflows the first failed block can sit early
    // in the batch.  Then most of the batch would be discarded -- shrink the batch and run it again instead.
    HH_CUDA(cudaMemcpyAsync(&ctx->h_sc->fail_min, &ctx->d_sc->fail_min, sizeof(u32), cudaMemcpyDeviceToHost, s));
    HH_CUDA(cudaStreamSynchronize(s));
#ifdef HH_PROF
    fprintf(stderr, "[HH_PROF] batch first=%lld nb=%u: %d iterations, wall %.1f ms, host waiting in sync %.1f ms, host between syncs (launching) %.1f ms\n", (long long)first, nb,
            prof_it, std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - prof_t0).count(), prof_sync, prof_launch);
#endif
    const u32 fm = ctx->h_sc->fail_min;
#ifdef HH_PROF
    fprintf(stderr, "[HH_PROF]   fail_min %u of [%lld, %u): %s, l_pred %.1f\n", fm, (long long)first, end, fm < end ? "OVERFLOW" : "fits", ctx->l_pred);
#endif
    if (fm < end && nb > 1 && (fm - (u32)first) < nb - nb / 4) {
      end_cap = (u32)first + (nb / 2 > 1 ? nb / 2 : 1);
      ctx->l_pred = ctx->l_pred * 1.25 > HH_MAX_RANK ? HH_MAX_RANK : ctx->l_pred * 1.25;
      continue;
    }
    return hh_aca_batch_finish(ctx, first, end, next);
  }
  return hh_fail(ctx, HH_ERR_WORKSPACE_TOO_SMALL, "lock-step ACA: could not fit a batch into the factor arena");
}
