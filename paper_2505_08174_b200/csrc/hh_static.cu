// hh_static.cu -- ONE entry point that allocates nothing: hh_dense_matvec_static (include/hh.h).
//
// Why: some callers cannot allocate -- code under CUDA graph capture, tight serving loops over small suspensions,
// harnesses that forbid cudaMalloc.  Every other entry point needs an hh_ctx, and hh_create allocates (the context struct,
// pinned host scratch, events) and synchronises (it reads the weights back to pack them).  This one takes inputs and
// outputs only and keeps its scratch -- the packed two-body weights and the per-column-split partial sums -- in a
// file-scope static __device__ array of a fixed, modest size (HH_STATIC_SCRATCH_BYTES, about 3.2 MB; every GPU that loads
// the library holds it until exit).  It calls no cudaMalloc / cudaFree / allocating library routine, no memcpy and no
// synchronisation: three kernel launches on the caller's stream.
//
// What it computes: the definition itself, U_i = F_i + sum_{j != i} M_ij F_j with M_ij = (1/r) R(MLP2([r_hat, a/r]))
// (Eq. (4), Eq. (6) L108-L113 with alpha_1 = I, S-1..S-5), i.e. what hh_matvec returns when nothing is
// admissible (L283) -- a variant of k_dense (hh_near.cu), the kernel that evaluates blocks densely from packed weights and
// a tile list in the workspace: here the "block" is the whole cloud, cut into tiles of 128 rows x one column split, each
// tile writes its partial velocities into the static scratch and a second kernel adds the splits and the self term.
// N <= HH_STATIC_MAX_N (16,384): above that the O(N^2) product is the wrong tool and the scratch would not hold the partials.
//
// The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to start at zero:
// the pack kernel rewrites all HH_MLP2_FLOATS weights (pads included) and every partial that the reduction reads is
// written by the same call (all S splits x N rows).  Two calls that OVERLAP on the GPU (different streams, or graph
// branches without a dependency) race on it; calls on one stream are ordered and safe.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address: the address is taken once per
// device, with that device current, by cudaGetSymbolAddress (st_scratch_ptr below) and only that pointer goes to kernels.
#include <mutex>

#include "hh_mlp.cuh"

#define ST_T 128                         /* threads = rows per CTA                                        */
#define ST_JT 256                        /* source columns staged in shared memory at a time              */
#define ST_SPLITS 16                     /* most column splits (partial-sum planes)                        */
#define ST_W_FLOATS 2048                 /* packed weights (HH_MLP2_FLOATS = 1612), padded                  */
#define ST_FLOATS (ST_W_FLOATS + ST_SPLITS * 3 * HH_STATIC_MAX_N)
#define ST_MAX_DEV 64

static_assert(sizeof(float) * ST_FLOATS == HH_STATIC_SCRATCH_BYTES, "hh.h states the size of the static scratch");
static_assert(HH_MLP2_FLOATS <= ST_W_FLOATS && HH_MLP2_FLOATS % 4 == 0, "packed weights must fit the scratch header");

static __device__ __align__(256) float g_static_scratch[ST_FLOATS];

static std::mutex g_static_mu;
static float* g_static_ptr[ST_MAX_DEV];  /* device address of g_static_scratch on device d (0 = not looked up yet) */

// W1 [32][4] | b1 [32] | W2 [32][32] | b2 [32] | W3T [32][12] (9 outputs of hidden unit h, 3 zero pads) | b3 [12]
// (the layout MlpOff<4, 32> of hh_mlp.cuh), written from the caller's row-major layers.  One CTA.
__global__ void __launch_bounds__(256) k_static_pack(const float* __restrict__ W1, const float* __restrict__ b1, const float* __restrict__ W2,
                                                      const float* __restrict__ b2, const float* __restrict__ W3, const float* __restrict__ b3,
                                                      float* __restrict__ out) {
  typedef MlpOff<HH_MLP2_INP, HH_MLP2_H> O;
  constexpr int H = HH_MLP2_H;
  for (int t = threadIdx.x; t < ST_W_FLOATS; t += blockDim.x) {
    float v = 0.f;
    if (t < O::B1) v = W1[t];
    else if (t < O::W2) v = b1[t - O::B1];
    else if (t < O::B2) v = W2[t - O::W2];
    else if (t < O::W3) v = b2[t - O::B2];
    else if (t < O::B3) { const int h = (t - O::W3) / 12, r = (t - O::W3) % 12; v = r < 9 ? W3[r * H + h] : 0.f; }
    else if (t < O::TOTAL) { const int r = t - O::B3; v = r < 9 ? b3[r] : 0.f; }
    out[t] = v;
  }
}

// tile (blockIdx.x, blockIdx.y) = rows [128 bx, 128 bx + 128) x columns [cps by, cps by + cps): one row per thread, the
// columns staged through shared memory (broadcast reads), the partial velocity of the tile to the scratch
__global__ void __launch_bounds__(ST_T, 3) k_static_dense(const float* __restrict__ gw, float a, const float* __restrict__ X,
                                                        const float* __restrict__ F, u32 N, u32 cps, float* __restrict__ partial) {
  __shared__ __align__(16) float sw[HH_MLP2_FLOATS];
  __shared__ float sX[ST_JT * 3], sF[ST_JT * 3];
  const u32 tid = threadIdx.x;
  load_weights(sw, gw, HH_MLP2_FLOATS);
  const u32 i = blockIdx.x * ST_T + tid, ic = i < N ? i : N - 1;
  float xi[1][3], xj[1][3], M[1][9];
#pragma unroll
  for (int c = 0; c < 3; ++c) xi[0][c] = X[3 * (size_t)ic + c];
  const u32 jb = blockIdx.y * cps, je = jb + cps < N ? jb + cps : N;
  float u0 = 0.f, u1 = 0.f, u2 = 0.f;
  for (u32 j0 = jb; j0 < je; j0 += ST_JT) {
    const u32 nt = je - j0 < ST_JT ? je - j0 : ST_JT;
    __syncthreads();
    for (u32 t = tid; t < 3 * nt; t += ST_T) { sX[t] = X[3 * (size_t)j0 + t]; sF[t] = F[3 * (size_t)j0 + t]; }
    __syncthreads();
#pragma unroll 1
    for (u32 jj = 0; jj < nt; ++jj) {
#pragma unroll
      for (int c = 0; c < 3; ++c) xj[0][c] = sX[3 * jj + c];
      entry2_eval<1>(sw, a, xi, xj, M);
      if (j0 + jj != i) {                                   // S-5: the pair i = j is the self term, added by k_static_reduce
        const float f0 = sF[3 * jj], f1 = sF[3 * jj + 1], f2 = sF[3 * jj + 2];
        u0 += M[0][0] * f0 + M[0][1] * f1 + M[0][2] * f2;
        u1 += M[0][3] * f0 + M[0][4] * f1 + M[0][5] * f2;
        u2 += M[0][6] * f0 + M[0][7] * f1 + M[0][8] * f2;
      }
    }
  }
  if (i < N) {
    float* p = partial + ((size_t)blockIdx.y * N + i) * 3;
    p[0] = u0; p[1] = u1; p[2] = u2;
  }
}

// U = F (alpha_1 = I, L56) + the S partial planes, added in split order
__global__ void __launch_bounds__(256) k_static_reduce(const float* __restrict__ partial, const float* __restrict__ F, u32 n3, u32 S,
                                                        float* __restrict__ U) {
  const u32 t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n3) return;
  float v = 0.f;
  for (u32 s = 0; s < S; ++s) v += partial[(size_t)s * n3 + t];
  U[t] = F[t] + v;
}

static int st_fail(char* err, size_t err_len, int code, const char* msg, const char* detail = nullptr) {
  if (err && err_len) snprintf(err, err_len, "%s%s%s", msg, detail ? ": " : "", detail ? detail : "");
  return code;
}

// device address of the static scratch on the CURRENT device: looked up once per device, with that device current
static int st_scratch_ptr(float** out, char* err, size_t err_len) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return st_fail(err, err_len, HH_ERR_CUDA, "hh_dense_matvec_static: cudaGetDevice failed (no CUDA device?)", cudaGetErrorString(e));
  if (dev < 0 || dev >= ST_MAX_DEV) return st_fail(err, err_len, HH_ERR_UNSUPPORTED, "hh_dense_matvec_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    float* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess || !p) return st_fail(err, err_len, HH_ERR_CUDA, "hh_dense_matvec_static: cudaGetSymbolAddress(static scratch) failed", cudaGetErrorString(e));
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return HH_OK;
}

extern "C" int hh_dense_matvec_static(const hh_mlp* mlp2, float radius_a, const float* X, const float* F, float* U, int64_t N,
                                      void* cuda_stream, char* err, size_t err_len) {
  if (err && err_len) err[0] = 0;
  if (!mlp2 || !X || !F || !U) return st_fail(err, err_len, HH_ERR_INVALID_ARG, "hh_dense_matvec_static: null mlp2, X, F or U");
  if (N < 1) return st_fail(err, err_len, HH_ERR_INVALID_ARG, "hh_dense_matvec_static: N < 1");
  if (N > HH_STATIC_MAX_N) {
    char d[160];
    snprintf(d, sizeof d, "N = %lld exceeds HH_STATIC_MAX_N = %d (the static scratch holds %d bytes); use hh_create + hh_matvec", (long long)N,
             HH_STATIC_MAX_N, (int)HH_STATIC_SCRATCH_BYTES);
    return st_fail(err, err_len, HH_ERR_WORKSPACE_TOO_SMALL, "hh_dense_matvec_static", d);
  }
  if (!(radius_a > 0.f) || !isfinite(radius_a)) return st_fail(err, err_len, HH_ERR_INVALID_ARG, "hh_dense_matvec_static: radius_a must be positive and finite");
  if (mlp2->n_layers != 3 || !mlp2->dims || !mlp2->W || !mlp2->b || mlp2->dims[0] != 4 || mlp2->dims[1] != HH_MLP2_H ||
      mlp2->dims[2] != HH_MLP2_H || mlp2->dims[3] != 9)
    return st_fail(err, err_len, HH_ERR_UNSUPPORTED, "hh_dense_matvec_static: the two-body MLP must be 4-32-32-9");
  for (int l = 0; l < 3; ++l)
    if (!mlp2->W[l] || !mlp2->b[l]) return st_fail(err, err_len, HH_ERR_INVALID_ARG, "hh_dense_matvec_static: null weight or bias pointer");
  float* scratch = nullptr;
  const int r = st_scratch_ptr(&scratch, err, err_len);
  if (r != HH_OK) return r;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const u32 n = (u32)N;
  u32 S = (n + ST_JT - 1) / ST_JT;
  if (S > ST_SPLITS) S = ST_SPLITS;
  const u32 cps = (n + S - 1) / S;                                 // columns per split
  S = (n + cps - 1) / cps;
  float* partial = scratch + ST_W_FLOATS;
  k_static_pack<<<1, 256, 0, s>>>(mlp2->W[0], mlp2->b[0], mlp2->W[1], mlp2->b[1], mlp2->W[2], mlp2->b[2], scratch);
  k_static_dense<<<dim3((n + ST_T - 1) / ST_T, S), ST_T, 0, s>>>(scratch, radius_a, X, F, n, cps, partial);
  k_static_reduce<<<(3 * n + 255) / 256, 256, 0, s>>>(partial, F, 3 * n, S, U);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return st_fail(err, err_len, HH_ERR_CUDA, "hh_dense_matvec_static: kernel launch failed", cudaGetErrorString(e));
  return HH_OK;
}
