// hh_mlp.cuh -- the HIGNN kernels (Eq. (4); MLP L92; S-1..S-4, S-23) evaluated in
// registers: E entries per thread share every weight fetched from shared memory (LDS.128 broadcast),
// so the FMA : LDS ratio is 4E : 1.  fp32, accurate tanh (S-6).
#pragma once
#include "hh_internal.cuh"

// S-6: the fp32 path needs a tanh good to a few ulp: CUDA's tanhf (<= 2 ulp).  tanh.approx (2^-11) is used only on the 2e-3
// tensor-core path (hh_near_tc.cu, near_path = 1).
#define HH_TANH(x) tanhf(x)

// Packed layout (floats): W1 [H][INP] | b1 [H] | W2 [H][H] | b2 [H] | W3T [H][12] | b3 [12]
template <int INP, int H>
struct MlpOff {
  static constexpr int W1 = 0, B1 = W1 + H * INP, W2 = B1 + H, B2 = W2 + H * H, W3 = B2 + H, B3 = W3 + H * 12,
                       TOTAL = B3 + 12;
};

// y = W3 tanh(W2 tanh(W1 x + b1) + b2) + b3 for E inputs at once.  sw: packed weights in shared memory.
template <int INP, int H, int E>
__device__ __forceinline__ void mlp_eval(const float* __restrict__ sw, const float (&x)[E][INP], float (&out)[E][9]) {
  typedef MlpOff<INP, H> O;
  float h1[E][H];
#pragma unroll
  for (int o = 0; o < H; ++o) {
    float a[E];
    const float b = sw[O::B1 + o];
#pragma unroll
    for (int e = 0; e < E; ++e) a[e] = b;
#pragma unroll
    for (int i4 = 0; i4 < INP / 4; ++i4) {
      const float4 w = *reinterpret_cast<const float4*>(sw + O::W1 + o * INP + 4 * i4);
#pragma unroll
      for (int e = 0; e < E; ++e) {
        a[e] = fmaf(w.x, x[e][4 * i4 + 0], a[e]);
        a[e] = fmaf(w.y, x[e][4 * i4 + 1], a[e]);
        a[e] = fmaf(w.z, x[e][4 * i4 + 2], a[e]);
        a[e] = fmaf(w.w, x[e][4 * i4 + 3], a[e]);
      }
    }
#pragma unroll
    for (int e = 0; e < E; ++e) h1[e][o] = HH_TANH(a[e]);
  }
#pragma unroll
  for (int e = 0; e < E; ++e)
#pragma unroll
    for (int r = 0; r < 9; ++r) out[e][r] = sw[O::B3 + r];
  // second layer in chunks of 8 hidden units; each is folded into the 9 outputs as soon as it is ready
#pragma unroll 1
  for (int oc = 0; oc < H; oc += 8) {
    float acc[E][8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const float b = sw[O::B2 + oc + u];
#pragma unroll
      for (int e = 0; e < E; ++e) acc[e][u] = b;
    }
#pragma unroll
    for (int i4 = 0; i4 < H / 4; ++i4) {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const float4 w = *reinterpret_cast<const float4*>(sw + O::W2 + (oc + u) * H + 4 * i4);
#pragma unroll
        for (int e = 0; e < E; ++e) {
          acc[e][u] = fmaf(w.x, h1[e][4 * i4 + 0], acc[e][u]);
          acc[e][u] = fmaf(w.y, h1[e][4 * i4 + 1], acc[e][u]);
          acc[e][u] = fmaf(w.z, h1[e][4 * i4 + 2], acc[e][u]);
          acc[e][u] = fmaf(w.w, h1[e][4 * i4 + 3], acc[e][u]);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const float4 wa = *reinterpret_cast<const float4*>(sw + O::W3 + (oc + u) * 12);
      const float4 wb = *reinterpret_cast<const float4*>(sw + O::W3 + (oc + u) * 12 + 4);
      const float wc = sw[O::W3 + (oc + u) * 12 + 8];
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const float t = HH_TANH(acc[e][u]);
        out[e][0] = fmaf(wa.x, t, out[e][0]); out[e][1] = fmaf(wa.y, t, out[e][1]);
        out[e][2] = fmaf(wa.z, t, out[e][2]); out[e][3] = fmaf(wa.w, t, out[e][3]);
        out[e][4] = fmaf(wb.x, t, out[e][4]); out[e][5] = fmaf(wb.y, t, out[e][5]);
        out[e][6] = fmaf(wb.z, t, out[e][6]); out[e][7] = fmaf(wb.w, t, out[e][7]);
        out[e][8] = fmaf(wc, t, out[e][8]);
      }
    }
  }
}

// Two-body entries M_ij = (1/r) R(MLP2([r_hat, a/r])), r_ij = X_j - X_i (S-1..S-3, S-7), E at once.
template <int E>
__device__ __forceinline__ void entry2_eval(const float* __restrict__ sw, float a, const float (&xi)[E][3], const float (&xj)[E][3],
                                            float (&M)[E][9]) {
  float x[E][HH_MLP2_INP], inv[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    float rx = xj[e][0] - xi[e][0], ry = xj[e][1] - xi[e][1], rz = xj[e][2] - xi[e][2];
    float d = sqrtf(fmaf(rx, rx, fmaf(ry, ry, rz * rz)));
    d = fmaxf(d, 1e-12f * a);
    float id = 1.0f / d;
    x[e][0] = rx * id; x[e][1] = ry * id; x[e][2] = rz * id; x[e][3] = a * id;
    inv[e] = id;
  }
  mlp_eval<HH_MLP2_INP, HH_MLP2_H, E>(sw, x, M);
#pragma unroll
  for (int e = 0; e < E; ++e)
#pragma unroll
    for (int r = 0; r < 9; ++r) M[e][r] *= inv[e];
}

// The same entry in fp64 (aca_precision = 1): weights as doubles in shared memory (same packed layout), one entry per call.
template <int INP, int H>
__device__ __forceinline__ void mlp_eval_d(const double* __restrict__ sw, const double (&x)[INP], double (&out)[9]) {
  typedef MlpOff<INP, H> O;
  double h1[H];
#pragma unroll
  for (int o = 0; o < H; ++o) {
    double a = sw[O::B1 + o];
#pragma unroll
    for (int i = 0; i < INP; ++i) a = fma(sw[O::W1 + o * INP + i], x[i], a);
    h1[o] = tanh(a);
  }
#pragma unroll
  for (int r = 0; r < 9; ++r) out[r] = sw[O::B3 + r];
#pragma unroll 1
  for (int o = 0; o < H; ++o) {
    double a = sw[O::B2 + o];
#pragma unroll
    for (int i = 0; i < H; ++i) a = fma(sw[O::W2 + o * H + i], h1[i], a);
    const double t = tanh(a);
#pragma unroll
    for (int r = 0; r < 9; ++r) out[r] = fma(sw[O::W3 + o * 12 + r], t, out[r]);
  }
}
__device__ __forceinline__ void entry2_eval_d(const double* __restrict__ sw, double a, const float (&xi)[3], const float (&xj)[3], double (&M)[9]) {
  const double rx = (double)xj[0] - (double)xi[0], ry = (double)xj[1] - (double)xi[1], rz = (double)xj[2] - (double)xi[2];
  double d = sqrt(rx * rx + ry * ry + rz * rz);
  d = fmax(d, 1e-12 * a);
  const double x[HH_MLP2_INP] = {rx / d, ry / d, rz / d, a / d};
  mlp_eval_d<HH_MLP2_INP, HH_MLP2_H>(sw, x, M);
#pragma unroll
  for (int r = 0; r < 9; ++r) M[r] /= d;
}

// cooperative copy of packed weights into shared memory (n floats, multiple of 4)
__device__ __forceinline__ void load_weights(float* sw, const float* __restrict__ gw, int n) {
  for (int i = threadIdx.x * 4; i < n; i += blockDim.x * 4)
    *reinterpret_cast<float4*>(sw + i) = *reinterpret_cast<const float4*>(gw + i);
}

// ---- 3x3 helpers (row-major) ----
__device__ __forceinline__ void mul33(const float* A, const float* B, float* C) {
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) C[3 * i + j] = fmaf(A[3 * i], B[j], fmaf(A[3 * i + 1], B[3 + j], A[3 * i + 2] * B[6 + j]));
}
__device__ __forceinline__ void submul33(float* R, const float* A, const float* B) {   // R -= A B
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) R[3 * i + j] -= fmaf(A[3 * i], B[j], fmaf(A[3 * i + 1], B[3 + j], A[3 * i + 2] * B[6 + j]));
}
__device__ __forceinline__ float det33(const float* A) {
  return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) + A[2] * (A[3] * A[7] - A[4] * A[6]);
}
__device__ __forceinline__ float fro2_33(const float* A) {
  float s = 0.f;
#pragma unroll
  for (int t = 0; t < 9; ++t) s = fmaf(A[t], A[t], s);
  return s;
}
