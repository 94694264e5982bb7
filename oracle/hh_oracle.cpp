// =============================================================================================
// hh_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU statement of what the H-HIGNN hot path computes
// (arxiv 2505.08174; citations are PAPER.md line numbers + section/equation/algorithm).
// fp64 arithmetic on the fp32 inputs.  It shares no code with the CUDA path under
// paper_2505_08174_b200/ and is never imported by it.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Two parts:
//   O-dense : the plain definition  U_i = F_i + sum_{j!=i} h(X_j - X_i)/|X_j-X_i| F_j  [+ 3-body]
//             (Eq. (2), Eq. (4), Eq. (6)), O(N^2) (+ O(N^3) triple loop).
//   O-H     : the algorithm step by step -- cluster tree (Def. 1), admissibility
//             (Def. 2 / Eq. (7)), BuildPartition (Alg. 1), ACA (Alg. 2,
//             L210-L234, Eqs. (8)-(10)), low-rank / dense block mat-vecs (L115, L252, L260).
//
// Readings of silent / ambiguous / garbled passages are labelled S-1 ... S-25.
// Pins (tests/test_oracle_*.py): closed forms, invariants, brute force, library SVD.
// Parity unpinned by the paper: any printed numerical value of U, factors, counts or eps_r
// (the paper prints none); everything else is pinned as listed in DESIGN.md.
//
// OpenMP is used only to shorten wall time (loops over independent targets / blocks); there is
// no blocking, fusion or re-ordering of the arithmetic beyond what the paper states.
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC  (see oracle/build.py)
// =============================================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <cstdlib>
#include <vector>
#include <algorithm>
#include <numeric>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------------------------- MLP
// S-4: y = W3 tanh(W2 tanh(W1 x + b1) + b2) + b3 (tanh on hidden layers only).
// W[l] is [out][in] row-major.  Parameters arrive as one flat fp32 array: W0,b0,W1,b1,...
struct Mlp {
  int nl = 0;
  std::vector<int> dims;
  std::vector<std::vector<double>> W, b;
};

Mlp make_mlp(const int* dims, int nl, const float* params) {
  Mlp m;
  m.nl = nl;
  m.dims.assign(dims, dims + nl + 1);
  size_t off = 0;
  for (int l = 0; l < nl; ++l) {
    int fi = dims[l], fo = dims[l + 1];
    m.W.emplace_back((size_t)fi * fo);
    for (size_t t = 0; t < (size_t)fi * fo; ++t) m.W[l][t] = (double)params[off + t];
    off += (size_t)fi * fo;
    m.b.emplace_back((size_t)fo);
    for (int t = 0; t < fo; ++t) m.b[l][t] = (double)params[off + t];
    off += fo;
  }
  return m;
}

void mlp_forward(const Mlp& m, const double* x, double* y) {
  std::vector<double> cur(x, x + m.dims[0]), nxt;
  for (int l = 0; l < m.nl; ++l) {
    int fi = m.dims[l], fo = m.dims[l + 1];
    nxt.assign(fo, 0.0);
    for (int o = 0; o < fo; ++o) {
      double s = m.b[l][o];
      for (int i = 0; i < fi; ++i) s += m.W[l][(size_t)o * fi + i] * cur[i];
      nxt[o] = (l + 1 < m.nl) ? std::tanh(s) : s;
    }
    cur.swap(nxt);
  }
  for (int o = 0; o < m.dims[m.nl]; ++o) y[o] = cur[o];
}

// ------------------------------------------------------------------------- two-body entry
// Eq. (4) L85 with the config's features.  S-1: r_ij = X_j - X_i (target i, source j).
// S-2: features [r_hat(3), a/r].  S-3: M_ij = (1/r) * R, R[alpha][beta] = out[3 alpha + beta].
// S-7: r clamped to >= 1e-12 a only to stay finite (coincident centres are undefined input).
void entry2(const Mlp& m, double a, const float* Xi, const float* Xj, double M[9]) {
  double r[3] = {(double)Xj[0] - (double)Xi[0], (double)Xj[1] - (double)Xi[1],
                 (double)Xj[2] - (double)Xi[2]};
  double d = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  if (d < 1e-12 * a) d = 1e-12 * a;
  double x[4] = {r[0] / d, r[1] / d, r[2] / d, a / d};
  double y[18];
  mlp_forward(m, x, y);
  // an 18-output network emits alpha_2 = [alpha_2^(s), alpha_2^(t)] (Eq. (2)): the H-matrix holds the transverse half
  const int off = m.dims[m.nl] == 18 ? 9 : 0;
  for (int t = 0; t < 9; ++t) M[t] = y[off + t] / d;
}
// the self half alpha_2^(s)(X_i, X_j) of an 18-output network (same normalisation, Eq. (4))
void entry2_self(const Mlp& m, double a, const float* Xi, const float* Xj, double M[9]) {
  double r[3] = {(double)Xj[0] - (double)Xi[0], (double)Xj[1] - (double)Xi[1], (double)Xj[2] - (double)Xi[2]};
  double d = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  if (d < 1e-12 * a) d = 1e-12 * a;
  double x[4] = {r[0] / d, r[1] / d, r[2] / d, a / d};
  double y[18];
  mlp_forward(m, x, y);
  for (int t = 0; t < 9; ++t) M[t] = y[t] / d;
}

inline void mat3_vec_acc(const double M[9], const double* f, double* u) {   // u += M f
  for (int al = 0; al < 3; ++al) u[al] += M[3 * al] * f[0] + M[3 * al + 1] * f[1] + M[3 * al + 2] * f[2];
}

// ----------------------------------------------------------------------- three-body faces
// S-22: face (j,k,i) exists iff i,j in N(k), i.e. |X_i-X_k| < Rcut and
// |X_j-X_k| < Rcut, i, j, k pairwise distinct.  The cutoff decision is an integer decision
// taken from floating point, so it is taken in the KERNEL's precision (fp32, fixed order
// ((dx*dx + dy*dy) + dz*dz), no contraction) on both sides.
inline bool within_cut_f32(const float* A, const float* B, float rcut) {
  float dx = A[0] - B[0], dy = A[1] - B[1], dz = A[2] - B[2];
  float d2 = (dx * dx + dy * dy) + dz * dz;
  return d2 < rcut * rcut;
}

// S-23: U_i += R(MLP3([X_j-X_i, X_k-X_i, |X_j-X_k|])) F_j / (|X_j-X_k| |X_k-X_i|)  (Eq. (4))
// An 18-output three-body network emits [alpha_3^(s), alpha_3^(t)] (L56): `self` selects the first half (it then multiplies F_i,
// passed in place of F_j), otherwise the transverse half (or the 9 outputs of a 9-output network) multiplies F_j.
void face_term(const Mlp& m3, const float* Xi, const float* Xj, const float* Xk, const float* Fj,
               double* u, bool self = false) {
  double x[7], djk = 0, dki = 0;
  for (int c = 0; c < 3; ++c) {
    x[c] = (double)Xj[c] - (double)Xi[c];
    x[3 + c] = (double)Xk[c] - (double)Xi[c];
    double e = (double)Xj[c] - (double)Xk[c];
    djk += e * e;
    dki += x[3 + c] * x[3 + c];
  }
  djk = std::sqrt(djk);
  dki = std::sqrt(dki);
  x[6] = djk;
  double yy[18];
  mlp_forward(m3, x, yy);
  const double* y = yy + ((!self && m3.dims[m3.nl] == 18) ? 9 : 0);
  double s = 1.0 / (djk * dki);
  double f[3] = {(double)Fj[0], (double)Fj[1], (double)Fj[2]};
  for (int al = 0; al < 3; ++al) u[al] += s * (y[3 * al] * f[0] + y[3 * al + 1] * f[1] + y[3 * al + 2] * f[2]);
}

// ------------------------------------------------------------------------------ 3x3 helpers
inline void mul33(const double* A, const double* B, double* C) {   // C = A B
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      C[3 * i + j] = A[3 * i] * B[j] + A[3 * i + 1] * B[3 + j] + A[3 * i + 2] * B[6 + j];
}
inline double det33(const double* A) {
  return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
         A[2] * (A[3] * A[7] - A[4] * A[6]);
}
inline double fro2(const double* A) {
  double s = 0;
  for (int t = 0; t < 9; ++t) s += A[t] * A[t];
  return s;
}
inline void inv33(const double* A, double det, double* B) {        // adjugate / det
  B[0] = (A[4] * A[8] - A[5] * A[7]) / det;
  B[1] = (A[2] * A[7] - A[1] * A[8]) / det;
  B[2] = (A[1] * A[5] - A[2] * A[4]) / det;
  B[3] = (A[5] * A[6] - A[3] * A[8]) / det;
  B[4] = (A[0] * A[8] - A[2] * A[6]) / det;
  B[5] = (A[2] * A[3] - A[0] * A[5]) / det;
  B[6] = (A[3] * A[7] - A[4] * A[6]) / det;
  B[7] = (A[1] * A[6] - A[0] * A[7]) / det;
  B[8] = (A[0] * A[4] - A[1] * A[3]) / det;
}

// ----------------------------------------------------------------------------- Morton keys
// S-8: root CUBE of side ext = max_d(max_d - min_d) anchored at the minimum corner; quantise in
// fp64: q_d = min(floor(((double)x_d - lo_d)/ext * 2^21), 2^21-1); ext = 0 -> all codes 0.
// Key = 63-bit interleave, x in the highest bit of each triple (x is split first, Fig. 2).
uint64_t spread21(uint64_t v) {           // plain loop: bit b of v -> bit 3b
  uint64_t r = 0;
  for (int b = 0; b < 21; ++b) r |= ((v >> b) & 1ull) << (3 * b);
  return r;
}
void morton_keys(int64_t N, const float* X, uint64_t* keys) {
  double lo[3], hi[3];
  for (int c = 0; c < 3; ++c) { lo[c] = (double)X[c]; hi[c] = (double)X[c]; }
  for (int64_t i = 0; i < N; ++i)
    for (int c = 0; c < 3; ++c) {
      double v = (double)X[3 * i + c];
      if (v < lo[c]) lo[c] = v;
      if (v > hi[c]) hi[c] = v;
    }
  double ext = 0;
  for (int c = 0; c < 3; ++c) ext = std::max(ext, hi[c] - lo[c]);
  for (int64_t i = 0; i < N; ++i) {
    uint64_t q[3] = {0, 0, 0};
    if (ext > 0)
      for (int c = 0; c < 3; ++c) {
        double t = (((double)X[3 * i + c] - lo[c]) / ext) * 2097152.0;
        double f = std::floor(t);
        uint64_t v = (f >= 2097151.0) ? 2097151ull : (uint64_t)f;
        q[c] = v;
      }
    keys[i] = (spread21(q[0]) << 2) | (spread21(q[1]) << 1) | spread21(q[2]);
  }
}

// ---------------------------------------------------------------------------- cluster tree
struct Node { int64_t lo, hi; int32_t left, right, parent, level; float bmin[3], bmax[3]; };

struct HMat {
  int64_t N = 0;
  int leaf = 0;
  double eta = 0;
  std::vector<float> X;            // caller order
  std::vector<uint64_t> keys;      // sorted
  std::vector<int64_t> perm;       // perm[k] = original index of k-th particle in tree order (S-9)
  std::vector<float> Xs;           // tree order
  std::vector<Node> nodes;         // BFS order, left before right (S-12: numbering is free)
  std::vector<std::pair<int32_t, int32_t>> G, H;   // P^G, P^H as (tau, sigma) node ids (S-16)
};

// Def. 1 (L123-L127) realised on the Morton order.  S-10: leaf iff hi-lo <= C_leaf.
// S-11: split at the highest bit in which key[lo], key[hi-1] differ; sons [lo,m), [m,hi) with
// m = first index whose that bit is 1 (geometric bisection of the root cube cycling x,y,z, empty
// halves skipped); all keys equal -> m = lo + (hi-lo)/2.  S-13: tight AABB of the centres.
void build_tree(HMat& h) {
  int64_t N = h.N;
  std::vector<uint64_t> k0(N);
  morton_keys(N, h.X.data(), k0.data());
  h.perm.resize(N);
  std::iota(h.perm.begin(), h.perm.end(), (int64_t)0);
  std::stable_sort(h.perm.begin(), h.perm.end(), [&](int64_t a, int64_t b) { return k0[a] < k0[b]; });  // S-9
  h.keys.resize(N);
  h.Xs.resize(3 * N);
  for (int64_t k = 0; k < N; ++k) {
    h.keys[k] = k0[h.perm[k]];
    for (int c = 0; c < 3; ++c) h.Xs[3 * k + c] = h.X[3 * h.perm[k] + c];
  }
  h.nodes.clear();
  Node root{};
  root.lo = 0; root.hi = N; root.left = root.right = -1; root.parent = -1; root.level = 0;
  h.nodes.push_back(root);
  for (size_t id = 0; id < h.nodes.size(); ++id) {       // queue order = BFS
    Node nd = h.nodes[id];
    if (nd.hi - nd.lo <= h.leaf) continue;                // S-10
    uint64_t a = h.keys[nd.lo], b = h.keys[nd.hi - 1];
    int64_t m;
    if (a == b) {
      m = nd.lo + (nd.hi - nd.lo) / 2;
    } else {
      int bit = 63;
      while (!(((a ^ b) >> bit) & 1ull)) --bit;
      m = nd.lo;
      while (!((h.keys[m] >> bit) & 1ull)) ++m;           // first index whose bit is 1
    }
    Node L{}, R{};
    L.lo = nd.lo; L.hi = m; R.lo = m; R.hi = nd.hi;
    L.left = L.right = R.left = R.right = -1;
    L.parent = R.parent = (int32_t)id;
    L.level = R.level = nd.level + 1;
    h.nodes[id].left = (int32_t)h.nodes.size();
    h.nodes.push_back(L);
    h.nodes[id].right = (int32_t)h.nodes.size();
    h.nodes.push_back(R);
  }
  for (auto& nd : h.nodes) {                              // S-13
    for (int c = 0; c < 3; ++c) { nd.bmin[c] = h.Xs[3 * nd.lo + c]; nd.bmax[c] = h.Xs[3 * nd.lo + c]; }
    for (int64_t k = nd.lo; k < nd.hi; ++k)
      for (int c = 0; c < 3; ++c) {
        nd.bmin[c] = std::min(nd.bmin[c], h.Xs[3 * k + c]);
        nd.bmax[c] = std::max(nd.bmax[c], h.Xs[3 * k + c]);
      }
  }
}

// Def. 2 / Eq. (7) L141 on bounding boxes (L144, Fig. 3(b)).  S-14: diam = |bmax-bmin|_2,
// dist = |max(0, bmin_t - bmax_s, bmin_s - bmax_t)|_2; test max(diam^2) <= eta^2 dist^2 in fp64,
// order x,y,z, no contraction.  S-15: tau == sigma is never admissible.
bool admissible(const HMat& h, int32_t t, int32_t s) {
  if (t == s) return false;
  const Node& a = h.nodes[t];
  const Node& b = h.nodes[s];
  double da = 0, db = 0, dist = 0;
  for (int c = 0; c < 3; ++c) {
    double ea = (double)a.bmax[c] - (double)a.bmin[c];
    double eb = (double)b.bmax[c] - (double)b.bmin[c];
    da = da + ea * ea;
    db = db + eb * eb;
    double g1 = (double)a.bmin[c] - (double)b.bmax[c];
    double g2 = (double)b.bmin[c] - (double)a.bmax[c];
    double g = std::max(0.0, std::max(g1, g2));
    dist = dist + g * g;
  }
  double e2 = h.eta * h.eta;
  return std::max(da, db) <= e2 * dist;
}

// Alg. 1 BuildPartition (L164-L184), typo at L181 read as BuildPartition(tau', sigma').
void build_partition(HMat& h, int32_t t, int32_t s) {
  bool tleaf = h.nodes[t].left < 0, sleaf = h.nodes[s].left < 0;
  if (admissible(h, t, s)) {
    h.G.emplace_back(t, s);
  } else if (tleaf && sleaf) {
    h.H.emplace_back(t, s);
  } else if (sleaf) {
    build_partition(h, h.nodes[t].left, s);
    build_partition(h, h.nodes[t].right, s);
  } else if (tleaf) {
    build_partition(h, t, h.nodes[s].left);
    build_partition(h, t, h.nodes[s].right);
  } else {
    int32_t tc[2] = {h.nodes[t].left, h.nodes[t].right}, sc[2] = {h.nodes[s].left, h.nodes[s].right};
    for (int i = 0; i < 2; ++i)
      for (int j = 0; j < 2; ++j) build_partition(h, tc[i], sc[j]);
  }
}

// ------------------------------------------------------------------------------------- ACA
// Alg. 2 (L210-L234) with 3x3 entries, reconstructed order:
//   c_k = G(:,j_k) - C Q(:,j_k);  i_k = argmax score(c_k(i)) over unused rows;
//   c_k <- c_k [c_k(i_k)]^{-1};   q_k = G(i_k,:) - C(i_k,:) Q;
//   j_{k+1} = argmax score(q_k(j)) over unused columns;  nu^2 = |c_k q_k^T|_F^2;
//   lambda^2 += nu^2 + 2 sum_p <c_p q_p^T, c_k q_k^T>_F;  append;  stop if nu <= zeta lambda.
// S-17 j_1 = 0.  S-18 score = |det| (pivot_rule 0, Eq. (9)) or Frobenius (rule 1,
// listing L219/L224); used rows AND columns excluded; ties -> lowest index; all |det| = 0 but some
// Frobenius != 0 -> Frobenius for that search; pivot with |det| < 1e-30 -> stop at current rank,
// flag 2.  The default is the listing as printed (L221: the pivot block is inverted, nothing else): kappa_max =
// infinity.  S-18b is an explicit OPT-IN (orc_h_set_kappa_max): a pivot block with cond_F(P) = |P|_F |P^-1|_F >
// kappa_max is then treated as numerically singular: Alg. 2 breaks down, the block is flagged (flag 2) and the
// mat-vec evaluates it densely like an inadmissible block (L252), which is exact (S-18b).
// S-19 norm recursion via 3x3 Gram matrices A_pk = sum_i C_p(i)^T c_k(i),
// B_kp = sum_j q_k(j) Q_p(j)^T:  nu^2 = tr(A_kk B_kk), cross term tr(A_pk B_kp).
// S-20 stop when nu <= zeta*lambda, lambda including the current term.  S-21 degenerate cases.
struct AcaOut {
  int rank = 0;
  int flag = 0;                 // 1 = hit max rank without meeting Eq. (10), 2 = singular pivot
  std::vector<double> C, Q;     // C[k][i][9], Q[k][j][9]
  std::vector<int32_t> piv_i, piv_j;
  std::vector<double> nu, lam;  // per step (after the step)
  int replay_bad = 0;           // replay mode: number of pivot / stop decisions outside the slack (and, if a unit
                                // roundoff u > 0 is given, outside the rounding bound of the replayed arithmetic)
  int replay_bad_strict = 0;    // same count with the slack alone (u = 0)
};

// ---- replay-mode rounding model (checker only; does not touch the oracle's own arithmetic) ----
// "any pivot sequence in which each pivot is an arg-max UP TO ROUNDING and the stop test holds UP TO
// ROUNDING is a correct run of Alg. 2".  When the replayed run was computed with unit roundoff u (fp32: 2^-24), a
// residual entry E(i,j) = G(i,j) - sum_p C_p(i) Q_p(j) carries the running error bound
//   err(i,j) = u * [ K_G |G(i,j)|_F + sum_p (K_T + kappa_p) |C_p(i)|_F |Q_p(j)|_F ],   kappa_p = |P_p|_F |P_p^-1|_F,
// K_G = 128 (the 4-32-32-9 MLP: 68 fused multiply-adds deep with |W| row sums up to ~10, 2-ulp tanh, feature
// division), K_T = 16 (3x3 product, subtraction, stored operands), kappa_p because the normalised column
// carries the entry noise of its residual amplified by the inverse pivot block.
const double K_G = 128.0, K_T = 16.0;

void adj33(const double* A, double* J) {
  J[0] = A[4] * A[8] - A[5] * A[7]; J[1] = A[2] * A[7] - A[1] * A[8]; J[2] = A[1] * A[5] - A[2] * A[4];
  J[3] = A[5] * A[6] - A[3] * A[8]; J[4] = A[0] * A[8] - A[2] * A[6]; J[5] = A[2] * A[3] - A[0] * A[5];
  J[6] = A[3] * A[7] - A[4] * A[6]; J[7] = A[1] * A[6] - A[0] * A[7]; J[8] = A[0] * A[4] - A[1] * A[3];
}
// how far score(A + E) can be from score(A) when |E|_F <= e
double score_slop(const double* A, int rule, double e) {
  if (rule != 0) return e;                                       // | |A+E|_F - |A|_F | <= |E|_F
  double J[9];
  adj33(A, J);
  double a = std::sqrt(fro2(A));
  return std::sqrt(fro2(J)) * e + 2.0 * a * e * e + e * e * e;   // d det = <adj(A)^T, E> + O(E^2)
}

double score_of(const double* A, int rule) { return rule == 0 ? std::fabs(det33(A)) : std::sqrt(fro2(A)); }

// argmax over unused indices, ties -> lowest index; det rule falls back to Frobenius when all zero.
int argmax_score(const std::vector<double>& v, int n, const std::vector<char>& used, int rule,
                 double* best_out, int* rule_used) {
  int best = -1;
  double bs = -1;
  for (int t = 0; t < n; ++t) {
    if (used[t]) continue;
    double s = score_of(&v[9 * (size_t)t], rule);
    if (s > bs) { bs = s; best = t; }
  }
  *rule_used = rule;
  if (rule == 0 && best >= 0 && bs == 0.0) {
    int b2 = -1;
    double s2 = -1;
    for (int t = 0; t < n; ++t) {
      if (used[t]) continue;
      double s = score_of(&v[9 * (size_t)t], 1);
      if (s > s2) { s2 = s; b2 = t; }
    }
    if (s2 > 0) { best = b2; bs = s2; *rule_used = 1; }
  }
  *best_out = bs;
  return best;
}

// replay: if rp_rank >= 0 the run uses the given pivots (rp_i[k], rp_j[k]) and rank, and counts
// decisions that are not an arg-max / a correct stop within `slack` (relative).
void aca_block(const HMat& h, const Mlp& mlp, double a, int32_t tnode, int32_t snode, double zeta,
               int max_rank, int rule, int rp_rank, const int32_t* rp_i, const int32_t* rp_j,
               double slack, AcaOut& out, double u_round = 0.0, double kappa_max = INFINITY, int rp_flag = 0,
               double dense_cap = 128.0) {
  const Node& T = h.nodes[tnode];
  const Node& S = h.nodes[snode];
  int c = (int)(T.hi - T.lo), q = (int)(S.hi - S.lo);
  const float* Xt = &h.Xs[3 * T.lo];
  const float* Xs = &h.Xs[3 * S.lo];
  int kmax = std::min(std::min(c, q), max_rank);
  bool replay = rp_rank >= 0;
  // a replayed run that broke down (flag 2) lists rp_rank accepted pivots plus the attempted one
  const int rp_len = replay ? rp_rank + (rp_flag == 2 ? 1 : 0) : 0;
  if (replay) kmax = std::min(kmax, rp_len);
  // S-18b applies where the dense evaluation is affordable: |tau||sigma| <= dense_cap (|tau| + |sigma|); a larger
  // block keeps the ill-conditioned pivot, as the plain listing does
  const bool dense_ok = (double)c * (double)q <= dense_cap * ((double)c + (double)q);
  std::vector<char> used_r(c, 0), used_c(q, 0);
  std::vector<double> ck((size_t)9 * c), qk((size_t)9 * q);
  std::vector<double> errc(c, 0.0), errq(q, 0.0), kappa;        // replay-mode rounding bounds (checker only)
  double lam2 = 0;
  int jk = 0;                                                   // S-17
  out = AcaOut();
  bool met = false;
  for (int k = 0; k < kmax; ++k) {
    if (replay) {
      if (k == 0 && rp_j[0] != 0) out.replay_bad++;
      jk = rp_j[k];
    }
    // line 4: column residual
    for (int i = 0; i < c; ++i) {
      double g[9];
      entry2(mlp, a, Xt + 3 * i, Xs + 3 * jk, g);
      double eb = K_G * std::sqrt(fro2(g));
      for (int p = 0; p < k; ++p) {
        double t[9];
        mul33(&out.C[((size_t)p * c + i) * 9], &out.Q[((size_t)p * q + jk) * 9], t);
        for (int e = 0; e < 9; ++e) g[e] -= t[e];
        if (replay) eb += (K_T + kappa[p]) * std::sqrt(fro2(&out.C[((size_t)p * c + i) * 9]) * fro2(&out.Q[((size_t)p * q + jk) * 9]));
      }
      errc[i] = u_round * eb;
      std::memcpy(&ck[9 * (size_t)i], g, sizeof g);
    }
    // line 5: row pivot
    double best;
    int ru;
    int ik = argmax_score(ck, c, used_r, rule, &best, &ru);
    if (ik < 0 || best == 0.0) { met = true; break; }           // S-21: zero residual column
    if (replay) {
      int gi = rp_i[k];
      if (gi < 0 || gi >= c || used_r[gi]) { out.replay_bad++; out.replay_bad_strict++; gi = ik; }
      else {
        double sg = score_of(&ck[9 * (size_t)gi], ru);
        if (sg < (1.0 - slack) * best) {
          out.replay_bad_strict++;
          double hi = sg + score_slop(&ck[9 * (size_t)gi], ru, errc[gi]);
          double lo = std::max(0.0, best - score_slop(&ck[9 * (size_t)ik], ru, errc[ik]));
          if (hi < (1.0 - slack) * lo) out.replay_bad++;
        }
      }
      ik = gi;
    }
    double P[9], Pinv[9];
    std::memcpy(P, &ck[9 * (size_t)ik], sizeof P);
    double dP = det33(P);
    const bool attempted = replay && rp_flag == 2 && k == rp_rank;       // the step at which the replayed run broke down
    if (std::fabs(dP) < 1e-30) {                                 // S-18: singular pivot -> breakdown, block goes dense
      if (replay && !attempted) { out.replay_bad++; out.replay_bad_strict++; }
      out.flag = 2;
      out.piv_i.push_back(ik); out.piv_j.push_back(jk);          // the attempted pivot, listed after the rank accepted ones
      break;
    }
    inv33(P, dP, Pinv);
    const double kap = std::sqrt(fro2(P) * fro2(Pinv)), pinv_n = std::sqrt(fro2(Pinv));
    if (!replay && dense_ok && kap > kappa_max) {                // S-18b: numerically singular pivot
      out.flag = 2;
      out.piv_i.push_back(ik); out.piv_j.push_back(jk);
      break;
    }
    // replay: cond_F of the pivot block as the replayed arithmetic can have seen it.  A perturbation of size
    // e = errc[ik] moves the smallest singular value (~ 1/|P^-1|_F) by up to e.
    const double e_piv = errc[ik] * pinv_n;
    const double kap_lo = kap / (1.0 + e_piv), kap_hi = e_piv < 1.0 ? kap / (1.0 - e_piv) : INFINITY;
    if (attempted) {                                             // replay: the breakdown must be plausible (factor 2 on cond)
      if (kap < 0.5 * kappa_max || !dense_ok) { out.replay_bad_strict++; if (kap_hi < 0.5 * kappa_max || !dense_ok) out.replay_bad++; }
      out.flag = 2;
      out.piv_i.push_back(ik); out.piv_j.push_back(jk);
      break;
    }
    if (replay && dense_ok && kap > 2.0 * kappa_max) {           // should have broken down here
      out.replay_bad_strict++;
      if (kap_lo > 2.0 * kappa_max) out.replay_bad++;
    }
    double dc2 = 0;                                             // rounding bound of the normalised column, squared
    // line 6: c_k <- c_k P^{-1}
    for (int i = 0; i < c; ++i) {
      double t[9];
      mul33(&ck[9 * (size_t)i], Pinv, t);
      std::memcpy(&ck[9 * (size_t)i], t, sizeof t);
      double d = errc[i] * pinv_n + u_round * (K_T + kap) * std::sqrt(fro2(t));
      dc2 += d * d;
    }
    // line 7: row residual
    for (int j = 0; j < q; ++j) {
      double g[9];
      entry2(mlp, a, Xt + 3 * ik, Xs + 3 * j, g);
      double eb = K_G * std::sqrt(fro2(g));
      for (int p = 0; p < k; ++p) {
        double t[9];
        mul33(&out.C[((size_t)p * c + ik) * 9], &out.Q[((size_t)p * q + j) * 9], t);
        for (int e = 0; e < 9; ++e) g[e] -= t[e];
        if (replay) eb += (K_T + kappa[p]) * std::sqrt(fro2(&out.C[((size_t)p * c + ik) * 9]) * fro2(&out.Q[((size_t)p * q + j) * 9]));
      }
      errq[j] = u_round * eb;
      std::memcpy(&qk[9 * (size_t)j], g, sizeof g);
    }
    kappa.push_back(kap);
    used_r[ik] = 1;
    used_c[jk] = 1;
    // line 8: next column pivot
    double bestc;
    int ruc;
    int jn = argmax_score(qk, q, used_c, rule, &bestc, &ruc);
    if (replay && k + 1 < rp_len && jn >= 0) {
      int gj = rp_j[k + 1];
      if (gj < 0 || gj >= q || used_c[gj]) { out.replay_bad++; out.replay_bad_strict++; }
      else {
        double sg = score_of(&qk[9 * (size_t)gj], ruc);
        if (sg < (1.0 - slack) * bestc) {
          out.replay_bad_strict++;
          double hi = sg + score_slop(&qk[9 * (size_t)gj], ruc, errq[gj]);
          double lo = std::max(0.0, bestc - score_slop(&qk[9 * (size_t)jn], ruc, errq[jn]));
          if (hi < (1.0 - slack) * lo) out.replay_bad++;
        }
      }
    }
    // lines 9-10: norm recursion (S-19)
    double Akk[9] = {0}, Bkk[9] = {0};
    for (int i = 0; i < c; ++i) {
      const double* v = &ck[9 * (size_t)i];                     // A_kk += v^T v
      for (int r = 0; r < 3; ++r)
        for (int s = 0; s < 3; ++s) Akk[3 * r + s] += v[r] * v[s] + v[3 + r] * v[3 + s] + v[6 + r] * v[6 + s];
    }
    for (int j = 0; j < q; ++j) {
      const double* v = &qk[9 * (size_t)j];                     // B_kk += v v^T
      for (int r = 0; r < 3; ++r)
        for (int s = 0; s < 3; ++s) Bkk[3 * r + s] += v[3 * r] * v[3 * s] + v[3 * r + 1] * v[3 * s + 1] + v[3 * r + 2] * v[3 * s + 2];
    }
    double AB[9];
    mul33(Akk, Bkk, AB);
    double nu2 = AB[0] + AB[4] + AB[8];
    double cross = 0;
    for (int p = 0; p < k; ++p) {
      double Apk[9] = {0}, Bkp[9] = {0};
      for (int i = 0; i < c; ++i) {
        const double* u = &out.C[((size_t)p * c + i) * 9];
        const double* v = &ck[9 * (size_t)i];                   // A_pk += u^T v
        for (int r = 0; r < 3; ++r)
          for (int s = 0; s < 3; ++s) Apk[3 * r + s] += u[r] * v[s] + u[3 + r] * v[3 + s] + u[6 + r] * v[6 + s];
      }
      for (int j = 0; j < q; ++j) {
        const double* u = &qk[9 * (size_t)j];
        const double* v = &out.Q[((size_t)p * q + j) * 9];      // B_kp += u v^T
        for (int r = 0; r < 3; ++r)
          for (int s = 0; s < 3; ++s) Bkp[3 * r + s] += u[3 * r] * v[3 * s] + u[3 * r + 1] * v[3 * s + 1] + u[3 * r + 2] * v[3 * s + 2];
      }
      double T2[9];
      mul33(Apk, Bkp, T2);
      cross += T2[0] + T2[4] + T2[8];
    }
    lam2 += nu2 + 2.0 * cross;
    // line 11: append (C is stored [k][i][9], Q [k][j][9]; resize keeps earlier columns)
    out.C.resize((size_t)(k + 1) * c * 9);
    out.Q.resize((size_t)(k + 1) * q * 9);
    std::memcpy(&out.C[(size_t)k * c * 9], ck.data(), sizeof(double) * 9 * c);
    std::memcpy(&out.Q[(size_t)k * q * 9], qk.data(), sizeof(double) * 9 * q);
    out.piv_i.push_back(ik);
    out.piv_j.push_back(jk);
    double nu = std::sqrt(std::max(nu2, 0.0)), lam = std::sqrt(std::max(lam2, 0.0));
    out.nu.push_back(nu);
    out.lam.push_back(lam);
    out.rank = k + 1;
    // line 12: Eq. (10) stop test (S-20)
    bool stop = nu <= zeta * lam;
    if (replay) {
      bool last = (k + 1 == rp_rank) && rp_flag != 2;
      // rounding bound of nu = |c_k q_k^T|_F:  |d nu| <= |dc|_F |q|_F + |c|_F |dq|_F
      double dq2 = 0, cn2 = 0, qn2 = 0;
      for (int j = 0; j < q; ++j) { dq2 += errq[j] * errq[j]; qn2 += fro2(&qk[9 * (size_t)j]); }
      for (int i = 0; i < c; ++i) cn2 += fro2(&ck[9 * (size_t)i]);
      const double dnu = std::sqrt(dc2 * qn2) + std::sqrt(cn2 * dq2);
      if (!last && nu <= zeta * lam * (1.0 - slack)) {                          // oracle would clearly have stopped
        out.replay_bad_strict++;
        if (nu + dnu <= zeta * lam * (1.0 - slack)) out.replay_bad++;
      }
      if (last && k + 1 < std::min(std::min(c, q), max_rank) && nu > zeta * lam * (1.0 + slack) &&
          jn >= 0 && bestc > 0.0) {                                             // GPU stopped clearly early
        out.replay_bad_strict++;
        if (nu - dnu > zeta * lam * (1.0 + slack)) out.replay_bad++;
      }
      // the replayed run chose to stop here: that choice is judged above; S-21's flag 1 is only "the rank cap
      // N_ite_max was reached without meeting Eq. (10)"
      if (last) { met = stop || (k + 1 < std::min(std::min(c, q), max_rank)); break; }
    } else {
      if (stop) { met = true; break; }
    }
    if (jn < 0) { met = true; break; }
    jk = jn;
  }
  if (!met && out.flag == 0 && out.rank == kmax && kmax < std::min(c, q)) out.flag = 1;   // S-21
}

struct Handle {
  HMat h;
  Mlp mlp2;
  double a = 1.0;
  double u_round = 0.0;         // replay checker: unit roundoff of the replayed arithmetic (0 = slack only)
  double kappa_max = INFINITY;  // S-18b (opt-in): pivot blocks with cond_F above this break Alg. 2 down (block goes dense); default = the plain listing (L221)
  double dense_cap = 128.0;     // S-18b only where |tau||sigma| <= dense_cap (|tau| + |sigma|)
  int64_t last_bad_strict = 0;  // slack-only count of the last replay call
};

}  // namespace

// =============================================================================================
// C ABI (ctypes).  All float arrays are fp32 inputs or fp64 outputs as named.
// =============================================================================================
extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_mlp_forward(const int* dims, int nl, const float* params, const double* x, double* y) {
  Mlp m = make_mlp(dims, nl, params);
  mlp_forward(m, x, y);
}

void orc_entry2(const int* dims, int nl, const float* params, double a, const float* Xi,
                const float* Xj, double* M9) {
  Mlp m = make_mlp(dims, nl, params);
  entry2(m, a, Xi, Xj, M9);
}

// O-dense: U_i = F_i + sum_{j != i} M_ij F_j   (Eq. (2)/(6); S-5: alpha_1 = I, diagonal of M^(t,2) zero)
void orc_dense_matvec(int64_t N, const float* X, const float* F, const int* dims, int nl,
                      const float* params, double a, int include_self, double* U) {
  Mlp m = make_mlp(dims, nl, params);
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t i = 0; i < N; ++i) {
    double u[3] = {0, 0, 0};
    if (include_self) for (int c = 0; c < 3; ++c) u[c] = (double)F[3 * i + c];
    for (int64_t j = 0; j < N; ++j) {
      if (j == i) continue;
      double M[9], f[3] = {(double)F[3 * j], (double)F[3 * j + 1], (double)F[3 * j + 2]};
      entry2(m, a, X + 3 * i, X + 3 * j, M);
      mat3_vec_acc(M, f, u);
    }
    for (int c = 0; c < 3; ++c) U[3 * i + c] = u[c];
  }
}

// rows of the dense product for a subset of targets (sampled eps_r at large N)
void orc_dense_rows(int64_t N, const float* X, const float* F, const int* dims, int nl,
                    const float* params, double a, int include_self, int64_t nrows,
                    const int64_t* rows, double* U) {
  Mlp m = make_mlp(dims, nl, params);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t t = 0; t < nrows; ++t) {
    int64_t i = rows[t];
    double u[3] = {0, 0, 0};
    if (include_self) for (int c = 0; c < 3; ++c) u[c] = (double)F[3 * i + c];
    for (int64_t j = 0; j < N; ++j) {
      if (j == i) continue;
      double M[9], f[3] = {(double)F[3 * j], (double)F[3 * j + 1], (double)F[3 * j + 2]};
      entry2(m, a, X + 3 * i, X + 3 * j, M);
      mat3_vec_acc(M, f, u);
    }
    for (int c = 0; c < 3; ++c) U[3 * t + c] = u[c];
  }
}

// Three-body term by the literal O(N^3) triple loop over ordered distinct (i, j, k).  U += .
void orc_three_body_brute(int64_t N, const float* X, const float* F, const int* dims, int nl,
                          const float* params, float rcut, double* U, int64_t* n_faces) {
  Mlp m = make_mlp(dims, nl, params);
  int64_t nf = 0;
  for (int64_t k = 0; k < N; ++k)
    for (int64_t i = 0; i < N; ++i) {
      if (i == k || !within_cut_f32(X + 3 * i, X + 3 * k, rcut)) continue;
      for (int64_t j = 0; j < N; ++j) {
        if (j == k || j == i || !within_cut_f32(X + 3 * j, X + 3 * k, rcut)) continue;
        face_term(m, X + 3 * i, X + 3 * j, X + 3 * k, F + 3 * j, U + 3 * i);
        ++nf;
      }
    }
  if (n_faces) *n_faces = nf;
}

// Same sum with a plain cell list (cell side >= Rcut) for the neighbour search (S-24).  U += .
void orc_three_body(int64_t N, const float* X, const float* F, const int* dims, int nl,
                    const float* params, float rcut, double* U, int64_t* n_faces) {
  Mlp m = make_mlp(dims, nl, params);
  if (N == 0 || !(rcut > 0)) { if (n_faces) *n_faces = 0; return; }
  double lo[3] = {X[0], X[1], X[2]}, hi[3] = {X[0], X[1], X[2]};
  for (int64_t i = 0; i < N; ++i)
    for (int c = 0; c < 3; ++c) { lo[c] = std::min(lo[c], (double)X[3 * i + c]); hi[c] = std::max(hi[c], (double)X[3 * i + c]); }
  double cs = (double)rcut * 1.0001;
  int64_t nc[3];
  for (int c = 0; c < 3; ++c) nc[c] = std::max<int64_t>(1, std::min<int64_t>(1024, (int64_t)std::floor((hi[c] - lo[c]) / cs) + 1));
  double cw[3];
  for (int c = 0; c < 3; ++c) cw[c] = std::max(cs, (hi[c] - lo[c]) / (double)nc[c] * 1.0000001);
  auto cell_of = [&](const float* p, int64_t* ijk) {
    for (int c = 0; c < 3; ++c) ijk[c] = std::min<int64_t>(nc[c] - 1, (int64_t)std::floor(((double)p[c] - lo[c]) / cw[c]));
  };
  std::vector<std::vector<int64_t>> cells((size_t)(nc[0] * nc[1] * nc[2]));
  for (int64_t i = 0; i < N; ++i) {
    int64_t c3[3];
    cell_of(X + 3 * i, c3);
    cells[(size_t)((c3[0] * nc[1] + c3[1]) * nc[2] + c3[2])].push_back(i);
  }
  int64_t nf = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : nf)
  for (int64_t k = 0; k < N; ++k) {
    int64_t c3[3];
    cell_of(X + 3 * k, c3);
    std::vector<int64_t> nb;                                 // N(k)
    for (int64_t dx = -1; dx <= 1; ++dx)
      for (int64_t dy = -1; dy <= 1; ++dy)
        for (int64_t dz = -1; dz <= 1; ++dz) {
          int64_t x = c3[0] + dx, y = c3[1] + dy, z = c3[2] + dz;
          if (x < 0 || y < 0 || z < 0 || x >= nc[0] || y >= nc[1] || z >= nc[2]) continue;
          for (int64_t p : cells[(size_t)((x * nc[1] + y) * nc[2] + z)])
            if (p != k && within_cut_f32(X + 3 * p, X + 3 * k, rcut)) nb.push_back(p);
        }
    std::sort(nb.begin(), nb.end());
    for (int64_t i : nb)
      for (int64_t j : nb) {
        if (i == j) continue;
        double u[3] = {0, 0, 0};
        face_term(m, X + 3 * i, X + 3 * j, X + 3 * k, F + 3 * j, u);
        for (int c = 0; c < 3; ++c) {
#pragma omp atomic
          U[3 * i + c] += u[c];
        }
        ++nf;
      }
  }
  if (n_faces) *n_faces = nf;
}

// The diagonal (self) terms of Eq. (6):  U_i += [ M^(s,2)_ii + M^(s,3)_ii ] F_i  with
//   M^(s,2)_ii = sum_{j != i, |X_j - X_i| < R_cut} alpha_2^(s)(X_i, X_j)          (Eq. (2); cutoff L56)
//   M^(s,3)_ii = sum_{faces (j,k,i): i, j in N(k), j != i} alpha_3^(s)(X_i, X_k, X_j)
// from the first 9 outputs of the 18-output networks.  Plain loops: every N(k) by an O(N) scan.  U += .
void orc_self_terms(int64_t N, const float* X, const float* F, const int* dims2, int nl2, const float* params2,
                    const int* dims3, int nl3, const float* params3, double a, float rcut, double* U,
                    int64_t* n_pairs, int64_t* n_faces) {
  int64_t np = 0, nf = 0;
  if (dims2 && dims2[nl2] == 18) {
    Mlp m2 = make_mlp(dims2, nl2, params2);
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : np)
    for (int64_t i = 0; i < N; ++i) {
      double S[9] = {0};
      for (int64_t j = 0; j < N; ++j) {
        if (j == i || !within_cut_f32(X + 3 * j, X + 3 * i, rcut)) continue;
        double M[9];
        entry2_self(m2, a, X + 3 * i, X + 3 * j, M);
        for (int t = 0; t < 9; ++t) S[t] += M[t];
        ++np;
      }
      for (int al = 0; al < 3; ++al)
        U[3 * i + al] += S[3 * al] * (double)F[3 * i] + S[3 * al + 1] * (double)F[3 * i + 1] + S[3 * al + 2] * (double)F[3 * i + 2];
    }
  }
  if (dims3 && dims3[nl3] == 18) {
    Mlp m3 = make_mlp(dims3, nl3, params3);
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : nf)
    for (int64_t k = 0; k < N; ++k) {
      std::vector<int64_t> nb;
      for (int64_t p = 0; p < N; ++p)
        if (p != k && within_cut_f32(X + 3 * p, X + 3 * k, rcut)) nb.push_back(p);
      for (int64_t i : nb)
        for (int64_t j : nb) {
          if (i == j) continue;
          double u[3] = {0, 0, 0};
          face_term(m3, X + 3 * i, X + 3 * j, X + 3 * k, F + 3 * i, u, true);
          for (int c = 0; c < 3; ++c) {
#pragma omp atomic
            U[3 * i + c] += u[c];
          }
          ++nf;
        }
    }
  }
  if (n_pairs) *n_pairs = np;
  if (n_faces) *n_faces = nf;
}

void orc_morton_keys(int64_t N, const float* X, uint64_t* keys) { morton_keys(N, X, keys); }

// ---- O-H handle: tree + block lists for (X, leaf, eta); two-body MLP and radius a -------------
void* orc_h_create(int64_t N, const float* X, int leaf, double eta, const int* dims, int nl,
                   const float* params, double a) {
  Handle* H = new Handle();
  H->h.N = N;
  H->h.leaf = leaf;
  H->h.eta = eta;
  H->h.X.assign(X, X + 3 * N);
  H->mlp2 = make_mlp(dims, nl, params);
  H->a = a;
  build_tree(H->h);
  build_partition(H->h, 0, 0);
  return H;
}
void orc_h_destroy(void* p) { delete (Handle*)p; }
// replay checker: unit roundoff of the arithmetic being replayed (2^-24 for the fp32 CUDA path; 0 = slack only)
void orc_h_set_replay_roundoff(void* p, double u) { ((Handle*)p)->u_round = u; }
void orc_h_set_kappa_max(void* p, double k) { ((Handle*)p)->kappa_max = k; }
void orc_h_set_dense_cap(void* p, double c) { ((Handle*)p)->dense_cap = c; }
int64_t orc_h_last_bad_strict(void* p) { return ((Handle*)p)->last_bad_strict; }

void orc_h_counts(void* p, int64_t* n_nodes, int64_t* n_leaves, int64_t* nG, int64_t* nH, int64_t* depth) {
  Handle* H = (Handle*)p;
  *n_nodes = (int64_t)H->h.nodes.size();
  int64_t nl = 0, d = 0;
  for (auto& nd : H->h.nodes) { if (nd.left < 0) ++nl; d = std::max<int64_t>(d, nd.level); }
  *n_leaves = nl;
  *nG = (int64_t)H->h.G.size();
  *nH = (int64_t)H->h.H.size();
  *depth = d;
}

void orc_h_get_tree(void* p, int64_t* perm, uint64_t* keys, int64_t* lo, int64_t* hi, int32_t* left,
                    int32_t* right, int32_t* parent, int32_t* level, float* bmin, float* bmax) {
  Handle* H = (Handle*)p;
  std::copy(H->h.perm.begin(), H->h.perm.end(), perm);
  std::copy(H->h.keys.begin(), H->h.keys.end(), keys);
  for (size_t t = 0; t < H->h.nodes.size(); ++t) {
    const Node& nd = H->h.nodes[t];
    lo[t] = nd.lo; hi[t] = nd.hi; left[t] = nd.left; right[t] = nd.right;
    parent[t] = nd.parent; level[t] = nd.level;
    for (int c = 0; c < 3; ++c) { bmin[3 * t + c] = nd.bmin[c]; bmax[3 * t + c] = nd.bmax[c]; }
  }
}

// blocks as node-id pairs: which = 0 -> P^G, 1 -> P^H
void orc_h_get_blocks(void* p, int which, int32_t* tau, int32_t* sigma) {
  Handle* H = (Handle*)p;
  auto& L = which == 0 ? H->h.G : H->h.H;
  for (size_t t = 0; t < L.size(); ++t) { tau[t] = L[t].first; sigma[t] = L[t].second; }
}

int orc_h_admissible(void* p, int32_t t, int32_t s) { return admissible(((Handle*)p)->h, t, s) ? 1 : 0; }

// One block of Alg. 2.  C_out [rank][c][9], Q_out [rank][q][9] (capacity cap_rank); returns rank.
// rp_rank < 0: free run.  rp_rank >= 0: replay with the given pivots (see aca_block).
int orc_h_aca_block(void* p, int64_t gblock, double zeta, int max_rank, int rule, int rp_rank, int rp_flag,
                    const int32_t* rp_i, const int32_t* rp_j, double slack, int cap_rank,
                    double* C_out, double* Q_out, int32_t* piv_i, int32_t* piv_j, double* nu,
                    double* lam, int* flag, int* replay_bad) {
  Handle* H = (Handle*)p;
  auto pr = H->h.G[(size_t)gblock];
  AcaOut o;
  aca_block(H->h, H->mlp2, H->a, pr.first, pr.second, zeta, max_rank, rule, rp_rank, rp_i, rp_j, slack, o, H->u_round,
            H->kappa_max, rp_flag, H->dense_cap);
  H->last_bad_strict = o.replay_bad_strict;
  int c = (int)(H->h.nodes[pr.first].hi - H->h.nodes[pr.first].lo);
  int q = (int)(H->h.nodes[pr.second].hi - H->h.nodes[pr.second].lo);
  int r = std::min(o.rank, cap_rank);
  if (C_out) std::memcpy(C_out, o.C.data(), sizeof(double) * (size_t)r * c * 9);
  if (Q_out) std::memcpy(Q_out, o.Q.data(), sizeof(double) * (size_t)r * q * 9);
  for (int k = 0; k < r; ++k) {
    if (piv_i) piv_i[k] = o.piv_i[k];
    if (piv_j) piv_j[k] = o.piv_j[k];
    if (nu) nu[k] = o.nu[k];
    if (lam) lam[k] = o.lam[k];
  }
  if (o.flag == 2 && r == o.rank && r < cap_rank && (int)o.piv_i.size() > r) {   // attempted pivot of a breakdown
    if (piv_i) piv_i[r] = o.piv_i[r];
    if (piv_j) piv_j[r] = o.piv_j[r];
  }
  if (flag) *flag = o.flag;
  if (replay_bad) *replay_bad = o.replay_bad;
  return o.rank;
}

// dense evaluation of one admissible block (for error-vs-SVD / error-vs-zeta pins): G_out [c][q][9]
void orc_h_dense_block(void* p, int64_t gblock, double* G_out) {
  Handle* H = (Handle*)p;
  auto pr = H->h.G[(size_t)gblock];
  const Node& T = H->h.nodes[pr.first];
  const Node& S = H->h.nodes[pr.second];
  int c = (int)(T.hi - T.lo), q = (int)(S.hi - S.lo);
  for (int i = 0; i < c; ++i)
    for (int j = 0; j < q; ++j)
      entry2(H->mlp2, H->a, &H->h.Xs[3 * (T.lo + i)], &H->h.Xs[3 * (S.lo + j)], &G_out[((size_t)i * q + j) * 9]);
}

// O-H mat-vec: U = F (self, S-5) + near-field dense blocks (L252, pair i == j skipped) +
// far-field C (Q F^sigma) (L115, L260).  F, U in CALLER order.  Optional replay: for admissible
// block g (oracle order) use rank rp_rank[g] and pivots rp_i/rp_j[rp_off[g] ...].
// ranks_out[g], flags_out[g] (optional); returns the number of replay decisions outside slack.
// only_rows: if non-null (tree-order flags, length N) only rows with flag 1 are produced (sampled
// parity at large N): blocks whose tau range contains no flagged row are skipped.
int64_t orc_h_matvec(void* p, const float* F, double zeta, int max_rank, int rule, int include_self,
                     int do_near, int do_far, const int32_t* rp_rank, const int32_t* rp_flag, const int64_t* rp_off,
                     const int32_t* rp_i, const int32_t* rp_j, double slack,
                     const uint8_t* only_rows, double* U, int32_t* ranks_out, int32_t* flags_out,
                     int64_t* n_entries) {
  Handle* Hd = (Handle*)p;
  HMat& h = Hd->h;
  int64_t N = h.N;
  std::vector<double> Fs(3 * N), Us(3 * N, 0.0);
  for (int64_t k = 0; k < N; ++k)
    for (int c = 0; c < 3; ++c) Fs[3 * k + c] = (double)F[3 * h.perm[k] + c];
  if (include_self) for (int64_t t = 0; t < 3 * N; ++t) Us[t] = Fs[t];
  auto touches = [&](const Node& T) {
    if (!only_rows) return true;
    for (int64_t k = T.lo; k < T.hi; ++k) if (only_rows[k]) return true;
    return false;
  };
  int64_t entries = 0, bad = 0, bad_strict = 0;
  if (do_near) {
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : entries)
    for (int64_t b = 0; b < (int64_t)h.H.size(); ++b) {
      const Node& T = h.nodes[h.H[b].first];
      const Node& S = h.nodes[h.H[b].second];
      if (!touches(T)) continue;
      for (int64_t i = T.lo; i < T.hi; ++i) {
        double u[3] = {0, 0, 0};
        for (int64_t j = S.lo; j < S.hi; ++j) {
          if (i == j) continue;                                  // S-5
          double M[9];
          entry2(Hd->mlp2, Hd->a, &h.Xs[3 * i], &h.Xs[3 * j], M);
          mat3_vec_acc(M, &Fs[3 * j], u);
          ++entries;
        }
        for (int c = 0; c < 3; ++c) {
#pragma omp atomic
          Us[3 * i + c] += u[c];
        }
      }
    }
  }
  if (do_far) {
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : entries, bad, bad_strict)
    for (int64_t g = 0; g < (int64_t)h.G.size(); ++g) {
      const Node& T = h.nodes[h.G[g].first];
      const Node& S = h.nodes[h.G[g].second];
      if (!touches(T)) { if (ranks_out) ranks_out[g] = -1; continue; }
      int c = (int)(T.hi - T.lo), q = (int)(S.hi - S.lo);
      AcaOut o;
      if (rp_rank)
        aca_block(h, Hd->mlp2, Hd->a, h.G[g].first, h.G[g].second, zeta, max_rank, rule, rp_rank[g],
                  rp_i + rp_off[g], rp_j + rp_off[g], slack, o, Hd->u_round, Hd->kappa_max, rp_flag ? rp_flag[g] : 0,
                  Hd->dense_cap);
      else
        aca_block(h, Hd->mlp2, Hd->a, h.G[g].first, h.G[g].second, zeta, max_rank, rule, -1, nullptr, nullptr, 0.0, o, 0.0,
                  Hd->kappa_max, 0, Hd->dense_cap);
      entries += (int64_t)o.rank * (c + q);
      bad += o.replay_bad;
      bad_strict += o.replay_bad_strict;
      if (ranks_out) ranks_out[g] = o.rank;
      if (flags_out) flags_out[g] = o.flag;
      if (o.flag == 2) {                                         // S-18b: Alg. 2 broke down -> the block is applied densely (L252)
        entries += (int64_t)c * q;
        for (int64_t i = T.lo; i < T.hi; ++i) {
          double u[3] = {0, 0, 0};
          for (int64_t j = S.lo; j < S.hi; ++j) {
            double M[9];
            entry2(Hd->mlp2, Hd->a, &h.Xs[3 * i], &h.Xs[3 * j], M);
            mat3_vec_acc(M, &Fs[3 * j], u);
          }
          for (int e = 0; e < 3; ++e) {
#pragma omp atomic
            Us[3 * i + e] += u[e];
          }
        }
        continue;
      }
      for (int k = 0; k < o.rank; ++k) {
        double t[3] = {0, 0, 0};                                 // t = Q_k F^sigma
        for (int j = 0; j < q; ++j) mat3_vec_acc(&o.Q[((size_t)k * q + j) * 9], &Fs[3 * (S.lo + j)], t);
        for (int i = 0; i < c; ++i) {                            // U^tau += C_k t
          double u[3] = {0, 0, 0};
          mat3_vec_acc(&o.C[((size_t)k * c + i) * 9], t, u);
          for (int e = 0; e < 3; ++e) {
#pragma omp atomic
            Us[3 * (T.lo + i) + e] += u[e];
          }
        }
      }
    }
  }
  for (int64_t k = 0; k < N; ++k)
    for (int c = 0; c < 3; ++c) U[3 * h.perm[k] + c] = Us[3 * k + c];
  if (n_entries) *n_entries = entries;
  Hd->last_bad_strict = bad_strict;
  return bad;
}

// S-25: X <- X + dt U in fp32 (L338)
void orc_euler(int64_t N, float* X, const double* U, float dt) {
  for (int64_t t = 0; t < 3 * N; ++t) X[t] = X[t] + dt * (float)U[t];
}

}  // extern "C"
