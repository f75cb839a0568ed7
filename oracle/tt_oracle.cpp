// oracle/tt_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, fp64 CPU oracle for the triangle-triangle intersection energy of
// arXiv 2606.06511.  It follows the paper's Appendix A listing
// step by step, in the listing's order and notation, with its own
// forward-mode dual numbers (value + 18 partials) -- the same technique the listing uses
// (PAPER.md L51, L59).  It shares no code with the CUDA path (which differentiates the
// end-points analytically) and is only ever imported by tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs.
//
// Every function is pinned by tests/test_oracle_*.py (-m "not gpu") against hand-worked
// examples, closed forms, invariants, finite differences and brute force; nothing here is
// "parity unpinned".  Readings of garbled/ambiguous passages (A1..A15) are listed in DESIGN.md.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC  (no -ffast-math; A14).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int NDOF = 18;  // x = [a0,a1,a2,b0,b1,b2], 6 vertices x 3 (`loc`)

// ---- forward-mode dual number: value + 18 partials (stands in for autodiff::dual, L59) ----
struct Dual {
  double val;
  double d[NDOF];
};

inline Dual constant(double c) {
  Dual r;
  r.val = c;
  for (int i = 0; i < NDOF; ++i) r.d[i] = 0.0;
  return r;
}
inline Dual variable(double c, int idx) {
  Dual r = constant(c);
  r.d[idx] = 1.0;
  return r;
}
inline Dual operator+(const Dual& a, const Dual& b) {
  Dual r;
  r.val = a.val + b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] + b.d[i];
  return r;
}
inline Dual operator-(const Dual& a, const Dual& b) {
  Dual r;
  r.val = a.val - b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] - b.d[i];
  return r;
}
inline Dual operator*(const Dual& a, const Dual& b) {
  Dual r;
  r.val = a.val * b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] * b.val + a.val * b.d[i];
  return r;
}
inline Dual operator*(double s, const Dual& a) {
  Dual r;
  r.val = s * a.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = s * a.d[i];
  return r;
}
inline Dual operator/(const Dual& a, const Dual& b) {
  Dual r;
  r.val = a.val / b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = (a.d[i] - r.val * b.d[i]) / b.val;
  return r;
}
inline Dual dsqrt(const Dual& a) {
  Dual r;
  r.val = std::sqrt(a.val);
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] / (2.0 * r.val);
  return r;
}
// min/max on duals select value AND partials of the selected argument (App. A).
inline Dual dmin(const Dual& a, const Dual& b) { return (b.val < a.val) ? b : a; }
inline Dual dmax(const Dual& a, const Dual& b) { return (b.val > a.val) ? b : a; }

// ---- second-order forward-mode dual number: value + 18 first + 18 x 18 second partials ----------
// Used only for the EXACT Hessian (second half: the terms Eq. 4 drops, PAPER.md L26
// "ignoring the asymmetric part of the exact Hessian").  The same listing code below runs on either
// dual type (it is a template on the scalar), so the exact Hessian is App. A differentiated twice.
struct Dual2 {
  double val;
  double d[NDOF];
  double h[NDOF][NDOF];
};
inline Dual2 constant2(double c) {
  Dual2 r;
  std::memset(&r, 0, sizeof(r));
  r.val = c;
  return r;
}
inline Dual2 operator+(const Dual2& a, const Dual2& b) {
  Dual2 r;
  r.val = a.val + b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] + b.d[i];
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) r.h[i][j] = a.h[i][j] + b.h[i][j];
  return r;
}
inline Dual2 operator-(const Dual2& a, const Dual2& b) {
  Dual2 r;
  r.val = a.val - b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] - b.d[i];
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) r.h[i][j] = a.h[i][j] - b.h[i][j];
  return r;
}
inline Dual2 operator*(const Dual2& a, const Dual2& b) {  // (ab)'' = a''b + a b'' + a'b'^T + b'a'^T
  Dual2 r;
  r.val = a.val * b.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] * b.val + a.val * b.d[i];
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j)
      r.h[i][j] = a.h[i][j] * b.val + a.val * b.h[i][j] + a.d[i] * b.d[j] + b.d[i] * a.d[j];
  return r;
}
inline Dual2 operator*(double s, const Dual2& a) {
  Dual2 r;
  r.val = s * a.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = s * a.d[i];
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) r.h[i][j] = s * a.h[i][j];
  return r;
}
inline Dual2 operator/(const Dual2& a, const Dual2& b) {  // a * (1/b): (1/b)' = -b'/b^2, (1/b)'' = 2 b'b'^T/b^3 - b''/b^2
  Dual2 q;
  const double v = 1.0 / b.val;
  q.val = v;
  for (int i = 0; i < NDOF; ++i) q.d[i] = -v * v * b.d[i];
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) q.h[i][j] = 2.0 * v * v * v * b.d[i] * b.d[j] - v * v * b.h[i][j];
  return a * q;
}
inline Dual2 dsqrt(const Dual2& a) {  // s = sqrt(a): s' = a'/(2s), s'' = a''/(2s) - a'a'^T/(4 s^3)
  Dual2 r;
  r.val = std::sqrt(a.val);
  const double s = r.val;
  for (int i = 0; i < NDOF; ++i) r.d[i] = a.d[i] / (2.0 * s);
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) r.h[i][j] = a.h[i][j] / (2.0 * s) - a.d[i] * a.d[j] / (4.0 * s * s * s);
  return r;
}
inline Dual2 dmin(const Dual2& a, const Dual2& b) { return (b.val < a.val) ? b : a; }
inline Dual2 dmax(const Dual2& a, const Dual2& b) { return (b.val > a.val) ? b : a; }

// seeds: the idx-th independent variable
template <class D> D seed(double c, int idx);
template <> inline Dual seed<Dual>(double c, int idx) { return variable(c, idx); }
template <> inline Dual2 seed<Dual2>(double c, int idx) {
  Dual2 r = constant2(c);
  r.d[idx] = 1.0;
  return r;
}

template <class D>
struct Vec3T {
  D x, y, z;
};
using Vec3 = Vec3T<Dual>;
template <class D> inline Vec3T<D> operator+(const Vec3T<D>& a, const Vec3T<D>& b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
template <class D> inline Vec3T<D> operator-(const Vec3T<D>& a, const Vec3T<D>& b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
template <class D> inline Vec3T<D> operator*(const D& s, const Vec3T<D>& a) { return {s * a.x, s * a.y, s * a.z}; }
template <class D> inline Vec3T<D> operator*(double s, const Vec3T<D>& a) { return {s * a.x, s * a.y, s * a.z}; }
template <class D> inline Vec3T<D> operator/(const Vec3T<D>& a, const D& s) { return {a.x / s, a.y / s, a.z / s}; }
template <class D> inline D dot(const Vec3T<D>& a, const Vec3T<D>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class D> inline Vec3T<D> cross(const Vec3T<D>& a, const Vec3T<D>& b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
template <class D> inline Vec3T<D> normalized(const Vec3T<D>& a) {  // Vector3dual::normalize()
  D n = dsqrt(dot(a, a));
  return a / n;
}

// ---- App. A `intersects` -----------------------------------------------
// Plane triangle (U0,U1,U2) cuts triangle (V0,V1,V2); on success segment0/1 are the two
// end-points of the cut.  Readings A1-A4 of DESIGN.md.
template <class D>
bool intersects(const Vec3T<D>& U0, const Vec3T<D>& U1, const Vec3T<D>& U2, const Vec3T<D>& V0, const Vec3T<D>& V1,
                const Vec3T<D>& V2, Vec3T<D>& segment0, Vec3T<D>& segment1) {
  using Vec3 = Vec3T<D>;
  using Dual = D;
  Vec3 edge1 = U1 - U0;                  // L78
  Vec3 edge2 = U2 - U0;                  // L79
  Vec3 normal = cross(edge1, edge2);     // L80
  // A degenerate plane triangle has no normal: "not coplanar" precondition (L11) fails.
  if (!(dot(normal, normal).val > 0.0)) return false;
  normal = normalized(normal);           // L81
  Dual d[3];
  int positive = 0, negative = 0, zero = 0;  // L83
  d[0] = dot(normal, V0 - U0);           // L84
  d[1] = dot(normal, V1 - U1);           // L85 (as printed: U1; n.(U1-U0) == 0 identically, A1)
  d[2] = dot(normal, V2 - U2);           // L86 (as printed: U2)
  for (int i = 0; i < 3; ++i) {          // L87-93 (A2)
    if (d[i].val > 0.0) ++positive;
    else if (d[i].val < 0.0) ++negative;
    else ++zero;
  }
  const Vec3* V[3] = {&V0, &V1, &V2};
  // crossing point of edge (V_i, V_k): (d_i V_k - d_k V_i) / (d_i - d_k)  (L100-101, L104-105)
  auto crossing = [&](int i, int k) -> Vec3 {
    return (d[i] * (*V[k]) - d[k] * (*V[i])) / (d[i] - d[k]);
  };
  if (positive > 0 && negative > 0) {    // L95
    if (positive == 2 || negative == 2) {  // L96 / L102: two on one side, one alone (A3)
      int k;                               // the lone vertex
      if (positive == 2) k = (d[0].val < 0.0) ? 0 : (d[1].val < 0.0) ? 1 : 2;
      else               k = (d[0].val > 0.0) ? 0 : (d[1].val > 0.0) ? 1 : 2;
      int i = (k + 1) % 3, j = (k + 2) % 3;
      // printed instances: k=1 -> (0,1),(2,1) at L100-101;  k=2 -> (0,2),(1,2) at L104-105.
      if (i > j) std::swap(i, j);
      segment0 = crossing(i, k);
      segment1 = crossing(j, k);
    } else {                              // L106: positive == 1, negative == 1, zero == 1 (A4)
      int z = (d[0].val == 0.0) ? 0 : (d[1].val == 0.0) ? 1 : 2;
      int i = (z + 1) % 3, j = (z + 2) % 3;
      segment0 = *V[z];                   // L109 / L112: the vertex lying on the plane
      segment1 = crossing(j, i);          // L110 prints (d2 V1 - d1 V2)/(d2 - d1) for z = 0
    }
    return true;                          // L117
  }
  return false;                           // L120
}

struct PairResult {
  bool active;
  double tc[2];
  double g[2][NDOF];  // g[0] = d tc0 / dx, g[1] = d tc1 / dx   (x = [a0,a1,a2,b0,b1,b2])
};

// ---- App. A `3DTTIT` + Eq. 1 ------------------------------------------
// x holds T_a = (a0,a1,a2) then T_b = (b0,b1,b2).  The listing names the triangle whose
// segment is S00/S01 (interval I_a) `U` and the other `V`; so U := T_a, V := T_b, and the dual
// seeds are placed so that partial index 3m+c is a_m[c] and 9+3m+c is b_m[c].
// (template on the dual type D: first order for Eq. 3 / Eq. 4, second order for the exact Hessian)
template <class D>
bool ttit_core(const double x[NDOF], double sigma, D& tc0_out, D& tc1_out) {
  using Vec3 = Vec3T<D>;
  using Dual = D;
  Vec3 U[3], V[3];
  for (int m = 0; m < 3; ++m) {
    U[m] = {seed<D>(x[3 * m + 0], 3 * m + 0), seed<D>(x[3 * m + 1], 3 * m + 1), seed<D>(x[3 * m + 2], 3 * m + 2)};
    V[m] = {seed<D>(x[9 + 3 * m + 0], 9 + 3 * m + 0), seed<D>(x[9 + 3 * m + 1], 9 + 3 * m + 1),
            seed<D>(x[9 + 3 * m + 2], 9 + 3 * m + 2)};
  }
  Vec3 S00, S01, S10, S11;
  if (intersects(V[0], V[1], V[2], U[0], U[1], U[2], S00, S01) &&   // L134: plane(V) cuts U
      intersects(U[0], U[1], U[2], V[0], V[1], V[2], S10, S11)) {   // L135: plane(U) cuts V
    Vec3 uNormal = cross(U[1] - U[0], U[2] - U[0]);                  // L137
    Vec3 vNormal = cross(V[1] - V[0], V[2] - V[0]);                  // L139
    Vec3 Dv = cross(uNormal, vNormal);                               // L141 (the listing's D)
    if (!(dot(Dv, Dv).val > 0.0)) return false;  // parallel planes: excluded by L11 ("not coplanar")
    Dv = normalized(Dv);                                             // L142
    Vec3 A = 0.25 * (S00 + S01 + S10 + S11);                         // L144
    Dual t00 = dot(Dv, S00 - A);                                     // L145
    Dual t01 = dot(Dv, S01 - A);
    Dual t10 = dot(Dv, S10 - A);
    Dual t11 = dot(Dv, S11 - A);
    Dual ta0 = dmin(t00, t01);                                       // L149
    Dual ta1 = dmax(t00, t01);
    Dual tb0 = dmin(t10, t11);
    Dual tb1 = dmax(t10, t11);
    bool intersected = (ta1.val > tb0.val && ta0.val < tb1.val);     // L153
    if (!intersected) return false;                                  // A11: tc := (0,0)
    tc0_out = sigma * (ta0 - tb1);   // Eq. 1 (L13) with sigma = 1; L154 prints sigma = 0.5 (A6)
    tc1_out = sigma * (ta1 - tb0);   // L155
    return true;
  }
  return false;
}

PairResult pair_3dttit(const double x[NDOF], double sigma) {
  PairResult r;
  r.active = false;
  r.tc[0] = r.tc[1] = 0.0;
  std::memset(r.g, 0, sizeof(r.g));
  Dual tc0, tc1;
  if (ttit_core<Dual>(x, sigma, tc0, tc1)) {
    r.active = true;
    r.tc[0] = tc0.val;
    r.tc[1] = tc1.val;
    for (int i = 0; i < NDOF; ++i) {
      r.g[0][i] = tc0.d[i];
      r.g[1][i] = tc1.d[i];
    }
  }
  return r;
}

// Exact Hessian of one pair (NEXT-3, second half): T = (tc0 tc1)^2 evaluated in second-order duals, so
// H_exact = the second partials of T itself -- Eq. 4 plus the terms 2 tc0 tc1^2 d2tc0 + 2 tc1 tc0^2 d2tc1
// that PAPER.md L26 drops.  Also returns tc, the gradient and the two second-derivative matrices.
bool pair_exact(const double x[NDOF], double sigma, double tc[2], double* T, double grad[NDOF], double* H /*[18*18]*/,
                double* H0 /*[18*18] or NULL*/, double* H1) {
  Dual2 tc0, tc1;
  if (!ttit_core<Dual2>(x, sigma, tc0, tc1)) return false;
  const Dual2 prod = tc0 * tc1;
  const Dual2 E = prod * prod;   // Eq. 2
  tc[0] = tc0.val;
  tc[1] = tc1.val;
  *T = E.val;
  for (int i = 0; i < NDOF; ++i) grad[i] = E.d[i];
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) {
      H[NDOF * i + j] = E.h[i][j];
      if (H0) H0[NDOF * i + j] = tc0.h[i][j];
      if (H1) H1[NDOF * i + j] = tc1.h[i][j];
    }
  return true;
}

// Eq. 2 (L17)
inline double energy_of(const double tc[2]) {
  double p = tc[0] * tc[1];
  return p * p;
}

// Eq. 3 coefficients (L21-24): grad = cg[0] g0 + cg[1] g1
inline void grad_coeffs(const double tc[2], double cg[2]) {
  cg[0] = 2.0 * tc[0] * (tc[1] * tc[1]);
  cg[1] = 2.0 * tc[1] * (tc[0] * tc[0]);
}

// Eq. 4 coefficients (L26-33) + eigenanalysis reading A7 (L47):
// H = c00 g0 g0^T + c11 g1 g1^T + c01 (g1 g0^T + g0 g1^T)
//   mode 0 EQ4    : all three parts verbatim
//   mode 1 FILTER : third part kept iff L47's quantity 8 tc0 tc1 (g0.g1) >= 0
//   mode 2 PSD2   : parts one and two only
inline void hess_coeffs(const double tc[2], const double g0[NDOF], const double g1[NDOF], int mode,
                        double c[3], double lam[3]) {
  double n0 = 0.0, n1 = 0.0, g01 = 0.0;
  for (int i = 0; i < NDOF; ++i) {
    n0 += g0[i] * g0[i];
    n1 += g1[i] * g1[i];
    g01 += g0[i] * g1[i];
  }
  lam[0] = 2.0 * (tc[1] * tc[1]) * n0;   // L47, first part
  lam[1] = 2.0 * (tc[0] * tc[0]) * n1;   // L47, second part
  lam[2] = 8.0 * tc[0] * tc[1] * g01;    // L47, third part ("might be negative")
  c[0] = 2.0 * (tc[1] * tc[1]);
  c[1] = 2.0 * (tc[0] * tc[0]);
  double keep = 1.0;
  if (mode == 1) keep = (lam[2] >= 0.0) ? 1.0 : 0.0;
  if (mode == 2) keep = 0.0;
  c[2] = 4.0 * tc[0] * tc[1] * keep;
}

// mode 3 PSDPROJ (the literal "eigenanalysis" of L47 carried through): the
// per-pair Hessian is the projection of Eq. 4's 18x18 matrix onto the positive semi-definite cone,
//   H+ = sum_i max(lambda_i, 0) v_i v_i^T,   H_EQ4 = sum_i lambda_i v_i v_i^T,
// written out as that definition: cyclic Jacobi eigen-decomposition of the dense symmetric matrix
// (no use of its rank-2 structure; the GPU path uses a closed 2x2 form instead).
inline void jacobi_eigh(double* A /*[n*n], destroyed: diagonal = eigenvalues*/, double* V /*[n*n] columns*/, int n) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) V[i * n + j] = (i == j) ? 1.0 : 0.0;
  for (int sweep = 0; sweep < 64; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) (i == j ? diag : off) += A[i * n + j] * A[i * n + j];
    if (off <= 1e-60 + 1e-32 * diag) break;
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = A[p * n + q];
        if (apq == 0.0) continue;
        const double theta = (A[q * n + q] - A[p * n + p]) / (2.0 * apq);
        const double t = (theta >= 0.0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        const double c = 1.0 / std::sqrt(t * t + 1.0), sn = t * c;
        for (int k = 0; k < n; ++k) {  // A <- A R (columns p, q)
          const double akp = A[k * n + p], akq = A[k * n + q];
          A[k * n + p] = c * akp - sn * akq;
          A[k * n + q] = sn * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {  // A <- R^T A (rows p, q)
          const double apk = A[p * n + k], aqk = A[q * n + k];
          A[p * n + k] = c * apk - sn * aqk;
          A[q * n + k] = sn * apk + c * aqk;
        }
        for (int k = 0; k < n; ++k) {  // V <- V R
          const double vkp = V[k * n + p], vkq = V[k * n + q];
          V[k * n + p] = c * vkp - sn * vkq;
          V[k * n + q] = sn * vkp + c * vkq;
        }
      }
  }
}
// Dense per-pair Hessian in the given mode.  Modes 0-2: Eq. 4 with hess_coeffs; mode 3: PSD projection.
inline void pair_hessian(const double tc[2], const double g0[NDOF], const double g1[NDOF], int mode,
                         double H[NDOF * NDOF]) {
  double c[3], lam[3];
  hess_coeffs(tc, g0, g1, mode == 3 ? 0 : mode, c, lam);
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j)
      H[i * NDOF + j] = c[0] * g0[i] * g0[j] + c[1] * g1[i] * g1[j] + c[2] * (g1[i] * g0[j] + g0[i] * g1[j]);
  if (mode != 3) return;
  double A[NDOF * NDOF], V[NDOF * NDOF];
  std::memcpy(A, H, sizeof(A));
  jacobi_eigh(A, V, NDOF);
  for (int i = 0; i < NDOF; ++i)
    for (int j = 0; j < NDOF; ++j) {
      double s = 0.0;
      for (int k = 0; k < NDOF; ++k) {
        const double lk = A[k * NDOF + k];
        if (lk > 0.0) s += lk * V[i * NDOF + k] * V[j * NDOF + k];
      }
      H[i * NDOF + j] = s;
    }
}

inline bool share_vertex(const int32_t* ta, const int32_t* tb) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      if (ta[i] == tb[j]) return true;
  return false;
}

inline void gather_x(const double* pos, const int32_t* tris, const int32_t* pr, double x[NDOF],
                     int32_t vid[6]) {
  const int32_t* ta = tris + 3 * (int64_t)pr[0];
  const int32_t* tb = tris + 3 * (int64_t)pr[1];
  for (int m = 0; m < 3; ++m) {
    vid[m] = ta[m];
    vid[3 + m] = tb[m];
  }
  for (int v = 0; v < 6; ++v)
    for (int c = 0; c < 3; ++c) x[3 * v + c] = pos[3 * (int64_t)vid[v] + c];
}

// Neumaier-compensated accumulation (oracle step 12)
struct Neumaier {
  double s = 0.0, c = 0.0;
  void add(double v) {
    double t = s + v;
    if (std::fabs(s) >= std::fabs(v)) c += (s - t) + v;
    else c += (v - t) + s;
    s = t;
  }
  double value() const { return s + c; }
};

}  // namespace

extern "C" {

// One pair given as 18 coordinates x = [a0,a1,a2,b0,b1,b2].  Any output pointer may be NULL.
// H is dense 18x18 row-major; lam = L47's three printed quantities.
void tt_oracle_pair(const double* x, double sigma, int hess_mode, int* active, double* tc,
                    double* energy, double* g0, double* g1, double* grad, double* H, double* lam) {
  PairResult r = pair_3dttit(x, sigma);
  if (active) *active = r.active ? 1 : 0;
  if (tc) { tc[0] = r.tc[0]; tc[1] = r.tc[1]; }
  double T = r.active ? energy_of(r.tc) : 0.0;
  if (energy) *energy = T;
  if (g0) std::memcpy(g0, r.g[0], sizeof(double) * NDOF);
  if (g1) std::memcpy(g1, r.g[1], sizeof(double) * NDOF);
  double cg[2] = {0, 0}, c[3] = {0, 0, 0}, l[3] = {0, 0, 0};
  if (r.active) {
    grad_coeffs(r.tc, cg);
    hess_coeffs(r.tc, r.g[0], r.g[1], hess_mode, c, l);
  }
  if (grad)
    for (int i = 0; i < NDOF; ++i) grad[i] = cg[0] * r.g[0][i] + cg[1] * r.g[1][i];
  if (H) {
    if (r.active) pair_hessian(r.tc, r.g[0], r.g[1], hess_mode, H);
    else std::memset(H, 0, sizeof(double) * NDOF * NDOF);
  }
  if (lam) { lam[0] = l[0]; lam[1] = l[1]; lam[2] = l[2]; }
}

// Steps 1-9 for every candidate pair.  Outputs (each may be NULL): active[P] (0/1), tc[P,2],
// T[P], J[P,2,18] (zero rows for inactive pairs).  Returns sum of T (Neumaier, ascending order).
// Pairs sharing a vertex index are "topologically adjacent" (L11, A9) -> inactive.
double tt_oracle_pairs(const double* pos, int64_t n_verts, const int32_t* tris, int64_t n_tris,
                       const int32_t* pairs, int64_t n_pairs, double sigma, uint8_t* active,
                       double* tc, double* T, double* J, int n_threads) {
  (void)n_verts; (void)n_tris;
  std::vector<double> Tloc((size_t)n_pairs, 0.0);
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < n_pairs; ++k) {
    const int32_t* pr = pairs + 2 * k;
    PairResult r;
    r.active = false;
    if (!share_vertex(tris + 3 * (int64_t)pr[0], tris + 3 * (int64_t)pr[1])) {
      double x[NDOF];
      int32_t vid[6];
      gather_x(pos, tris, pr, x, vid);
      r = pair_3dttit(x, sigma);
    }
    if (active) active[k] = r.active ? 1 : 0;
    if (tc) { tc[2 * k] = r.active ? r.tc[0] : 0.0; tc[2 * k + 1] = r.active ? r.tc[1] : 0.0; }
    Tloc[k] = r.active ? energy_of(r.tc) : 0.0;
    if (J) {
      if (r.active) {
        std::memcpy(J + 36 * k, r.g[0], sizeof(double) * NDOF);
        std::memcpy(J + 36 * k + 18, r.g[1], sizeof(double) * NDOF);
      } else {
        std::memset(J + 36 * k, 0, sizeof(double) * 36);
      }
    }
  }
  Neumaier acc;
  for (int64_t k = 0; k < n_pairs; ++k) acc.add(Tloc[k]);
  if (T) std::memcpy(T, Tloc.data(), sizeof(double) * (size_t)n_pairs);
  return acc.value();
}

// Step 12, pattern: sorted-unique (p,q) over the 6x6 vertex pairs of every active pair.
// Writes rowptr[nV+1]; if colind != NULL (capacity >= returned nnzb) also writes colind.
int64_t tt_oracle_bsr_pattern(int64_t n_verts, const int32_t* tris, const int32_t* pairs,
                              int64_t n_pairs, const uint8_t* active, int32_t* rowptr,
                              int32_t* colind) {
  std::vector<uint64_t> keys;
  for (int64_t k = 0; k < n_pairs; ++k) {
    if (!active[k]) continue;
    int32_t vid[6];
    for (int m = 0; m < 3; ++m) {
      vid[m] = tris[3 * (int64_t)pairs[2 * k] + m];
      vid[3 + m] = tris[3 * (int64_t)pairs[2 * k + 1] + m];
    }
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) keys.push_back(((uint64_t)(uint32_t)vid[i] << 32) | (uint32_t)vid[j]);
  }
  std::sort(keys.begin(), keys.end());
  keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
  for (int64_t v = 0; v <= n_verts; ++v) rowptr[v] = 0;
  for (uint64_t key : keys) rowptr[(key >> 32) + 1] += 1;
  for (int64_t v = 0; v < n_verts; ++v) rowptr[v + 1] += rowptr[v];
  if (colind)
    for (size_t i = 0; i < keys.size(); ++i) colind[i] = (int32_t)(keys[i] & 0xffffffffu);
  return (int64_t)keys.size();
}

// Steps 10-12, numeric: grad[nV,3] and vals[nnzb,3,3] (row-major blocks) accumulated in
// ASCENDING PAIR ORDER from the per-pair J = [g0; g1] and tc produced by tt_oracle_pairs.
// rowptr/colind are the pattern from tt_oracle_bsr_pattern.  grad / vals may be NULL.
void tt_oracle_assemble(int64_t n_verts, const int32_t* tris, const int32_t* pairs, int64_t n_pairs,
                        const uint8_t* active, const double* tc, const double* J, int hess_mode,
                        const int32_t* rowptr, const int32_t* colind, double* grad, double* vals) {
  if (grad) std::memset(grad, 0, sizeof(double) * 3 * (size_t)n_verts);
  if (vals) std::memset(vals, 0, sizeof(double) * 9 * (size_t)rowptr[n_verts]);
  for (int64_t k = 0; k < n_pairs; ++k) {
    if (!active[k]) continue;
    int32_t vid[6];
    for (int m = 0; m < 3; ++m) {
      vid[m] = tris[3 * (int64_t)pairs[2 * k] + m];
      vid[3 + m] = tris[3 * (int64_t)pairs[2 * k + 1] + m];
    }
    const double* g0 = J + 36 * k;
    const double* g1 = g0 + 18;
    double cg[2], Hk[NDOF * NDOF];
    grad_coeffs(tc + 2 * k, cg);
    if (vals) pair_hessian(tc + 2 * k, g0, g1, hess_mode, Hk);
    if (grad)
      for (int v = 0; v < 6; ++v)
        for (int a = 0; a < 3; ++a)
          grad[3 * (int64_t)vid[v] + a] += cg[0] * g0[3 * v + a] + cg[1] * g1[3 * v + a];
    if (vals)
      for (int p = 0; p < 6; ++p)
        for (int q = 0; q < 6; ++q) {
          const int32_t* lo = colind + rowptr[vid[p]];
          const int32_t* hi = colind + rowptr[vid[p] + 1];
          const int32_t* it = std::lower_bound(lo, hi, vid[q]);
          double* blk = vals + 9 * (int64_t)(it - colind);
          for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) blk[3 * a + b] += Hk[(3 * p + a) * NDOF + 3 * q + b];
        }
  }
}

// H.p, way one: per active pair y_loc = J^T M (J p_loc), scattered in ascending pair order.
void tt_oracle_hess_vec_pairs(int64_t n_verts, const int32_t* tris, const int32_t* pairs,
                              int64_t n_pairs, const uint8_t* active, const double* tc,
                              const double* J, int hess_mode, const double* p, double* y) {
  std::memset(y, 0, sizeof(double) * 3 * (size_t)n_verts);
  for (int64_t k = 0; k < n_pairs; ++k) {
    if (!active[k]) continue;
    int32_t vid[6];
    for (int m = 0; m < 3; ++m) {
      vid[m] = tris[3 * (int64_t)pairs[2 * k] + m];
      vid[3 + m] = tris[3 * (int64_t)pairs[2 * k + 1] + m];
    }
    const double* g0 = J + 36 * k;
    const double* g1 = g0 + 18;
    if (hess_mode == 3) {   // y_loc = H+ p_loc with the dense projected matrix
      double Hk[NDOF * NDOF];
      pair_hessian(tc + 2 * k, g0, g1, 3, Hk);
      for (int i = 0; i < NDOF; ++i) {
        double acc = 0.0;
        for (int j = 0; j < NDOF; ++j) acc += Hk[i * NDOF + j] * p[3 * (int64_t)vid[j / 3] + j % 3];
        y[3 * (int64_t)vid[i / 3] + i % 3] += acc;
      }
      continue;
    }
    double c[3], lam[3];
    hess_coeffs(tc + 2 * k, g0, g1, hess_mode, c, lam);
    double s0 = 0.0, s1 = 0.0;   // J p_loc
    for (int v = 0; v < 6; ++v)
      for (int a = 0; a < 3; ++a) {
        s0 += g0[3 * v + a] * p[3 * (int64_t)vid[v] + a];
        s1 += g1[3 * v + a] * p[3 * (int64_t)vid[v] + a];
      }
    double u0 = c[0] * s0 + c[2] * s1;   // M (J p_loc),  M = [[c00, c01], [c01, c11]]
    double u1 = c[2] * s0 + c[1] * s1;
    for (int v = 0; v < 6; ++v)
      for (int a = 0; a < 3; ++a) y[3 * (int64_t)vid[v] + a] += u0 * g0[3 * v + a] + u1 * g1[3 * v + a];
  }
}

// H.p, way two: plain BSR (3x3 row-major blocks) times vector.
void tt_oracle_bsr_matvec(int64_t n_verts, const int32_t* rowptr, const int32_t* colind,
                          const double* vals, const double* p, double* y) {
  for (int64_t r = 0; r < n_verts; ++r) {
    double acc[3] = {0, 0, 0};
    for (int32_t e = rowptr[r]; e < rowptr[r + 1]; ++e) {
      const double* blk = vals + 9 * (int64_t)e;
      const double* pv = p + 3 * (int64_t)colind[e];
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) acc[a] += blk[3 * a + b] * pv[b];
    }
    for (int a = 0; a < 3; ++a) y[3 * r + a] = acc[a];
  }
}

// Broad phase (PAPER.md L51 names spatial hashing [Pabst et al. 2010] and gives
// no detail, so the operation is defined by its RESULT): all pairs i < j of triangles that share no
// vertex index and whose axis-aligned bounding boxes, each grown by `inflate` on every side, overlap
// (closed intervals), in lexicographic order.  Written out as that definition: every pair is tested.
// Pass pairs = NULL to count; returns the number of pairs (written only up to `capacity`).
int64_t tt_oracle_broad_phase(const double* pos, const int32_t* tris, int64_t n_tris, double inflate,
                              int32_t* pairs, int64_t capacity) {
  std::vector<double> lo(3 * (size_t)n_tris), hi(3 * (size_t)n_tris);
  for (int64_t t = 0; t < n_tris; ++t)
    for (int c = 0; c < 3; ++c) {
      double a = pos[3 * (int64_t)tris[3 * t] + c], b = pos[3 * (int64_t)tris[3 * t + 1] + c],
             d = pos[3 * (int64_t)tris[3 * t + 2] + c];
      lo[3 * t + c] = std::min(a, std::min(b, d)) - inflate;
      hi[3 * t + c] = std::max(a, std::max(b, d)) + inflate;
    }
  std::vector<int64_t> cnt((size_t)n_tris + 1, 0);
  for (int pass = 0; pass < 2; ++pass) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n_tris; ++i) {
      int64_t k = pass ? cnt[i] : 0;
      for (int64_t j = i + 1; j < n_tris; ++j) {
        bool ov = true;
        for (int c = 0; c < 3; ++c) ov = ov && lo[3 * i + c] <= hi[3 * j + c] && lo[3 * j + c] <= hi[3 * i + c];
        if (!ov || share_vertex(tris + 3 * i, tris + 3 * j)) continue;
        if (pass) {
          if (k < capacity) {
            pairs[2 * k] = (int32_t)i;
            pairs[2 * k + 1] = (int32_t)j;
          }
        }
        ++k;
      }
      if (!pass) cnt[i + 1] = k;
    }
    if (!pass) {
      for (int64_t i = 0; i < n_tris; ++i) cnt[i + 1] += cnt[i];  // cnt[i] = first output slot of row i
      if (!pairs) break;
    }
  }
  return cnt[n_tris];
}

// ---- exact Hessian (second half; the terms Eq. 4 ignores) -------------
// One pair: active flag, tc, T, gradient (18), exact Hessian H (18 x 18), and the second derivatives of
// tc0 / tc1 (H0, H1; may be NULL).  Inactive pairs: everything zero.
void tt_oracle_pair_exact(const double* x, double sigma, int* active, double* tc, double* T, double* grad,
                          double* H, double* H0, double* H1) {
  std::memset(grad, 0, sizeof(double) * NDOF);
  std::memset(H, 0, sizeof(double) * NDOF * NDOF);
  if (H0) std::memset(H0, 0, sizeof(double) * NDOF * NDOF);
  if (H1) std::memset(H1, 0, sizeof(double) * NDOF * NDOF);
  tc[0] = tc[1] = 0.0;
  *T = 0.0;
  *active = pair_exact(x, sigma, tc, T, grad, H, H0, H1) ? 1 : 0;
}

// y = H_exact p, summed over the active pairs in ascending pair order (adjacent pairs skipped, L11).
void tt_oracle_exact_hess_vec(const double* pos, int64_t n_verts, const int32_t* tris, const int32_t* pairs,
                              int64_t n_pairs, double sigma, const double* p, double* y) {
  for (int64_t i = 0; i < 3 * n_verts; ++i) y[i] = 0.0;
  std::vector<double> yl((size_t)n_pairs * NDOF, 0.0);
  std::vector<uint8_t> act((size_t)n_pairs, 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t k = 0; k < n_pairs; ++k) {
    const int32_t* pr = pairs + 2 * k;
    if (share_vertex(tris + 3 * (int64_t)pr[0], tris + 3 * (int64_t)pr[1])) continue;
    double x[NDOF], tc[2], T, grad[NDOF];
    int32_t vid[6];
    gather_x(pos, tris, pr, x, vid);
    std::vector<double> H(NDOF * NDOF);
    if (!pair_exact(x, sigma, tc, &T, grad, H.data(), nullptr, nullptr)) continue;
    act[k] = 1;
    for (int i = 0; i < NDOF; ++i) {
      double a = 0.0;
      for (int j = 0; j < NDOF; ++j) a += H[NDOF * i + j] * p[3 * (int64_t)vid[j / 3] + j % 3];
      yl[(size_t)k * NDOF + i] = a;
    }
  }
  for (int64_t k = 0; k < n_pairs; ++k) {
    if (!act[k]) continue;
    int32_t vid[6];
    double x[NDOF];
    gather_x(pos, tris, pairs + 2 * k, x, vid);
    for (int i = 0; i < NDOF; ++i) y[3 * (int64_t)vid[i / 3] + i % 3] += yl[(size_t)k * NDOF + i];
  }
}

// BSR values of the EXACT Hessian: vals[nnzb,3,3] accumulated in ASCENDING PAIR ORDER from pair_exact's 18 x 18
// matrices, on the pattern tt_oracle_bsr_pattern built for the same active set (the pattern does not depend on
// the Hessian variant: every active pair fills its 6 x 6 vertex blocks).
void tt_oracle_assemble_exact(const double* pos, int64_t n_verts, const int32_t* tris, const int32_t* pairs,
                              int64_t n_pairs, const uint8_t* active, double sigma, const int32_t* rowptr,
                              const int32_t* colind, double* vals) {
  std::memset(vals, 0, sizeof(double) * 9 * (size_t)rowptr[n_verts]);
  std::vector<double> H(NDOF * NDOF);
  for (int64_t k = 0; k < n_pairs; ++k) {
    if (!active[k]) continue;
    double x[NDOF], tc[2], T, grad[NDOF];
    int32_t vid[6];
    gather_x(pos, tris, pairs + 2 * k, x, vid);
    if (!pair_exact(x, sigma, tc, &T, grad, H.data(), nullptr, nullptr)) continue;
    for (int p = 0; p < 6; ++p)
      for (int q = 0; q < 6; ++q) {
        const int32_t* lo = colind + rowptr[vid[p]];
        const int32_t* hi = colind + rowptr[vid[p] + 1];
        const int32_t* it = std::lower_bound(lo, hi, vid[q]);
        double* blk = vals + 9 * (int64_t)(it - colind);
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) blk[3 * a + b] += H[(3 * p + a) * NDOF + 3 * q + b];
      }
  }
}

// ---- inexact-Newton linear solve ("inexact Newton optimization route") ------
// The paper names the route and gives no detail, so the operations are their textbook definitions:
//   * block-Jacobi preconditioner: the inverse of every 3x3 diagonal block of (H + shift I)
//     (a row without a stored diagonal block has the block shift I);
//   * preconditioned conjugate gradients (Hestenes-Stiefel; e.g. Saad, "Iterative Methods for Sparse
//     Linear Systems", Alg. 9.1) for (H + shift I) x = b from x_0 = 0:
//         r_0 = b, z_0 = M r_0, p_0 = z_0;
//         alpha_k = (r_k.z_k)/(p_k.A p_k); x_{k+1} = x_k + alpha_k p_k; r_{k+1} = r_k - alpha_k A p_k;
//         z_{k+1} = M r_{k+1}; beta_k = (r_{k+1}.z_{k+1})/(r_k.z_k); p_{k+1} = z_{k+1} + beta_k p_k,
//     stopped before step k when |r_k|_2 <= rtol |b|_2, or after max_iter steps.
// Written out as those definitions: Gauss-Jordan with partial pivoting for the 3x3 inverses, the plain BSR
// product above for A p, Neumaier-compensated dot products.  (The GPU inverts by cofactors and sums in trees.)
void tt_oracle_block_jacobi(int64_t n_verts, const int32_t* rowptr, const int32_t* colind, const double* vals,
                            double shift, double* minv /*[n_verts,3,3]*/) {
  for (int64_t r = 0; r < n_verts; ++r) {
    double a[3][6];
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 6; ++j) a[i][j] = (j == i + 3) ? 1.0 : 0.0;
    for (int32_t e = rowptr[r]; e < rowptr[r + 1]; ++e)
      if (colind[e] == r)
        for (int i = 0; i < 3; ++i)
          for (int j = 0; j < 3; ++j) a[i][j] += vals[9 * (int64_t)e + 3 * i + j];
    for (int i = 0; i < 3; ++i) a[i][i] += shift;
    for (int c = 0; c < 3; ++c) {  // Gauss-Jordan, partial pivoting
      int piv = c;
      for (int i = c + 1; i < 3; ++i)
        if (std::fabs(a[i][c]) > std::fabs(a[piv][c])) piv = i;
      for (int j = 0; j < 6; ++j) std::swap(a[c][j], a[piv][j]);
      const double d = a[c][c];
      for (int j = 0; j < 6; ++j) a[c][j] /= d;
      for (int i = 0; i < 3; ++i)
        if (i != c) {
          const double f = a[i][c];
          for (int j = 0; j < 6; ++j) a[i][j] -= f * a[c][j];
        }
    }
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) minv[9 * r + 3 * i + j] = a[i][3 + j];
  }
}

namespace {
double ndot(const double* a, const double* b, int64_t n) {
  Neumaier s;
  for (int64_t i = 0; i < n; ++i) s.add(a[i] * b[i]);
  return s.value();
}
void apply_blocks(int64_t nv, const double* minv, const double* r, double* z) {  // z = M r; minv == NULL: identity
  for (int64_t v = 0; v < nv; ++v)
    for (int i = 0; i < 3; ++i)
      z[3 * v + i] = minv ? minv[9 * v + 3 * i] * r[3 * v] + minv[9 * v + 3 * i + 1] * r[3 * v + 1] +
                                minv[9 * v + 3 * i + 2] * r[3 * v + 2]
                          : r[3 * v + i];
}
}  // namespace

// Returns the number of steps taken.  x [n] = last iterate; x_hist (or NULL) [(max_iter+1) n]: every iterate
// x_0..x_k; res_hist (or NULL) [max_iter+1]: |r_k|_2 of the RECURRED residual.  minv: tt_oracle_block_jacobi's
// output, or NULL for plain CG.
int64_t tt_oracle_pcg(int64_t n_verts, const int32_t* rowptr, const int32_t* colind, const double* vals,
                      double shift, const double* minv, const double* b, int64_t max_iter, double rtol,
                      double* x, double* x_hist, double* res_hist) {
  const int64_t n = 3 * n_verts;
  std::vector<double> r(b, b + n), z((size_t)n), p((size_t)n), q((size_t)n);
  for (int64_t i = 0; i < n; ++i) x[i] = 0.0;
  apply_blocks(n_verts, minv, r.data(), z.data());
  p = z;
  double rz = ndot(r.data(), z.data(), n);
  const double bnorm = std::sqrt(ndot(b, b, n));
  int64_t k = 0;
  for (;; ++k) {
    const double rnorm = std::sqrt(ndot(r.data(), r.data(), n));
    if (res_hist) res_hist[k] = rnorm;
    if (x_hist) std::memcpy(x_hist + k * n, x, sizeof(double) * (size_t)n);
    if (k == max_iter || rnorm <= rtol * bnorm) break;
    tt_oracle_bsr_matvec(n_verts, rowptr, colind, vals, p.data(), q.data());
    for (int64_t i = 0; i < n; ++i) q[i] += shift * p[i];
    const double alpha = rz / ndot(p.data(), q.data(), n);
    for (int64_t i = 0; i < n; ++i) {
      x[i] += alpha * p[i];
      r[i] -= alpha * q[i];
    }
    apply_blocks(n_verts, minv, r.data(), z.data());
    const double rz_new = ndot(r.data(), z.data(), n);
    const double beta = rz_new / rz;
    rz = rz_new;
    for (int64_t i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];
  }
  return k;
}

int tt_oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
