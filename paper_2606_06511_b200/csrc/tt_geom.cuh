// tt_geom.cuh -- per-pair device arithmetic of the hot path (sm_100a), fp64 registers only.
//
// Steps a1-a3 of DESIGN.md (Eq. 1-4, App. A), written the GPU's own way:
// where the paper's listing pushes 18-partial dual numbers through Moeller's test, this file
// differentiates the four segment end-points ANALYTICALLY ("manually construct the computation
// graph to reduce the number of multiplications").  Because P - Q is parallel to
// the unit line direction D and D . dD = 0, d(D.(P-Q)) = D^T (dP - dQ): neither dD, nor the
// normalisation of the plane normals, nor the origin A of App. A L144 contribute (DESIGN.md
// "analytic form").  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace ttg {

// 3-vector over the scalar S: double everywhere a discrete decision is taken (K1) and in the fp64
// variant; float in the derivative / outer-product arithmetic of the fp32 variant (reading A12).
template <typename S>
struct v3 {
  S x, y, z;
};
using d3 = v3<double>;
template <typename S> __device__ __forceinline__ v3<S> mk(S x, S y, S z) { return v3<S>{x, y, z}; }
template <typename S> __device__ __forceinline__ v3<S> operator+(v3<S> a, v3<S> b) { return mk<S>(a.x + b.x, a.y + b.y, a.z + b.z); }
template <typename S> __device__ __forceinline__ v3<S> operator-(v3<S> a, v3<S> b) { return mk<S>(a.x - b.x, a.y - b.y, a.z - b.z); }
template <typename S> __device__ __forceinline__ v3<S> operator*(S s, v3<S> a) { return mk<S>(s * a.x, s * a.y, s * a.z); }
template <typename S> __device__ __forceinline__ S dot(v3<S> a, v3<S> b) { return fma(a.x, b.x, fma(a.y, b.y, a.z * b.z)); }
template <typename S> __device__ __forceinline__ v3<S> cross(v3<S> a, v3<S> b) {
  return mk<S>(fma(a.y, b.z, -(a.z * b.y)), fma(a.z, b.x, -(a.x * b.z)), fma(a.x, b.y, -(a.y * b.x)));
}
template <typename S> __device__ __forceinline__ v3<S> axpy(S s, v3<S> a, v3<S> b) {  // s*a + b
  return mk<S>(fma(s, a.x, b.x), fma(s, a.y, b.y), fma(s, a.z, b.z));
}
__device__ __forceinline__ double inv_sqrt(double x) { return rsqrt(x); }
__device__ __forceinline__ float inv_sqrt(float x) { return rsqrtf(x); }
__device__ __forceinline__ d3 sel3(int i, d3 v0, d3 v1, d3 v2) {
  d3 r = v2;
  if (i == 1) r = v1;
  if (i == 0) r = v0;
  return r;
}
__device__ __forceinline__ double sel3(int i, double v0, double v1, double v2) {
  double r = v2;
  if (i == 1) r = v1;
  if (i == 0) r = v0;
  return r;
}

// One cut of triangle X (vertices x[0..2], plane distances d[0..2] w.r.t. the other plane):
// two end-points E_e = x_k + tau_e (x_i - x_k), e = 0 (smaller t) and e = 1 (larger t).
// k == i encodes App. A's "vertex exactly on the plane" branch (L106-115): E = x_k, d tau = 0.
struct Cut {
  int k[2], i[2];
  double tau[2];
  double t[2];
};

// Plane-side classification + end-points of one triangle (App. A).  Returns false when
// the triangle does not strictly straddle the plane (L95 / L120).
__device__ __forceinline__ bool make_cut(const d3 x0, const d3 x1, const d3 x2, double d0, double d1,
                                         double d2, const d3 Dh, Cut& c) {
  const int pos = (d0 > 0.0) + (d1 > 0.0) + (d2 > 0.0);
  const int neg = (d0 < 0.0) + (d1 < 0.0) + (d2 < 0.0);
  if (!(pos > 0 && neg > 0)) return false;
  int k0, i0, k1, i1;
  if (pos + neg == 3) {  // two on one side, one alone: k = the lone vertex (L96-105)
    const bool s0 = d0 > 0.0, s1 = d1 > 0.0, s2 = d2 > 0.0;
    const int k = (s0 == s1) ? 2 : ((s0 == s2) ? 1 : 0);
    k0 = k1 = k;
    i0 = (k == 0) ? 1 : 0;
    i1 = (k == 2) ? 1 : 2;
  } else {  // one +, one -, one exactly 0 (L106-115): end-point 0 is the vertex itself
    const int z = (d0 == 0.0) ? 0 : ((d1 == 0.0) ? 1 : 2);
    k0 = i0 = z;
    k1 = (z == 0) ? 1 : 0;
    i1 = (z == 2) ? 1 : 2;
  }
  const double dk0 = sel3(k0, d0, d1, d2), di0 = sel3(i0, d0, d1, d2);
  const double dk1 = sel3(k1, d0, d1, d2), di1 = sel3(i1, d0, d1, d2);
  // opposite signs: |dk - di| = |dk| + |di|, no cancellation
  const double tau0 = (k0 == i0) ? 0.0 : dk0 / (dk0 - di0);
  const double tau1 = dk1 / (dk1 - di1);
  const d3 xk0 = sel3(k0, x0, x1, x2), xi0 = sel3(i0, x0, x1, x2);
  const d3 xk1 = sel3(k1, x0, x1, x2), xi1 = sel3(i1, x0, x1, x2);
  const double t0 = dot(Dh, axpy(tau0, xi0 - xk0, xk0));
  const double t1 = dot(Dh, axpy(tau1, xi1 - xk1, xk1));
  const bool sw = t1 < t0;  // min/max of App. A L149-152 (selects the argument and its partials)
  c.k[0] = sw ? k1 : k0;  c.i[0] = sw ? i1 : i0;  c.tau[0] = sw ? tau1 : tau0;  c.t[0] = sw ? t1 : t0;
  c.k[1] = sw ? k0 : k1;  c.i[1] = sw ? i0 : i1;  c.tau[1] = sw ? tau0 : tau1;  c.t[1] = sw ? t0 : t1;
  return true;
}

struct PairGeom {
  d3 na, nb, Dh;
  double alpha[3], beta[3];
  Cut ca, cb;
  double tc0, tc1;  // already multiplied by sigma
};

// Steps a1: Moeller intervals and I_c (Eq. 1; App. A).  a*, b* are the
// six vertices in any common frame (callers translate by -a0 first).  Returns the `intersected`
// flag of L153, evaluated in fp64.
__device__ __forceinline__ bool pair_intervals(const d3 a0, const d3 a1, const d3 a2, const d3 b0,
                                               const d3 b1, const d3 b2, double sigma, PairGeom& g) {
  g.na = cross(a1 - a0, a2 - a0);
  g.nb = cross(b1 - b0, b2 - b0);
  // signed (unnormalised) distances: same signs as App. A's normalised d[] (L84-86)
  g.alpha[0] = dot(g.nb, a0 - b0);
  g.alpha[1] = dot(g.nb, a1 - b0);
  g.alpha[2] = dot(g.nb, a2 - b0);
  {
    const int pos = (g.alpha[0] > 0.0) + (g.alpha[1] > 0.0) + (g.alpha[2] > 0.0);
    const int neg = (g.alpha[0] < 0.0) + (g.alpha[1] < 0.0) + (g.alpha[2] < 0.0);
    if (!(pos > 0 && neg > 0)) return false;  // early exit: most candidates leave here
  }
  g.beta[0] = dot(g.na, b0 - a0);
  g.beta[1] = dot(g.na, b1 - a0);
  g.beta[2] = dot(g.na, b2 - a0);
  {
    const int pos = (g.beta[0] > 0.0) + (g.beta[1] > 0.0) + (g.beta[2] > 0.0);
    const int neg = (g.beta[0] < 0.0) + (g.beta[1] < 0.0) + (g.beta[2] < 0.0);
    if (!(pos > 0 && neg > 0)) return false;
  }
  const d3 D = cross(g.na, g.nb);  // App. A L141 (u = T_a)
  const double D2 = dot(D, D);
  if (!(D2 > 0.0)) return false;   // parallel planes (L11 "not coplanar")
  g.Dh = rsqrt(D2) * D;            // L142
  if (!make_cut(a0, a1, a2, g.alpha[0], g.alpha[1], g.alpha[2], g.Dh, g.ca)) return false;
  if (!make_cut(b0, b1, b2, g.beta[0], g.beta[1], g.beta[2], g.Dh, g.cb)) return false;
  const double ta0 = g.ca.t[0], ta1 = g.ca.t[1], tb0 = g.cb.t[0], tb1 = g.cb.t[1];
  g.tc0 = sigma * (ta0 - tb1);     // Eq. 1 / L154
  g.tc1 = sigma * (ta1 - tb0);     // L155
  return (ta1 > tb0) && (ta0 < tb1);  // L153, strict
}

// ---- recorded branch decisions ("record the computation graph") ----------------
// K1 classifies every candidate with the generic code above and RECORDS, per active pair and per
// triangle X, the discrete decisions of App. A in 6 bits:
//   k (bits 0-1): the vertex both end-points hang off (the lone vertex, L96-105)
//   p (bits 2-3): the other vertex of the edge carrying the end-point with the SMALLER t (L149-152);
//                 q = 3 - k - p carries the larger one
//   z (bits 4-5): 1 / 2 = the smaller / larger end-point is a vertex lying exactly on the other
//                 plane (L106-115): it is then represented as the edge (k, p or q) with tau = 1
//                 and d tau := 0, which is App. A's S0 = V_z
// K4 / K6 permute the vertex IDS by (k, p, q) before gathering, so the derivative code below is
// straight-line: no sign tests, no min/max, no selects on doubles.
__device__ __forceinline__ unsigned cut_config(const Cut& c) {
  unsigned k, p, q, z;
  if (c.k[0] == c.i[0]) {         // smaller end-point is the on-plane vertex
    z = 1u; k = (unsigned)c.k[1]; p = (unsigned)c.k[0]; q = (unsigned)c.i[1];
  } else if (c.k[1] == c.i[1]) {  // larger end-point is the on-plane vertex
    z = 2u; k = (unsigned)c.k[0]; p = (unsigned)c.i[0]; q = (unsigned)c.k[1];
  } else {
    z = 0u; k = (unsigned)c.k[0]; p = (unsigned)c.i[0]; q = (unsigned)c.i[1];
  }
  (void)q;
  return k | (p << 2) | (z << 4);
}
__device__ __forceinline__ unsigned pair_config(const PairGeom& g) {
  return cut_config(g.ca) | (cut_config(g.cb) << 6);
}

// One end-point E = x_k + tau (x_e - x_k) of triangle X = (x_k, x_p, x_q) cut by plane(Y), and the
// blocks of  s * D^T dE  (s = +-sigma):
//   own blocks: (1-tau) D at x_k, tau D at x_e, plus c dtau/dx with c = D.(x_e - x_k),
//               dtau/dx_e = d_k nY / den^2, dtau/dx_k = -d_e nY / den^2, den = d_k - d_e
//   other blocks: dtau/dy_p = (y_q - y_k) x (E - y_k) / den, dtau/dy_q = (E - y_k) x (y_p - y_k) / den,
//               y_k from translation invariance (all six blocks of D^T dE sum to D).
// nY = (y_p - y_k) x (y_q - y_k) and the distances d are taken with THAT normal, so the formulas hold
// for any labelling (k, p, q) of Y (an odd one flips nY and d together).
template <typename S>
struct EndPoint {
  S t;                            // D . E
  v3<S> E;                        // the end-point itself (used by the exact Hessian only)
  v3<S> ownk, owne, yk, yp, yq;   // blocks of s D^T dE
};
// tau of an end-point that IS a vertex (zmask == 0, App. A): the vertex does not slide along its edge, so
// tau is the constant 1 -- which is what d_k / (d_k - 0) evaluates to; types that carry derivatives overload this
// to drop tau's (tt_exact.cuh).
__device__ __forceinline__ double vertex_tau(double tau, double) { return tau; }
__device__ __forceinline__ float vertex_tau(float tau, float) { return tau; }
template <typename S>
__device__ __forceinline__ EndPoint<S> end_point(S s, const v3<S> Dh, const v3<S> xk, const v3<S> ex, S dk,
                                                 S de, S zmask, const v3<S> yk, const v3<S> eyp,
                                                 const v3<S> eyq, const v3<S> nY) {
  EndPoint<S> r;
  const S inv = S(1) / (dk - de);  // opposite signs: |dk - de| = |dk| + |de|, no cancellation
  const S tau = vertex_tau(dk * inv, zmask);
  const v3<S> E = axpy(tau, ex, xk);
  r.E = E;
  r.t = dot(Dh, E);
  const S w = s * zmask * dot(Dh, ex) * inv;  // s c / den
  const S wn = w * inv;                       // s c / den^2
  r.ownk = axpy(s * (S(1) - tau), Dh, (-(wn * de)) * nY);
  r.owne = axpy(s * tau, Dh, (wn * dk) * nY);
  const v3<S> u = E - yk;
  r.yp = w * cross(eyq, u);
  r.yq = w * cross(u, eyp);
  r.yk = mk<S>(-fma(w, nY.x, r.yp.x + r.yq.x), -fma(w, nY.y, r.yp.y + r.yq.y), -fma(w, nY.z, r.yp.z + r.yq.z));
  return r;
}

// Step a3, first half, straight-line: both triangles arrive permuted to (k, p, q) as recorded.
//   g0 = d tc0/dx = sigma (D^T dE(a,p) - D^T dE(b,q)),  g1 = d tc1/dx = sigma (D^T dE(a,q) - D^T dE(b,p)),
//   x = [a_k, a_p, a_q, b_k, b_p, b_q].  The line direction is taken from the PERMUTED normals, so
//   (tc0, tc1, g0, g1) may come out as (-tc0, -tc1, -g0, -g1): Eq. 2-4 and L47's third quantity are
//   even in that sign (every term pairs two of them), so energy, gradient and Hessian are unchanged.
// What the exact Hessian (tt_exact.cuh) needs beyond g0, g1: the two interval differences as VECTORS (c0 = P_a - Q_b,
// c1 = Q_a - P_b; both parallel to D at any regular point), the normals, the edge vectors and 1 / |n_a x n_b|.
template <typename S>
struct PairAux {
  v3<S> c0, c1, na, nb, eap, eaq, ebp, ebq, Dh;
  S rinv;
};
template <typename S>
__device__ __forceinline__ void pair_derivs_core(const v3<S> ak, const v3<S> ap, const v3<S> aq, const v3<S> bk,
                                                 const v3<S> bp, const v3<S> bq, S sigma, unsigned za,
                                                 unsigned zb, S& tc0, S& tc1,
                                                 S (&g0)[18], S (&g1)[18], PairAux<S>& aux) {
  const v3<S> eap = ap - ak, eaq = aq - ak, ebp = bp - bk, ebq = bq - bk;
  const v3<S> na = cross(eap, eaq), nb = cross(ebp, ebq);
  const v3<S> ab = ak - bk;
  const S dak = dot(nb, ab), dap = dot(nb, ap - bk), daq = dot(nb, aq - bk);
  const S dbk = -dot(na, ab), dbp = dot(na, bp - ak), dbq = dot(na, bq - ak);
  const v3<S> D = cross(na, nb);
  const S rinv = inv_sqrt(dot(D, D));
  const v3<S> Dh = rinv * D;
  const EndPoint<S> Pa = end_point<S>(sigma, Dh, ak, eap, dak, dap, za == 1u ? S(0) : S(1), bk, ebp, ebq, nb);
  const EndPoint<S> Qa = end_point<S>(sigma, Dh, ak, eaq, dak, daq, za == 2u ? S(0) : S(1), bk, ebp, ebq, nb);
  const EndPoint<S> Pb = end_point<S>(-sigma, Dh, bk, ebp, dbk, dbp, zb == 1u ? S(0) : S(1), ak, eap, eaq, na);
  const EndPoint<S> Qb = end_point<S>(-sigma, Dh, bk, ebq, dbk, dbq, zb == 2u ? S(0) : S(1), ak, eap, eaq, na);
  tc0 = sigma * (Pa.t - Qb.t);  // Eq. 1
  tc1 = sigma * (Qa.t - Pb.t);
  auto put = [](S (&g)[18], int o, const v3<S> v) { g[o] = v.x; g[o + 1] = v.y; g[o + 2] = v.z; };
  put(g0, 0, Pa.ownk + Qb.yk);   put(g0, 3, Pa.owne + Qb.yp);   put(g0, 6, Qb.yq);
  put(g0, 9, Pa.yk + Qb.ownk);   put(g0, 12, Pa.yp);            put(g0, 15, Pa.yq + Qb.owne);
  put(g1, 0, Qa.ownk + Pb.yk);   put(g1, 3, Pb.yp);             put(g1, 6, Qa.owne + Pb.yq);
  put(g1, 9, Qa.yk + Pb.ownk);   put(g1, 12, Qa.yp + Pb.owne);  put(g1, 15, Qa.yq);
  aux.c0 = Pa.E - Qb.E;  aux.c1 = Qa.E - Pb.E;
  aux.na = na;  aux.nb = nb;  aux.eap = eap;  aux.eaq = eaq;  aux.ebp = ebp;  aux.ebq = ebq;  aux.Dh = Dh;  aux.rinv = rinv;
}
template <typename S>
__device__ __forceinline__ void pair_derivs_recorded(const v3<S> ak, const v3<S> ap, const v3<S> aq, const v3<S> bk,
                                                     const v3<S> bp, const v3<S> bq, S sigma, unsigned za,
                                                     unsigned zb, S& tc0, S& tc1,
                                                     S (&g0)[18], S (&g1)[18]) {
  PairAux<S> aux;  // never read here: the compiler drops it
  pair_derivs_core<S>(ak, ap, aq, bk, bp, bq, sigma, za, zb, tc0, tc1, g0, g1, aux);
}

// Step a3, second half: Eq. 3 and Eq. 4 coefficients.  keep = tt_hess_mode's treatment of the
// third part (L47): EQ4 -> 1, PSD2 -> 0, FILTER -> [8 tc0 tc1 (g0.g1) >= 0].
// PSDPROJ (mode 3): H = J^T M J has rank 2, so its projection onto the PSD cone is J^T M+ J with a
// 2x2 M+ in closed form.  With G = J J^T = L L^T (Cholesky), Q = L^-1 J has orthonormal rows and
// H = Q^T S Q, S = L^T M L; det M = -12 tc0^2 tc1^2 < 0 makes S indefinite for every active pair, so
// S+ = lambda_+ (S - lambda_- I) / (lambda_+ - lambda_-) (spectral projector of the positive
// eigenvalue) and M+ = L^-T S+ L^-1.  The coefficients (c00, c11, c01) become the entries of M+ and
// everything downstream is unchanged.  (The oracle projects the dense 18x18 matrix instead.)
template <typename S>
struct Coefs {
  S cg0, cg1;       // Eq. 3: grad = cg0 g0 + cg1 g1
  S c00, c11, c01;  // Eq. 4: H = c00 g0g0^T + c11 g1g1^T + c01 (g1g0^T + g0g1^T)
};
// PSDPROJ's 2x2 algebra, kept out of line (scalars in, scalars out): the three default modes then
// compile as without it -- K4 runs at ~254 of 255 registers and is sensitive to every live value.
// G = J J^T = [[p, q], [q, r]], M = [[a, b], [b, d]]; returns M+ as (m00, m11, m01).
struct Sym2 {
  double m00, m11, m01;
};
__device__ __noinline__ Sym2 psd_project_2x2(double p, double q, double r, double a, double b, double d) {
  Sym2 o{a, d, 0.0};  // fallback (g0 parallel to g1: cannot happen away from degenerate pairs): PSD2
  const double l11 = sqrt(p), l21 = q / l11;
  const double l22sq = r - l21 * l21;
  if (l22sq > 1e-24 * r) {
    const double l22 = sqrt(l22sq);
    // S = L^T M L
    const double t1 = a * l11 + b * l21, t2 = b * l11 + d * l21;
    const double s11 = l11 * t1 + l21 * t2, s12 = l22 * t2, s22 = l22 * l22 * d;
    const double mid = 0.5 * (s11 + s22), half = 0.5 * (s11 - s22);
    const double rad = sqrt(fma(half, half, s12 * s12));
    const double lp = mid + rad, lm = mid - rad;
    const double f = (lp > 0.0) ? lp / (lp - lm) : 0.0;  // S+ = f (S - lm I)
    const double p11 = f * (s11 - lm), p12 = f * s12, p22 = f * (s22 - lm);
    // M+ = L^-T S+ L^-1,  L^-1 = [[1/l11, 0], [-l21/(l11 l22), 1/l22]]
    const double i11 = 1.0 / l11, i22 = 1.0 / l22, i21 = -l21 * i11 * i22;
    const double u1 = p11 * i11 + p12 * i21, u2 = p12 * i11 + p22 * i21;  // (S+ L^-1)[:, 0]
    o.m00 = i11 * u1 + i21 * u2;
    o.m01 = i22 * u2;
    o.m11 = i22 * i22 * p22;
  }
  return o;
}

template <typename S, bool PROJ = true>  // PROJ = false: TT_HESS_PSDPROJ compiled out (K4's default instantiation)
__device__ __forceinline__ Coefs<S> pair_coefs(S tc0, S tc1, const S (&g0)[18], const S (&g1)[18], int hess_mode) {
  Coefs<S> c;
  c.cg0 = S(2) * tc0 * (tc1 * tc1);
  c.cg1 = S(2) * tc1 * (tc0 * tc0);
  c.c00 = S(2) * (tc1 * tc1);
  c.c11 = S(2) * (tc0 * tc0);
  S keep = S(1);
  if (hess_mode == 1) {
    S g01 = S(0);
#pragma unroll
    for (int i = 0; i < 18; ++i) g01 = fma(g0[i], g1[i], g01);
    keep = (tc0 * tc1 * g01 >= S(0)) ? S(1) : S(0);  // sign of L47's 8 tc0 tc1 (g0.g1)
  } else if (hess_mode == 2) {
    keep = S(0);
  }
  c.c01 = S(4) * tc0 * tc1 * keep;
  if (PROJ && hess_mode == 3) {
    S p = S(0), q = S(0), r = S(0);
#pragma unroll
    for (int i = 0; i < 18; ++i) {
      p = fma(g0[i], g0[i], p);
      q = fma(g0[i], g1[i], q);
      r = fma(g1[i], g1[i], r);
    }
    // the 2x2 algebra (a Cholesky factor with a cancelling pivot) always in fp64: six scalars
    const Sym2 m = psd_project_2x2((double)p, (double)q, (double)r, (double)c.c00, (double)c.c01, (double)c.c11);
    c.c00 = (S)m.m00;
    c.c11 = (S)m.m11;
    c.c01 = (S)m.m01;
  }
  return c;
}

}  // namespace ttg
