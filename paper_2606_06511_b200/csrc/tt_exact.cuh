// tt_exact.cuh -- TT_HESS_EXACT (hess_mode 4): the exact Hessian of T = (tc0 tc1)^2 (second half).
//
// PAPER.md L26 ("ignoring the asymmetric part of the exact Hessian") / Eq. 4 (L28-33) keep only the outer products
// of g0 = d tc0 and g1 = d tc1; the exact Hessian adds the second derivatives of the end-points,
//     H_exact = H_EQ4 + 2 tc0 tc1^2 d2 tc0 + 2 tc1 tc0^2 d2 tc1.
// The GPU's own route (the oracle pushes second-order duals with 171 second partials through App. A instead): the
// analytic gradient code of tt_geom.cuh is a template on its scalar, so it is run on a number that carries ONE
// directional derivative (forward mode over the analytic gradient):
//     d/d eps  g_r(x + eps v) = (d2 tc_r) v,
// i.e. one evaluation gives a Hessian-vector product (H.p: one pass with v = p) and nine evaluations with v = the
// unit vectors of a triangle's own 9 DOF give the 9 x 18 rows an assembly lane owns.
//
// One term has to come back first.  tt_geom.cuh uses d(D.(P - Q)) = D^T (dP - dQ): the other half of the product
// rule, (dD)^T (P - Q), vanishes because P - Q is parallel to the unit vector D and D . dD = 0.  That is an identity
// in x -- so it may be differentiated again -- EXCEPT on App. A's "vertex exactly on the plane" branch (L106-115),
// where the end-point is pinned to the vertex and leaves the line as soon as x moves.  grad_line_term below is that
// half in closed form,
//     f(x) = D(x) . c,  D = (n_a x n_b) / |n_a x n_b|:   grad f = (grad (n_a x n_b))^T u,  u = (c - D (D . c)) / |n_a x n_b|,
// identically zero (value and derivative) for regular pairs and exactly the missing part for the others.
#pragma once
#include "tt_geom.cuh"
#include "tt_kernels.cuh"

namespace ttx {

struct Dual {
  double v, d;
  __device__ __forceinline__ Dual() {}
  __device__ __forceinline__ Dual(double v_) : v(v_), d(0.0) {}
  __device__ __forceinline__ Dual(double v_, double d_) : v(v_), d(d_) {}
};
__device__ __forceinline__ Dual operator+(Dual a, Dual b) { return Dual(a.v + b.v, a.d + b.d); }
__device__ __forceinline__ Dual operator-(Dual a, Dual b) { return Dual(a.v - b.v, a.d - b.d); }
__device__ __forceinline__ Dual operator-(Dual a) { return Dual(-a.v, -a.d); }
__device__ __forceinline__ Dual operator*(Dual a, Dual b) { return Dual(a.v * b.v, fma(a.v, b.d, a.d * b.v)); }
__device__ __forceinline__ Dual fma(Dual a, Dual b, Dual c) {
  return Dual(::fma(a.v, b.v, c.v), ::fma(a.v, b.d, ::fma(a.d, b.v, c.d)));
}
__device__ __forceinline__ Dual operator/(Dual a, Dual b) {  // only 1 / x is used
  const double r = 1.0 / b.v;
  const double q = a.v * r;
  return Dual(q, (a.d - q * b.d) * r);
}
__device__ __forceinline__ Dual inv_sqrt(Dual a) {
  const double r = rsqrt(a.v);
  return Dual(r, -0.5 * r * r * r * a.d);
}
// an end-point that is a vertex: tau is the constant 1 (tt_geom.cuh)
__device__ __forceinline__ Dual vertex_tau(Dual tau, Dual zmask) { return zmask.v == 0.0 ? Dual(1.0) : tau; }

using DV = ttg::v3<Dual>;
__device__ __forceinline__ DV operator-(DV a) { return ttg::mk<Dual>(-a.x, -a.y, -a.z); }

// gradient of f(x) = D(x) . c (c held fixed) over [a_k, a_p, a_q, b_k, b_p, b_q], times s, ADDED to g
__device__ __forceinline__ void grad_line_term(Dual s, const DV c, const ttg::PairAux<Dual>& A, Dual (&g)[18]) {
  const Dual dc = ttg::dot(A.Dh, c);
  const DV u = A.rinv * (c - dc * A.Dh);
  const DV wa = ttg::cross(A.nb, u), wb = ttg::cross(u, A.na);
  const DV gap = s * ttg::cross(A.eaq, wa), gaq = s * ttg::cross(wa, A.eap);
  const DV gbp = s * ttg::cross(A.ebq, wb), gbq = s * ttg::cross(wb, A.ebp);
  auto add = [](Dual (&t)[18], int o, const DV v) { t[o] = t[o] + v.x; t[o + 1] = t[o + 1] + v.y; t[o + 2] = t[o + 2] + v.z; };
  add(g, 0, -(gap + gaq));  add(g, 3, gap);   add(g, 6, gaq);
  add(g, 9, -(gbp + gbq));  add(g, 12, gbp);  add(g, 15, gbq);
}

// Values and one directional derivative of everything a pair contributes:
//   x  [a_k, a_p, a_q, b_k, b_p, b_q] (recorded order, raw positions),  v  the direction in the same order
//   tc[2], g0[18], g1[18]  values;   h0 = (d2 tc0) v,  h1 = (d2 tc1) v
struct PairDir {
  double tc0, tc1, dtc0, dtc1;  // dtc_r = g_r . v
  double g0[18], g1[18], h0[18], h1[18];
};
// (inlined: the callers' loops are not unrolled, so there is one copy per kernel; assembly 47.7 -> 35.0 ms and H.p 4.7 ->
// 4.0 ms at 10 M pairs against the out-of-line call, measured.  Folding the gradient pass into the first row pass was also
// measured and is slower: 44 ms.)
__device__ __forceinline__ void pair_second_dir(const double (&x)[18], const double (&v)[18], unsigned za, unsigned zb,
                                             double sigma, PairDir& o) {
  // local frame: translate by -a_k (the direction of a_k is subtracted with it)
  auto pt = [&](int i) {
    return ttg::mk<Dual>(Dual(x[3 * i] - x[0], v[3 * i] - v[0]), Dual(x[3 * i + 1] - x[1], v[3 * i + 1] - v[1]),
                         Dual(x[3 * i + 2] - x[2], v[3 * i + 2] - v[2]));
  };
  const DV ak = ttg::mk<Dual>(Dual(0.0), Dual(0.0), Dual(0.0));
  Dual tc0, tc1, g0[18], g1[18];
  ttg::PairAux<Dual> A;
  ttg::pair_derivs_core<Dual>(ak, pt(1), pt(2), pt(3), pt(4), pt(5), Dual(sigma), za, zb, tc0, tc1, g0, g1, A);
  grad_line_term(Dual(sigma), A.c0, A, g0);
  grad_line_term(Dual(sigma), A.c1, A, g1);
  o.tc0 = tc0.v;  o.tc1 = tc1.v;  o.dtc0 = tc0.d;  o.dtc1 = tc1.d;
#pragma unroll
  for (int i = 0; i < 18; ++i) {
    o.g0[i] = g0[i].v;  o.h0[i] = g0[i].d;
    o.g1[i] = g1[i].v;  o.h1[i] = g1[i].d;
  }
}

}  // namespace ttx

// ---------------------------------------------------------------------------------------- kernels
// Both kernels take the work partition of K4 / K6 as it is (rounds, slots, parts, ranks, row bases): one warp per
// round -- ordinary rounds, parts of split triangles and long triangles alike -- lane = directed entry, entries in
// groups of 32.  They are a VARIANT, not the headline path: plain global stores instead of the row-run tile + TMA,
// per-lane results in local memory.  No floating-point atomics; every sum over the entries of a triangle runs in
// entry order.
namespace ttk {

constexpr int EX_WARPS = (RND_MAX_TRI > 12) ? 2 : 4;
constexpr int EX_NACC = 90;  // 9 own rows x 9 own columns (diagonal blocks) + 9 gradient values
struct ExactWarpSmem {
  double stage[32 * 9];                // per entry: the 9 own-column values of the current row (or the gradient)
  double acc[RND_MAX_TRI][EX_NACC];    // per slot sums
  long long rb[RND_MAX_TRI][3];
  int dr[RND_MAX_TRI][3];
  int first[RND_MAX_TRI + 1];
};

struct EntryCfg {
  bool side;
  unsigned za, zb;
  int po[3], pp[3];  // recorded position r -> index inside the own / partner triangle
  int oh, ph;        // offsets of the own / partner half in the canonical 18-vector
};
__device__ __forceinline__ EntryCfg entry_cfg(unsigned pay) {
  EntryCfg c;
  c.side = (pay & 1u) != 0u;
  const unsigned ca = (pay >> 1) & 63u, cb = (pay >> 7) & 63u;
  int pa[3], pb[3];
  pa[0] = (int)(ca & 3u); pa[1] = (int)((ca >> 2) & 3u); pa[2] = 3 - pa[0] - pa[1];
  pb[0] = (int)(cb & 3u); pb[1] = (int)((cb >> 2) & 3u); pb[2] = 3 - pb[0] - pb[1];
  c.za = ca >> 4;
  c.zb = cb >> 4;
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    c.po[r] = c.side ? pb[r] : pa[r];
    c.pp[r] = c.side ? pa[r] : pb[r];
  }
  c.oh = c.side ? 9 : 0;
  c.ph = 9 - c.oh;
  return c;
}
__device__ __forceinline__ void load_entry_ids(const int* __restrict__ everts, int64_t e, int (&ids)[6]) {
  const int2* iv = reinterpret_cast<const int2*>(everts + 6 * e);
  const int2 v0 = __ldg(iv), v1 = __ldg(iv + 1), v2 = __ldg(iv + 2);
  ids[0] = v0.x; ids[1] = v0.y; ids[2] = v1.x; ids[3] = v1.y; ids[4] = v2.x; ids[5] = v2.y;
}

// y = H_exact p, per-slot partials into tslot (then k_split_finish / k_gather3 as after K6).
//   y_loc = J^T M (J p_loc) + 2 tc0 tc1^2 (d2 tc0) p_loc + 2 tc1 tc0^2 (d2 tc1) p_loc,   M = Eq. 4's, all three parts
template <typename T>
__global__ void __launch_bounds__(RED_THREADS)
k_hess_vec_exact(const AsmParams<T> P) {
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t c = (int64_t)blockIdx.x * (RED_THREADS / 32) + warp;
  if (c >= P.n_chunks) return;
  const int4 d = __ldg(P.rdesc + c);
  const int e_lo = d.x, e_hi = d.x + d.y;
  const bool is_long = d.y > RND_MAX_ENT;
  unsigned heads = 1u;
  if (!is_long) {
    const int f = (lane < d.w) ? __ldg(P.tfirst + d.z + lane) - e_lo : 0;
    heads = __reduce_or_sync(FULL, (lane < d.w) ? (1u << f) : 0u);
  }
  const unsigned below = heads & (0xffffffffu >> (31 - lane));
  const int segf = 31 - __clz((int)below);
  double carry[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) carry[k] = 0.0;
  for (int base = e_lo; base < e_hi; base += 32) {
    const int nvalid = min(32, e_hi - base);
    double v[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) v[k] = 0.0;
    if (lane < nvalid) {
      const int64_t e = (int64_t)base + lane;
      int ids[6];
      load_entry_ids(P.everts, e, ids);
      double x[18], pv[18];
      load_pos18(P.pos, ids, x);
      load_pos18(P.pvec, ids, pv);
      const EntryCfg cf = entry_cfg((unsigned)__ldg(P.dvals + e));
      ttx::PairDir o;
      ttx::pair_second_dir(x, pv, cf.za, cf.zb, P.sigma, o);
      const double c00 = 2.0 * o.tc1 * o.tc1, c11 = 2.0 * o.tc0 * o.tc0, c01 = 4.0 * o.tc0 * o.tc1;
      const double u0 = c00 * o.dtc0 + c01 * o.dtc1, u1 = c01 * o.dtc0 + c11 * o.dtc1;  // M (J p_loc)
      const double w0 = 2.0 * o.tc0 * o.tc1 * o.tc1, w1 = 2.0 * o.tc1 * o.tc0 * o.tc0;
      double yr[9];
#pragma unroll
      for (int i = 0; i < 9; ++i) {
        const int q = cf.oh + i;
        yr[i] = u0 * o.g0[q] + u1 * o.g1[q] + w0 * o.h0[q] + w1 * o.h1[q];
      }
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int cc = 0; cc < 3; ++cc)
          v[3 * i + cc] = (cf.po[0] == i) ? yr[cc] : ((cf.po[1] == i) ? yr[3 + cc] : yr[6 + cc]);
    }
#pragma unroll
    for (int o2 = 1; o2 < 32; o2 <<= 1) {
      const bool take = (lane - o2) >= segf;
#pragma unroll
      for (int k = 0; k < 9; ++k) {
        const double up = __shfl_up_sync(FULL, v[k], o2);
        if (take) v[k] += up;
      }
    }
    if (!is_long) {
      const bool last = (lane < nvalid) && (lane == nvalid - 1 || (((heads >> 1) >> lane) & 1u));
      if (last) {
        const int64_t ti = (int64_t)d.z + __popc(below) - 1;
#pragma unroll
        for (int k = 0; k < 9; ++k) P.tslot[9 * ti + k] = (T)v[k];
      }
    } else {
#pragma unroll
      for (int k = 0; k < 9; ++k) carry[k] += __shfl_sync(FULL, v[k], nvalid - 1);
    }
  }
  if (is_long && lane == 0) {
#pragma unroll
    for (int k = 0; k < 9; ++k) P.tslot[9 * (int64_t)d.z + k] = (T)carry[k];
  }
}

// Energy, gradient partials and ALL BSR values of the exact Hessian.  For each of a lane's 9 own DOF (row 3m + i of
// the triangle's three block rows) one directional evaluation gives the whole 18-wide row
//     R = A0 g0 + A1 g1 + w0 (d2 tc0) e_row + w1 (d2 tc1) e_row,   A = M [g0_row, g1_row],
// whose partner half goes straight to the three blocks the entry owns in row m (ranks as in K4) and whose own half
// is summed over the triangle's entries into the diagonal blocks.
template <typename T>
__global__ void __launch_bounds__(32 * EX_WARPS)
k_assemble_exact(const AsmParams<T> P) {
  __shared__ ExactWarpSmem s_all[EX_WARPS];
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  ExactWarpSmem& S = s_all[warp];
  const int64_t c = (int64_t)blockIdx.x * EX_WARPS + warp;
  if (c >= P.n_chunks) return;
  const int4 d = __ldg(P.rdesc + c);
  const int e_lo = d.x, e_hi = d.x + d.y, s_lo = d.z, nsl = d.w;
  const bool is_long = d.y > RND_MAX_ENT;  // one slot, several groups
  if (lane < nsl) {
    const int64_t sl = (int64_t)s_lo + lane;
    S.first[lane] = __ldg(P.tfirst + sl) - e_lo;
    if (lane == nsl - 1) S.first[nsl] = d.y;
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      S.rb[lane][m] = (long long)__ldg(P.rowbase + 3 * sl + m);
      S.dr[lane][m] = __ldg(P.drank + 3 * sl + m);
    }
  }
  for (int i = lane; i < nsl * EX_NACC; i += 32) S.acc[i / EX_NACC][i % EX_NACC] = 0.0;
  __syncwarp();
  unsigned heads = 1u;
  if (!is_long) heads = __reduce_or_sync(FULL, (lane < nsl) ? (1u << S.first[lane]) : 0u);
  const int my_ti = __popc(heads & (0xffffffffu >> (31 - lane))) - 1;
  double e_acc = 0.0;
  for (int base = e_lo; base < e_hi; base += 32) {
    const int nvalid = min(32, e_hi - base);
    const bool valid = lane < nvalid;
    double x[18];
    int er[3] = {0, 0, 0};
    EntryCfg cf = entry_cfg(0u);
    T* rowp[3] = {nullptr, nullptr, nullptr};
    if (valid) {
      const int64_t e = (int64_t)base + lane;
      int ids[6];
      load_entry_ids(P.everts, e, ids);
      load_pos18(P.pos, ids, x);
      cf = entry_cfg((unsigned)__ldg(P.dvals + e));
      int rk[3];
#pragma unroll
      for (int n = 0; n < 3; ++n) rk[n] = __ldg(P.erank + 3 * e + n);
#pragma unroll
      for (int r = 0; r < 3; ++r) er[r] = (cf.pp[r] == 0) ? rk[0] : ((cf.pp[r] == 1) ? rk[1] : rk[2]);  // recorded order
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const long long rb = S.rb[my_ti][m];
        rowp[m] = (rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1));
      }
    }
#pragma unroll 1
    for (int j = 0; j < 10; ++j) {  // 9 own rows, then the gradient
      if (valid) {
        const int m = (j < 9) ? j / 3 : 0, i = (j < 9) ? j % 3 : 0;
        const int r = (cf.po[0] == m) ? 0 : ((cf.po[1] == m) ? 1 : 2);  // recorded position of own vertex m
        const int jc = cf.oh + 3 * r + i;
        double dir[18];
#pragma unroll
        for (int q = 0; q < 18; ++q) dir[q] = (j < 9 && q == jc) ? 1.0 : 0.0;
        ttx::PairDir o;
        ttx::pair_second_dir(x, dir, cf.za, cf.zb, P.sigma, o);
        double R[18];
        if (j < 9) {
          const double c00 = 2.0 * o.tc1 * o.tc1, c11 = 2.0 * o.tc0 * o.tc0, c01 = 4.0 * o.tc0 * o.tc1;
          const double A0 = c00 * o.g0[jc] + c01 * o.g1[jc], A1 = c01 * o.g0[jc] + c11 * o.g1[jc];
          const double w0 = 2.0 * o.tc0 * o.tc1 * o.tc1, w1 = 2.0 * o.tc1 * o.tc0 * o.tc0;
#pragma unroll
          for (int q = 0; q < 18; ++q) R[q] = A0 * o.g0[q] + A1 * o.g1[q] + w0 * o.h0[q] + w1 * o.h1[q];
          // partner half: the three blocks this entry owns in row m
#pragma unroll
          for (int rr = 0; rr < 3; ++rr) {
            T* dst = rowp[m] + 9 * (int64_t)er[rr] + 3 * i;
#pragma unroll
            for (int jj = 0; jj < 3; ++jj) dst[jj] = (T)R[cf.ph + 3 * rr + jj];
          }
        } else {
          const double cg0 = 2.0 * o.tc0 * o.tc1 * o.tc1, cg1 = 2.0 * o.tc1 * o.tc0 * o.tc0;  // Eq. 3
#pragma unroll
          for (int q = 0; q < 18; ++q) R[q] = cg0 * o.g0[q] + cg1 * o.g1[q];
          const double tt = o.tc0 * o.tc1;
          if (!cf.side) e_acc += tt * tt;  // Eq. 2, once per pair
        }
        // own half in the triangle's own vertex order
#pragma unroll
        for (int rr = 0; rr < 3; ++rr)
#pragma unroll
          for (int jj = 0; jj < 3; ++jj) S.stage[lane * 9 + 3 * cf.po[rr] + jj] = R[cf.oh + 3 * rr + jj];
      }
      __syncwarp();
      for (int it = lane; it < 9 * nsl; it += 32) {
        const int tt = it / 9, c9 = it - 9 * tt;
        const int f = is_long ? 0 : S.first[tt], l = is_long ? nvalid : S.first[tt + 1];
        double a = 0.0;
        for (int en = f; en < l; ++en) a += S.stage[en * 9 + c9];
        S.acc[tt][9 * j + c9] += a;
      }
      __syncwarp();
    }
  }
  // ---- per-slot results ----
  for (int it = lane; it < nsl * EX_NACC; it += 32) {
    const int tt = it / EX_NACC, k = it - EX_NACC * tt;
    const double a = S.acc[tt][k];
    if (k >= 81) {
      P.tslot[9 * ((int64_t)s_lo + tt) + (k - 81)] = (T)a;
      continue;
    }
    const int jrow = k / 9, c9 = k - 9 * jrow;
    const int m = jrow / 3, i = jrow - 3 * m, n = c9 / 3, jj = c9 - 3 * n;
    if (S.dr[tt][0] < 0) {  // a part: its diagonal partial sums go to k_split_finish (packed upper triangle)
      if (jrow <= c9) {
        const int uidx = jrow * 9 - (jrow * (jrow - 1)) / 2 + (c9 - jrow);
        P.dpart[(int64_t)NDIAG * (-1 - S.dr[tt][0]) + uidx] = a;
      }
    } else {
      const long long rb = S.rb[tt][m];
      T* rowp = (rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1));
      rowp[9 * (int64_t)S.dr[tt][n] + 3 * i + jj] = (T)a;
    }
  }
#pragma unroll
  for (int o2 = 16; o2 > 0; o2 >>= 1) e_acc += __shfl_down_sync(FULL, e_acc, o2);
  if (lane == 0) P.chunk_energy[c] = e_acc;
}

}  // namespace ttk
