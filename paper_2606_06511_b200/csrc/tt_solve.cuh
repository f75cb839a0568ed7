// tt_solve.cuh -- the consumer of the assembly ("GPU-based inexact
// Newton optimization route"): BSR(3x3) product, block-Jacobi preconditioner, and the vector kernels of
// preconditioned conjugate gradients for (H + shift I) x = b.  The paper gives no detail, so the
// operations are their textbook definitions (Hestenes-Stiefel recurrences; Saad, Alg. 9.1), done the GPU's
// way: 3x3 inverses by cofactors, dot products as fixed-order trees (deterministic, no floating-point
// atomics), all scalars of the recurrence (alpha, beta, r.z, |r|^2) kept in DEVICE memory so that an
// iteration needs no host round trip.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace tts {

constexpr int VEC_THREADS = 256;

// Scalars of one solve, in device memory.
struct PcgScalars {
  double rz;        // r_k . z_k
  double pq;        // p_k . A p_k
  double alpha, beta;
  double rr;        // |r_k|^2
  double bb;        // |b|^2
  double stop2;     // rtol^2 |b|^2
  int iters;        // steps taken so far
  int done;         // 1: |r_k| <= rtol |b| reached -- later kernels leave x, r, p untouched
};

// ---- y = (A + shift I) x, A in BSR with 3x3 row-major blocks -----------------------------------------
// One warp per block row; the lanes stride over the row's VALUES (9 per block), so the reads of `vals`
// -- 9w of the (9w + 4) bytes a block costs -- are perfectly coalesced whatever the row length.  Value i
// of the row belongs to block i / 9, element (r, c) = ((i % 9) / 3, i % 3), and adds vals[i] * x[3 col + c]
// to component r.  Accumulation in fp64, fixed order: deterministic.
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_bsr_spmv(const int* __restrict__ rowptr, const int* __restrict__ colind, const T* __restrict__ vals,
           const T* __restrict__ x, T* __restrict__ y, int64_t n_rows, double shift) {
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int64_t row = ((int64_t)blockIdx.x * VEC_THREADS + threadIdx.x) >> 5;
  if (row >= n_rows) return;
  const int64_t b0 = __ldg(rowptr + row), b1 = __ldg(rowptr + row + 1);
  // Lanes 0..26 walk the row THREE BLOCKS at a time: lane l always holds element (r, c) = ((l % 9) / 3, l % 3) of block
  // 3 k + l / 9, so nothing about a value's place has to be computed inside the loop (a 32-wide stride needs a division by
  // 9 and three predicated adds per value: with 64-bit indices that made 87 instructions per 32 values and the kernel was
  // bound by instruction issue at 34 % of the HBM roofline -- ncu, profiles/r2_step_breakdown.md).  Reads of `vals` stay
  // contiguous (27 consecutive values per trip) and are streamed (ld.global.cs): what is read once should not push x out
  // of the L2.  Lanes 27..31 idle.
  const int nb = (int)(b1 - b0);
  const int bo = lane / 9, e = lane - 9 * bo, c = e % 3;
  const T* __restrict__ vp = vals + 9 * b0 + lane;
  const int* __restrict__ cp = colind + b0 + bo;
  double acc = 0.0;
  if (lane < 27) {
#pragma unroll 2
    for (int k = bo; k < nb; k += 3) {
      acc = fma((double)__ldcs(vp), (double)__ldg(x + 3 * (int64_t)__ldg(cp) + c), acc);
      vp += 27;
      cp += 3;
    }
  }
  // lane l < 9 collects element l of the three block slots (lanes l, l + 9, l + 18), then lanes 0, 3, 6 the three columns of
  // rows 0, 1, 2: four shuffles in a fixed order (deterministic)
  const double t1 = __shfl_down_sync(FULL, acc, 9), t2 = __shfl_down_sync(FULL, acc, 18);
  const double s9 = acc + t1 + t2;
  const double u1 = __shfl_down_sync(FULL, s9, 1), u2 = __shfl_down_sync(FULL, s9, 2);
  const double tot = s9 + u1 + u2;
  if (lane < 9 && e == 3 * (lane / 3)) {
    const int rr = lane / 3;
    y[3 * row + rr] = (T)(tot + shift * (double)__ldg(x + 3 * row + rr));
  }
}

// ---- block-Jacobi: minv[v] = (A_vv + shift I)^-1 by cofactors (a row without a stored diagonal block: I / shift)
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_block_jacobi(const int* __restrict__ rowptr, const int* __restrict__ colind, const T* __restrict__ vals,
               int64_t n_rows, double shift, T* __restrict__ minv) {
  const int64_t v = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  if (v >= n_rows) return;
  double a[9] = {shift, 0, 0, 0, shift, 0, 0, 0, shift};
  int lo = __ldg(rowptr + v), hi = __ldg(rowptr + v + 1);
  while (lo < hi) {  // columns ascend inside a row: binary search for column v
    const int mid = (lo + hi) >> 1;
    const int c = __ldg(colind + mid);
    if (c < (int)v) lo = mid + 1;
    else hi = mid;
  }
  if (lo < __ldg(rowptr + v + 1) && __ldg(colind + lo) == (int)v) {
#pragma unroll
    for (int k = 0; k < 9; ++k) a[k] += (double)__ldg(vals + 9 * (int64_t)lo + k);
  }
  // 2x2 minors as Kahan's difference of products (error <= 1.5 ulp each: with a large low-rank block plus a
  // small shift the plain a*d - b*c loses every digit the shift contributes), determinant along the first row
  auto dop = [](double p, double q, double r, double t) {  // p*q - r*t
    const double w = r * t;
    const double e = fma(-r, t, w);
    const double f = fma(p, q, -w);
    return f + e;
  };
  const double c00 = dop(a[4], a[8], a[5], a[7]), c01 = dop(a[5], a[6], a[3], a[8]), c02 = dop(a[3], a[7], a[4], a[6]);
  const double det = fma(a[0], c00, fma(a[1], c01, a[2] * c02));
  const double id = 1.0 / det;
  T* o = minv + 9 * v;
  o[0] = (T)(c00 * id);
  o[1] = (T)(dop(a[2], a[7], a[1], a[8]) * id);
  o[2] = (T)(dop(a[1], a[5], a[2], a[4]) * id);
  o[3] = (T)(c01 * id);
  o[4] = (T)(dop(a[0], a[8], a[2], a[6]) * id);
  o[5] = (T)(dop(a[2], a[3], a[0], a[5]) * id);
  o[6] = (T)(c02 * id);
  o[7] = (T)(dop(a[1], a[6], a[0], a[7]) * id);
  o[8] = (T)(dop(a[0], a[4], a[1], a[3]) * id);
}

// ---- fixed-order reductions -------------------------------------------------------------------------
// CTA partial sums of up to two values per thread (shuffle tree, then warp 0): part[k][blockIdx.x].
__device__ __forceinline__ void cta_sum2(double v0, double v1, double* __restrict__ p0, double* __restrict__ p1) {
  __shared__ double s[2][VEC_THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v0 += __shfl_down_sync(0xffffffffu, v0, o);
    v1 += __shfl_down_sync(0xffffffffu, v1, o);
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) {
    s[0][w] = v0;
    s[1][w] = v1;
  }
  __syncthreads();
  if (w == 0) {
    v0 = (l < VEC_THREADS / 32) ? s[0][l] : 0.0;
    v1 = (l < VEC_THREADS / 32) ? s[1][l] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      v0 += __shfl_down_sync(0xffffffffu, v0, o);
      v1 += __shfl_down_sync(0xffffffffu, v1, o);
    }
    if (l == 0) {
      p0[blockIdx.x] = v0;
      if (p1) p1[blockIdx.x] = v1;
    }
  }
}
// one CTA: sum of n partials in a fixed order (strided lanes, then the same tree)
__device__ __forceinline__ double final_sum(const double* __restrict__ part, int64_t n, double* smem /*[32]*/) {
  double v = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) v += part[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) smem[w] = v;
  __syncthreads();
  double r = 0.0;
  if (w == 0) {
    r = smem[l];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
  }
  return r;  // valid in thread 0
}

template <typename T>
__device__ __forceinline__ void apply_minv(const T* __restrict__ minv, int64_t v, double r0, double r1, double r2,
                                           double& z0, double& z1, double& z2) {
  if (minv) {
    const T* m = minv + 9 * v;
    z0 = (double)m[0] * r0 + (double)m[1] * r1 + (double)m[2] * r2;
    z1 = (double)m[3] * r0 + (double)m[4] * r1 + (double)m[5] * r2;
    z2 = (double)m[6] * r0 + (double)m[7] * r1 + (double)m[8] * r2;
  } else {
    z0 = r0; z1 = r1; z2 = r2;
  }
}

// x = 0, r = b, z = M r, p = z; partials of r.z and b.b.  One thread per vertex.
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_pcg_init(const T* __restrict__ b, const T* __restrict__ minv, int64_t nV, T* __restrict__ x, T* __restrict__ r,
           T* __restrict__ p, double* __restrict__ part_rz, double* __restrict__ part_rr) {
  const int64_t v = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  double rz = 0.0, rr = 0.0;
  if (v < nV) {
    const double r0 = (double)b[3 * v], r1 = (double)b[3 * v + 1], r2 = (double)b[3 * v + 2];
    double z0, z1, z2;
    apply_minv(minv, v, r0, r1, r2, z0, z1, z2);
    x[3 * v] = (T)0; x[3 * v + 1] = (T)0; x[3 * v + 2] = (T)0;
    r[3 * v] = (T)r0; r[3 * v + 1] = (T)r1; r[3 * v + 2] = (T)r2;
    p[3 * v] = (T)z0; p[3 * v + 1] = (T)z1; p[3 * v + 2] = (T)z2;
    rz = r0 * z0 + r1 * z1 + r2 * z2;
    rr = r0 * r0 + r1 * r1 + r2 * r2;
  }
  cta_sum2(rz, rr, part_rz, part_rr);
}
__global__ void __launch_bounds__(1024) k_pcg_init_final(const double* __restrict__ part_rz, const double* __restrict__ part_rr,
                                                         int64_t n, double rtol, PcgScalars* __restrict__ sc,
                                                         double* __restrict__ hist) {
  __shared__ double s[32];
  const double rz = final_sum(part_rz, n, s);
  const double rr = final_sum(part_rr, n, s);
  if (threadIdx.x == 0) {
    sc->rz = rz;
    sc->rr = rr;
    sc->bb = rr;
    sc->stop2 = rtol * rtol * rr;
    sc->pq = 0.0;
    sc->alpha = 0.0;
    sc->beta = 0.0;
    sc->iters = 0;
    sc->done = (rr <= rtol * rtol * rr) ? 1 : 0;   // b = 0 (or rtol >= 1): x = 0 is the answer
    hist[0] = sqrt(rr);
  }
}

// q += shift p (matrix-free back end: the product came without the shift); partial of p.q
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_pcg_pq(const T* __restrict__ p, T* __restrict__ q, int64_t n, double shift, int add_shift, double* __restrict__ part) {
  const int64_t i = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  double v = 0.0;
  if (i < n) {
    const double pi = (double)p[i];
    double qi = (double)q[i];
    if (add_shift) {
      qi += shift * pi;
      q[i] = (T)qi;
    }
    v = pi * qi;
  }
  cta_sum2(v, 0.0, part, nullptr);
}
__global__ void __launch_bounds__(1024) k_pcg_alpha(const double* __restrict__ part, int64_t n, PcgScalars* __restrict__ sc) {
  __shared__ double s[32];
  const double pq = final_sum(part, n, s);
  if (threadIdx.x == 0) {
    sc->pq = pq;
    sc->alpha = sc->done ? 0.0 : sc->rz / pq;
  }
}

// x += alpha p, r -= alpha q, z = M r (stored in q's place: q is dead); partials of r.z and r.r
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_pcg_update(const T* __restrict__ p, T* __restrict__ q, const T* __restrict__ minv, int64_t nV, T* __restrict__ x,
             T* __restrict__ r, const PcgScalars* __restrict__ sc, double* __restrict__ part_rz, double* __restrict__ part_rr) {
  const int64_t v = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  const bool done = sc->done != 0;
  const double alpha = sc->alpha;
  double rz = 0.0, rr = 0.0;
  if (v < nV && !done) {
    double rn[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int64_t i = 3 * v + c;
      x[i] = (T)((double)x[i] + alpha * (double)p[i]);
      rn[c] = (double)r[i] - alpha * (double)q[i];
      r[i] = (T)rn[c];
      rn[c] = (double)r[i];   // the stored (rounded, for T = float) residual is the one recurred
    }
    double z0, z1, z2;
    apply_minv(minv, v, rn[0], rn[1], rn[2], z0, z1, z2);
    q[3 * v] = (T)z0; q[3 * v + 1] = (T)z1; q[3 * v + 2] = (T)z2;
    rz = rn[0] * z0 + rn[1] * z1 + rn[2] * z2;
    rr = rn[0] * rn[0] + rn[1] * rn[1] + rn[2] * rn[2];
  }
  cta_sum2(rz, rr, part_rz, part_rr);
}
__global__ void __launch_bounds__(1024) k_pcg_beta(const double* __restrict__ part_rz, const double* __restrict__ part_rr,
                                                   int64_t n, PcgScalars* __restrict__ sc, double* __restrict__ hist) {
  __shared__ double s[32];
  const double rz = final_sum(part_rz, n, s);
  const double rr = final_sum(part_rr, n, s);
  if (threadIdx.x == 0 && !sc->done) {
    sc->beta = rz / sc->rz;
    sc->rz = rz;
    sc->rr = rr;
    sc->iters += 1;
    hist[sc->iters] = sqrt(rr);
    if (rr <= sc->stop2) sc->done = 1;
  }
}
// p = z + beta p (z sits in q)
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_pcg_dir(const T* __restrict__ z, T* __restrict__ p, int64_t n, const PcgScalars* __restrict__ sc) {
  const int64_t i = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  if (i < n && !sc->done) p[i] = (T)((double)z[i] + sc->beta * (double)p[i]);
}

// ---- the Newton step around the solve (tt_newton_step; reading A16) ----------------------------------
// partials of g.d and g.g (fixed order), then both sums in one CTA
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_dot2(const T* __restrict__ g, const T* __restrict__ d, int64_t n, double* __restrict__ part_gd, double* __restrict__ part_gg) {
  const int64_t i = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  double a = 0.0, b = 0.0;
  if (i < n) {
    const double gi = (double)g[i];
    a = gi * (double)d[i];
    b = gi * gi;
  }
  cta_sum2(a, b, part_gd, part_gg);
}
__global__ void __launch_bounds__(1024) k_dot2_final(const double* __restrict__ part_gd, const double* __restrict__ part_gg,
                                                     int64_t n, double* __restrict__ out /*[2]*/) {
  __shared__ double s[32];
  const double gd = final_sum(part_gd, n, s);
  const double gg = final_sum(part_gg, n, s);
  if (threadIdx.x == 0) {
    out[0] = gd;
    out[1] = gg;
  }
}
// x_try = x - alpha d
template <typename T>
__global__ void __launch_bounds__(VEC_THREADS)
k_step(const T* __restrict__ x, const T* __restrict__ d, double alpha, int64_t n, T* __restrict__ x_try) {
  const int64_t i = (int64_t)blockIdx.x * VEC_THREADS + threadIdx.x;
  if (i < n) x_try[i] = (T)((double)x[i] - alpha * (double)d[i]);
}

}  // namespace tts
