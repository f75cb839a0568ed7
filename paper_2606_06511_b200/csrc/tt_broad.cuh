// tt_broad.cuh -- broad phase ("spatial hashing structure
// [Pabst et al. 2010] to eliminate redundant computations", no detail given).  The operation is
// defined by its result: all pairs i < j of triangles that share no vertex index and whose
// axis-aligned bounding boxes, each grown by `inflate` on every side, overlap (closed intervals),
// in lexicographic order -- the `pairs` array the hot path consumes.
//
// Uniform grid (cell size: k_bp_grid; a box touches at most 5 cells per axis):
//   k_bp_aabb      boxes in fp64 + per-CTA partial bounds          (HBM: 3 vertices in, 48 B out)
//   k_bp_grid      origin, cell size, grid dimensions (one CTA, fixed order)
//   k_bp_cells     <COUNT / EMIT> (cell key, triangle) records, <= 125 per triangle (typically 2-4)
//   CUB radix sort of the records by (cell, quantised lo.x): sweep-and-prune inside a cell
//   k_bp_pairs     <COUNT / EMIT> one thread per record walks the later records of its cell; a pair is
//                  reported only in the cell that owns the point max(lo_i, lo_j), which lies in both
//                  boxes when they overlap, so every pair is reported exactly once
//   CUB radix sort of the pair keys i * nT + j, k_bp_unpack -> int32 [P,2]
// No floating-point result leaves this file except through comparisons, and the oracle evaluates
// the same comparisons on the same fp64 box bounds: the candidate set is bit-exact.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ttb {

struct Grid {
  double org[3];
  double inv_cell;
  int dims[3];
  int pad;
};

constexpr int BP_THREADS = 256;

template <typename T>
__global__ void __launch_bounds__(BP_THREADS)
k_bp_aabb(const T* __restrict__ pos, const int* __restrict__ tris, int64_t nT, double inflate,
          double* __restrict__ box /*[nT][6] lo, hi*/, double* __restrict__ part /*[grid][8] min lo, max hi, max extent, sum of extents*/) {
  __shared__ double s[BP_THREADS / 32][8];
  const int64_t t = (int64_t)blockIdx.x * BP_THREADS + threadIdx.x;
  double v[8] = {1e300, 1e300, 1e300, -1e300, -1e300, -1e300, 0.0, 0.0};
  if (t < nT) {
    double lo[3], hi[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double a = (double)pos[3 * (int64_t)tris[3 * t] + c], b = (double)pos[3 * (int64_t)tris[3 * t + 1] + c],
                   d = (double)pos[3 * (int64_t)tris[3 * t + 2] + c];
      lo[c] = fmin(a, fmin(b, d)) - inflate;
      hi[c] = fmax(a, fmax(b, d)) + inflate;
      box[6 * t + c] = lo[c];
      box[6 * t + 3 + c] = hi[c];
      v[c] = lo[c];
      v[3 + c] = hi[c];
      v[6] = fmax(v[6], hi[c] - lo[c]);
    }
    v[7] = v[6];  // this triangle's largest extent
  }
#pragma unroll
  for (int k = 0; k < 8; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double u = __shfl_xor_sync(0xffffffffu, v[k], o);
      v[k] = (k < 3) ? fmin(v[k], u) : ((k < 7) ? fmax(v[k], u) : v[k] + u);
    }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0)
#pragma unroll
    for (int k = 0; k < 8; ++k) s[w][k] = v[k];
  __syncthreads();
  if (threadIdx.x < 8) {
    const int k = threadIdx.x;
    double r = s[0][k];
    for (int i = 1; i < BP_THREADS / 32; ++i) r = (k < 3) ? fmin(r, s[i][k]) : ((k < 7) ? fmax(r, s[i][k]) : r + s[i][k]);
    part[8 * (int64_t)blockIdx.x + k] = r;
  }
}

// Cell size: never larger than the largest box (then a box touches <= 2 cells per axis), but when a
// few boxes are much larger than the rest, 2 x the mean extent, floored at a quarter of the largest
// (a box then touches <= 5 cells per axis, <= 125 in all): the candidate list does not depend on it.
constexpr int BP_MAX_DIM = 32768;  // cells per axis: the cell key stays below 2^45
__global__ void __launch_bounds__(BP_THREADS)
k_bp_grid(const double* __restrict__ part, int64_t n_part, int64_t nT, Grid* __restrict__ g) {
  __shared__ double s[BP_THREADS][8];
  double v[8] = {1e300, 1e300, 1e300, -1e300, -1e300, -1e300, 0.0, 0.0};
  for (int64_t i = threadIdx.x; i < n_part; i += BP_THREADS)
#pragma unroll
    for (int k = 0; k < 8; ++k)
      v[k] = (k < 3) ? fmin(v[k], part[8 * i + k]) : ((k < 7) ? fmax(v[k], part[8 * i + k]) : v[k] + part[8 * i + k]);
#pragma unroll
  for (int k = 0; k < 8; ++k) s[threadIdx.x][k] = v[k];
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < BP_THREADS; ++i)
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = (k < 3) ? fmin(v[k], s[i][k]) : ((k < 7) ? fmax(v[k], s[i][k]) : v[k] + s[i][k]);
    const double big = v[6] * 1.0001, mean = v[7] / (double)(nT > 0 ? nT : 1);
    double cell = fmin(big, fmax(2.0 * mean, 0.25 * big));
    // a sparse scene (domain >> boxes) must not overflow the cell coordinates: at most BP_MAX_DIM cells per
    // axis (a larger cell only registers a box in fewer cells; the candidate list does not depend on it)
    for (int c = 0; c < 3; ++c)
      if (n_part > 0 && v[3 + c] >= v[c]) cell = fmax(cell, (v[3 + c] - v[c]) / (double)(BP_MAX_DIM - 1));
    if (!(cell > 0.0) || !(cell < 1e300)) cell = 1.0;
    g->inv_cell = 1.0 / cell;
    for (int c = 0; c < 3; ++c) {
      g->org[c] = v[c];
      double d = (n_part > 0 && v[3 + c] >= v[c]) ? floor((v[3 + c] - v[c]) * g->inv_cell) + 1.0 : 1.0;
      d = fmin(fmax(d, 1.0), (double)BP_MAX_DIM);   // computed in double: never wraps an int
      g->dims[c] = (int)d;
    }
    g->pad = 0;
  }
}

__device__ __forceinline__ int cell_coord(double x, double org, double inv_cell, int dim) {
  const int c = (int)floor((x - org) * inv_cell);
  return min(max(c, 0), dim - 1);
}
__device__ __forceinline__ uint64_t cell_key(const Grid& g, int cx, int cy, int cz) {
  return ((uint64_t)cx * (uint64_t)g.dims[1] + (uint64_t)cy) * (uint64_t)g.dims[2] + (uint64_t)cz;
}

// Sweep-and-prune inside a cell: the records of a cell are sorted by the x of their box's lower bound,
// quantised to BP_QBITS bits of the cell width (monotone, so the pruning below is conservative):
// a walk stops at the first record whose quantised lo.x exceeds the walker's quantised hi.x.
constexpr int BP_QBITS = 16;
__device__ __forceinline__ unsigned quant_x(double x, const Grid& g, int cx) {
  const double f = (x - g.org[0]) * g.inv_cell - (double)cx;  // position inside cell cx, in cell widths
  const double q = floor(f * (double)(1u << BP_QBITS));
  return (unsigned)fmin(fmax(q, 0.0), (double)((1u << BP_QBITS) - 1u));
}

// COUNT: cnt[t] = cells box t touches (1..125).  EMIT: records at off[t],
// key = cell << BP_QBITS | quantised lo.x inside that cell.
template <bool EMIT>
__global__ void __launch_bounds__(BP_THREADS)
k_bp_cells(const double* __restrict__ box, int64_t nT, const Grid* __restrict__ gp, int* __restrict__ cnt,
           const int* __restrict__ off, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  const int64_t t = (int64_t)blockIdx.x * BP_THREADS + threadIdx.x;
  if (t >= nT) return;
  const Grid g = *gp;
  int lo[3], hi[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = cell_coord(box[6 * t + c], g.org[c], g.inv_cell, g.dims[c]);
    hi[c] = cell_coord(box[6 * t + 3 + c], g.org[c], g.inv_cell, g.dims[c]);
  }
  if (!EMIT) {
    cnt[t] = (hi[0] - lo[0] + 1) * (hi[1] - lo[1] + 1) * (hi[2] - lo[2] + 1);
    return;
  }
  int64_t o = off[t];
  for (int cx = lo[0]; cx <= hi[0]; ++cx)
    for (int cy = lo[1]; cy <= hi[1]; ++cy)
      for (int cz = lo[2]; cz <= hi[2]; ++cz) {
        keys[o] = (cell_key(g, cx, cy, cz) << BP_QBITS) | quant_x(box[6 * t], g, cx);
        vals[o] = (uint32_t)t;
        ++o;
      }
}

__device__ __forceinline__ bool bp_share_vertex(const int* __restrict__ tris, int64_t i, int64_t j) {
  const int a0 = tris[3 * i], a1 = tris[3 * i + 1], a2 = tris[3 * i + 2];
  const int b0 = tris[3 * j], b1 = tris[3 * j + 1], b2 = tris[3 * j + 2];
  return a0 == b0 || a0 == b1 || a0 == b2 || a1 == b0 || a1 == b1 || a1 == b2 || a2 == b0 || a2 == b1 || a2 == b2;
}

// COUNT: cnt[r] = pairs record r reports.  EMIT: pair keys i * nT + j at off[r].
template <bool EMIT>
__global__ void __launch_bounds__(BP_THREADS)
k_bp_pairs(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ vals, int64_t n_rec,
           const double* __restrict__ box, const int* __restrict__ tris, int64_t nT, const Grid* __restrict__ gp,
           int* __restrict__ cnt, const int64_t* __restrict__ off, uint64_t* __restrict__ pair_keys) {
  const int64_t r = (int64_t)blockIdx.x * BP_THREADS + threadIdx.x;
  if (r >= n_rec) return;
  const Grid g = *gp;
  const uint64_t key = keys[r] >> BP_QBITS;  // the cell
  const int64_t i = vals[r];
  double lo[3], hi[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = box[6 * i + c];
    hi[c] = box[6 * i + 3 + c];
  }
  // last quantised lo.x a partner can have: hi.x of this box inside this cell
  const int cx = (int)(key / ((uint64_t)g.dims[1] * (uint64_t)g.dims[2]));
  const uint64_t stop = (key << BP_QBITS) | quant_x(hi[0], g, cx);
  int n = 0;
  int64_t o = EMIT ? off[r] : 0;
  for (int64_t q = r + 1; q < n_rec && keys[q] <= stop; ++q) {
    const int64_t j = vals[q];
    double m[3];
    bool ov = true;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double lj = box[6 * j + c], hj = box[6 * j + 3 + c];
      ov = ov && (lo[c] <= hj) && (lj <= hi[c]);
      m[c] = fmax(lo[c], lj);
    }
    if (!ov) continue;
    // the cell that owns max(lo_i, lo_j) reports the pair (both boxes are registered there)
    const uint64_t owner = cell_key(g, cell_coord(m[0], g.org[0], g.inv_cell, g.dims[0]),
                                    cell_coord(m[1], g.org[1], g.inv_cell, g.dims[1]),
                                    cell_coord(m[2], g.org[2], g.inv_cell, g.dims[2]));
    if (owner != key || bp_share_vertex(tris, i, j)) continue;
    if (EMIT) {
      const int64_t a = i < j ? i : j, b = i < j ? j : i;
      pair_keys[o++] = (uint64_t)a * (uint64_t)nT + (uint64_t)b;
    }
    ++n;
  }
  if (!EMIT) cnt[r] = n;
}

__global__ void k_bp_unpack(const uint64_t* __restrict__ pair_keys, int64_t P, int64_t nT, int2* __restrict__ pairs) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= P) return;
  const uint64_t key = pair_keys[k];
  pairs[k] = make_int2((int)(key / (uint64_t)nT), (int)(key % (uint64_t)nT));
}

}  // namespace ttb
