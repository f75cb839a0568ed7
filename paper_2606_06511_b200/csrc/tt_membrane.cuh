// tt_membrane.cuh -- the membrane term of the untangling demo (Fig. 2: the paper
// optimises meshes inside a simulation whose elastic model it does not give; reading A18 takes the simplest
// textbook one, springs on the mesh's own edges):
//     E_m(x) = k/2 sum over unique edges (i, j) of (|x_i - x_j| - L_ij)^2,     L_ij = |r_i - r_j| at the rest positions,
//     grad_i = k sum_j (|d| - L) n,  d = x_i - x_j,  n = d / |d|,
//     H p at i = sum_j K (p_i - p_j),   K = k [ n n^T + max(0, 1 - L / |d|) (I - n n^T) ]   (compressed springs clamped: PSD).
// The GPU's way: a vertex -> neighbour adjacency (every edge twice, as two half-edges) built once per mesh by sort +
// unique; one THREAD PER VERTEX walks its neighbours in ascending order, so gradient, H p and the diagonal blocks need
// no atomics and are deterministic; arithmetic in fp64 whatever the storage type.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ttm {

constexpr int MB_THREADS = 256;

// the six half-edges of every triangle as keys (v << 32 | u); a degenerate edge (v == u) gets the key n_verts << 32,
// which sorts after every real one
__global__ void __launch_bounds__(MB_THREADS)
k_half_edges(const int* __restrict__ tris, int64_t nT, int64_t nV, unsigned long long* __restrict__ keys) {
  const int64_t t = (int64_t)blockIdx.x * MB_THREADS + threadIdx.x;
  if (t >= nT) return;
  const int a = tris[3 * t], b = tris[3 * t + 1], c = tris[3 * t + 2];
  const int e[6][2] = {{a, b}, {b, a}, {b, c}, {c, b}, {c, a}, {a, c}};
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    const unsigned long long v = (unsigned)e[i][0], u = (unsigned)e[i][1];
    keys[6 * t + i] = (v == u) ? ((unsigned long long)nV << 32) : ((v << 32) | u);
  }
}
// unique sorted keys -> neighbour ids and rest lengths
template <typename T>
__global__ void __launch_bounds__(MB_THREADS)
k_adjacency(const unsigned long long* __restrict__ keys, int64_t n, int64_t nV, const T* __restrict__ rest_pos,
            int* __restrict__ adj, double* __restrict__ rest) {
  const int64_t e = (int64_t)blockIdx.x * MB_THREADS + threadIdx.x;
  if (e >= n) return;
  const int64_t v = (int64_t)(keys[e] >> 32), u = (int64_t)(keys[e] & 0xffffffffull);
  if (v >= nV) {
    adj[e] = 0;
    rest[e] = 0.0;
    return;
  }
  const double dx = (double)rest_pos[3 * v] - (double)rest_pos[3 * u], dy = (double)rest_pos[3 * v + 1] - (double)rest_pos[3 * u + 1],
               dz = (double)rest_pos[3 * v + 2] - (double)rest_pos[3 * u + 2];
  adj[e] = (int)u;
  rest[e] = sqrt(dx * dx + dy * dy + dz * dz);
}

// MODE 0: energy partial per CTA + gradient (written, or added to `out` with accumulate; `out` may be NULL)
// MODE 1: out (+)= H_m p          MODE 2: out[v] = (D_v + mu I)^-1, D_v = sum of the K of v's edges  (3 x 3, row major)
template <typename T, int MODE>
__global__ void __launch_bounds__(MB_THREADS)
k_membrane(const T* __restrict__ pos, const int* __restrict__ ptr, const int* __restrict__ adj, const double* __restrict__ rest,
           int64_t nV, double k, const T* __restrict__ p, double mu, int accumulate, T* __restrict__ out,
           double* __restrict__ e_part) {
  __shared__ double s_e[MB_THREADS / 32];
  const int64_t v = (int64_t)blockIdx.x * MB_THREADS + threadIdx.x;
  double en = 0.0;
  if (v < nV) {
    const double x0 = (double)pos[3 * v], x1 = (double)pos[3 * v + 1], x2 = (double)pos[3 * v + 2];
    double p0 = 0.0, p1 = 0.0, p2 = 0.0;
    if (MODE == 1) { p0 = (double)p[3 * v]; p1 = (double)p[3 * v + 1]; p2 = (double)p[3 * v + 2]; }
    double a[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};  // MODE 0 / 1: a[0..2]; MODE 2: the block
    for (int e = ptr[v]; e < ptr[v + 1]; ++e) {
      const int64_t u = adj[e];
      const double d0 = x0 - (double)pos[3 * u], d1 = x1 - (double)pos[3 * u + 1], d2 = x2 - (double)pos[3 * u + 2];
      const double ln = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
      if (!(ln > 0.0)) continue;  // coincident vertices: no direction, no force
      const double L = rest[e], inv = 1.0 / ln;
      const double n0 = d0 * inv, n1 = d1 * inv, n2 = d2 * inv;
      if (MODE == 0) {
        const double s = k * (ln - L);
        a[0] += s * n0; a[1] += s * n1; a[2] += s * n2;
        en += 0.25 * k * (ln - L) * (ln - L);  // every edge is seen from both ends
      } else {
        const double c = fmax(0.0, 1.0 - L * inv);
        if (MODE == 1) {
          const double q0 = p0 - (double)p[3 * u], q1 = p1 - (double)p[3 * u + 1], q2 = p2 - (double)p[3 * u + 2];
          const double nq = n0 * q0 + n1 * q1 + n2 * q2;
          a[0] += k * (n0 * nq + c * (q0 - n0 * nq));
          a[1] += k * (n1 * nq + c * (q1 - n1 * nq));
          a[2] += k * (n2 * nq + c * (q2 - n2 * nq));
        } else {
          const double n[3] = {n0, n1, n2};
#pragma unroll
          for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) a[3 * i + j] += k * (n[i] * n[j] * (1.0 - c) + (i == j ? c : 0.0));
        }
      }
    }
    if (MODE == 2) {
      a[0] += mu; a[4] += mu; a[8] += mu;
      const double c00 = a[4] * a[8] - a[5] * a[7], c01 = a[5] * a[6] - a[3] * a[8], c02 = a[3] * a[7] - a[4] * a[6];
      const double id = 1.0 / (a[0] * c00 + a[1] * c01 + a[2] * c02);
      T* o = out + 9 * v;
      o[0] = (T)(c00 * id); o[1] = (T)((a[2] * a[7] - a[1] * a[8]) * id); o[2] = (T)((a[1] * a[5] - a[2] * a[4]) * id);
      o[3] = (T)(c01 * id); o[4] = (T)((a[0] * a[8] - a[2] * a[6]) * id); o[5] = (T)((a[2] * a[3] - a[0] * a[5]) * id);
      o[6] = (T)(c02 * id); o[7] = (T)((a[1] * a[6] - a[0] * a[7]) * id); o[8] = (T)((a[0] * a[4] - a[1] * a[3]) * id);
    } else if (out) {
#pragma unroll
      for (int i = 0; i < 3; ++i) out[3 * v + i] = (T)((accumulate ? (double)out[3 * v + i] : 0.0) + a[i]);
    }
  }
  if (MODE == 0) {  // fixed-order CTA sum (shuffle tree, then warp 0)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) en += __shfl_down_sync(0xffffffffu, en, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) s_e[w] = en;
    __syncthreads();
    if (w == 0) {
      double r = (l < MB_THREADS / 32) ? s_e[l] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
      if (l == 0) e_part[blockIdx.x] = r;
    }
  }
}

}  // namespace ttm
