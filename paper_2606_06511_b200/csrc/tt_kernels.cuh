// tt_kernels.cuh -- sm_100a kernels of the hot path.
//
//   K1  k_classify      a1+a2  : one thread per candidate pair, Moeller intervals, I_c, energy,
//                                ballot bitmask, per-CTA active count and energy partial
//   K2  k_compact       a2'    : order-preserving compaction of active pair ids (ballot/popc)
//   K3* symbolic kernels a4    : directed (triangle -> partner) entries, per-triangle column
//                                ranks, exclusive-row detection, general-row merge records
//   K4  k_assemble      a3+a4  : triangle-centric numeric phase, one thread per directed entry:
//                                recompute J analytically, write the 9 off-diagonal 3x3 blocks
//                                once, reduce diagonal blocks + gradient inside the CTA in fixed
//                                order (no atomics)
//   K5  k_merge / k_gather3    : general rows (vertices shared by several touched triangles)
//   K6  k_hessvec       a5     : matrix-free H.p with the same decomposition
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tt_geom.cuh"

namespace ttk {
using ttg::d3;

constexpr int CLS_THREADS = 256;   // K1 / K2 CTA size (8 warps -> 8 mask words per CTA)
constexpr int ASM_THREADS = 128;   // K4 / K6 CTA size: 4 independent warps
constexpr int ASM_CHUNK = 32;      // directed entries per warp chunk (snapped to triangle boundaries)
constexpr int SYM_WARPS = 4;       // warps per CTA in the per-triangle symbolic kernels
constexpr int SYM_LMAX = 1536;     // longest row (in blocks) ranked in shared memory

template <typename T>
__device__ __forceinline__ d3 load_vertex(const T* __restrict__ pos, int v) {
  const T* p = pos + 3 * (int64_t)v;
  return ttg::mk((double)__ldg(p), (double)__ldg(p + 1), (double)__ldg(p + 2));
}

// Gathers the six vertices of candidate (ta, tb) translated by -a0 (local frame: kills the
// cancellation in D.P and keeps fp32 inputs well scaled).  Returns false if the triangles share a
// vertex index ("topologically adjacent").
template <typename T>
__device__ __forceinline__ bool gather_pair(const T* __restrict__ pos, const int* __restrict__ tris,
                                            int ta, int tb, int (&va)[3], int (&vb)[3], d3 (&a)[3],
                                            d3 (&b)[3]) {
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    va[m] = __ldg(tris + 3 * (int64_t)ta + m);
    vb[m] = __ldg(tris + 3 * (int64_t)tb + m);
  }
  bool adj = false;
#pragma unroll
  for (int m = 0; m < 3; ++m)
#pragma unroll
    for (int n = 0; n < 3; ++n) adj |= (va[m] == vb[n]);
  if (adj) return false;
  const d3 o = load_vertex(pos, va[0]);
  a[0] = ttg::mk(0.0, 0.0, 0.0);
  a[1] = load_vertex(pos, va[1]) - o;
  a[2] = load_vertex(pos, va[2]) - o;
#pragma unroll
  for (int m = 0; m < 3; ++m) b[m] = load_vertex(pos, vb[m]) - o;
  return true;
}

// Fixed-order CTA reduction of one double per thread (warp shuffle tree, then warp 0).
template <int THREADS>
__device__ __forceinline__ double block_sum(double v, double* smem /*[THREADS/32]*/) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) smem[w] = v;
  __syncthreads();
  double r = 0.0;
  if (w == 0) {
    r = (l < THREADS / 32) ? smem[l] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
  }
  return r;  // valid in thread 0
}

// ------------------------------------------------------------------------------------------ K1
template <typename T>
__global__ void __launch_bounds__(CLS_THREADS)
k_classify(const T* __restrict__ pos, const int* __restrict__ tris, const int2* __restrict__ pairs,
           int64_t P, double sigma, uint32_t* __restrict__ mask, int* __restrict__ blk_count,
           double* __restrict__ blk_energy, T* __restrict__ e_pp, T* __restrict__ tc_out) {
  __shared__ double s_e[CLS_THREADS / 32];
  __shared__ int s_c[CLS_THREADS / 32];
  const int64_t k = (int64_t)blockIdx.x * CLS_THREADS + threadIdx.x;
  bool active = false;
  double tc0 = 0.0, tc1 = 0.0, en = 0.0;
  if (k < P) {
    const int2 pr = __ldg(pairs + k);
    int va[3], vb[3];
    d3 a[3], b[3];
    if (gather_pair(pos, tris, pr.x, pr.y, va, vb, a, b)) {
      ttg::PairGeom g;
      active = ttg::pair_intervals(a[0], a[1], a[2], b[0], b[1], b[2], sigma, g);
      if (active) {
        tc0 = g.tc0;
        tc1 = g.tc1;
        const double pr2 = tc0 * tc1;
        en = pr2 * pr2;  // Eq. 2
      }
    }
    if (e_pp) e_pp[k] = (T)en;
    if (tc_out) {
      tc_out[2 * k] = (T)tc0;
      tc_out[2 * k + 1] = (T)tc1;
    }
  }
  const uint32_t bal = __ballot_sync(0xffffffffu, active);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) {
    const int64_t word = (int64_t)blockIdx.x * (CLS_THREADS / 32) + w;
    if (word * 32 < P) mask[word] = bal;
    s_c[w] = __popc(bal);
  }
  const double e = block_sum<CLS_THREADS>(en, s_e);
  if (threadIdx.x == 0) {
    int c = 0;
#pragma unroll
    for (int i = 0; i < CLS_THREADS / 32; ++i) c += s_c[i];
    blk_count[blockIdx.x] = c;
    blk_energy[blockIdx.x] = e;
  }
}

// Fixed-order sum of n doubles by ONE CTA (deterministic), scaled, written as T.
template <typename T>
__global__ void __launch_bounds__(1024) k_sum_partials(const double* __restrict__ part, int64_t n,
                                                       double scale, T* __restrict__ out) {
  __shared__ double s[32];
  double v = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) v += part[i];
  const double r = block_sum<1024>(v, s);
  if (threadIdx.x == 0) out[0] = (T)(r * scale);
}

__global__ void k_set_count(const int* __restrict__ blk_off, const int* __restrict__ blk_count,
                            int64_t nblk, int64_t* __restrict__ out_a, int64_t* __restrict__ out_b) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    const int64_t a = nblk > 0 ? (int64_t)blk_off[nblk - 1] + blk_count[nblk - 1] : 0;
    if (out_a) *out_a = a;
    if (out_b) *out_b = a;
  }
}

// ------------------------------------------------------------------------------------------ K2
__global__ void __launch_bounds__(CLS_THREADS)
k_compact(const uint32_t* __restrict__ mask, const int* __restrict__ blk_off, int64_t P,
          int* __restrict__ active_ids) {
  const int64_t k = (int64_t)blockIdx.x * CLS_THREADS + threadIdx.x;
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t word0 = (int64_t)blockIdx.x * (CLS_THREADS / 32);
  int before = 0;
  uint32_t mine = 0;
#pragma unroll
  for (int i = 0; i < CLS_THREADS / 32; ++i) {
    const uint32_t m = ((word0 + i) * 32 < P) ? __ldg(mask + word0 + i) : 0u;
    if (i < w) before += __popc(m);
    if (i == w) mine = m;
  }
  if ((mine >> l) & 1u) active_ids[blk_off[blockIdx.x] + before + __popc(mine & ((1u << l) - 1u))] = (int)k;
}

// ------------------------------------------------------------------------------------------ K3
// Directed entries: active pair k = (s,t) -> (s -> t, side 0) and (t -> s, side 1).
// key = (source << bitsT) | partner, payload = 2k + side (k = index into active_ids).
__global__ void k_emit_directed(const int2* __restrict__ pairs, const int* __restrict__ active_ids,
                                int64_t A, int bitsT, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= A) return;
  const int2 pr = __ldg(pairs + active_ids[k]);
  keys[2 * k] = ((uint64_t)(uint32_t)pr.x << bitsT) | (uint32_t)pr.y;
  keys[2 * k + 1] = ((uint64_t)(uint32_t)pr.y << bitsT) | (uint32_t)pr.x;
  vals[2 * k] = (uint32_t)(2 * k);
  vals[2 * k + 1] = (uint32_t)(2 * k + 1);
}

// Segment pointers from sorted keys: ptr[g] = first entry whose (key >> shift) >= g, g = 0..G.
__global__ void k_segment_ptr(const uint64_t* __restrict__ keys, int64_t n, int shift, int64_t G,
                              int* __restrict__ ptr) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e > n) return;
  const int64_t cur = (e < n) ? (int64_t)(keys[e] >> shift) : G;
  const int64_t prev = (e > 0) ? (int64_t)(keys[e - 1] >> shift) : -1;
  for (int64_t g = prev + 1; g <= cur; ++g) ptr[g] = (int)e;
}

// Touched triangles count their vertices (integer atomics: the RESULT is order independent).
__global__ void k_vertex_touch(const int* __restrict__ tris, const int* __restrict__ tptr, int64_t nT,
                               int* __restrict__ vcnt, int* __restrict__ tflag) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nT) return;
  const int touched = tptr[s + 1] > tptr[s];
  tflag[s] = touched;
  if (touched) {
#pragma unroll
    for (int m = 0; m < 3; ++m) atomicAdd(vcnt + tris[3 * s + m], 1);
  }
}

// Per touched triangle s (one warp): candidate columns C = verts(partners in tadj order) ++ verts(s),
// L = 3 (deg + 1).  Ranks each candidate among C by counting (shared memory, all pairs), detects
// duplicates, decides which of the three rows are EXCLUSIVE (vertex used by no other touched
// triangle, no duplicate column) and records:
//   erank[e][n]   position of partner column (e, n) inside the row       (rank, or identity if dup)
//   drank[s][n]   position of the diagonal column n
//   rowlen[p]     = L for exclusive rows;  tlen[3s+m] = L for general rows (their blocks go to
//                 the merge workspace, one merge record each)
// layout = rank (columns ascending) when there is no duplicate, else identity (3j+n, diag last).
__global__ void __launch_bounds__(32 * SYM_WARPS)
k_tri_symbolic(const int* __restrict__ tris, const int* __restrict__ touched, int64_t n_touched,
               const int* __restrict__ tptr, const uint64_t* __restrict__ keys, int bitsT,
               const int* __restrict__ vcnt, int force_general, int* __restrict__ erank /*[2A][3]*/,
               int* __restrict__ drank /*[nT][3]*/, int* __restrict__ rowlen, int64_t* __restrict__ tlen /*[3nT]*/,
               uint8_t* __restrict__ slot_excl /*[3nT]*/) {
  __shared__ int s_c[SYM_WARPS][SYM_LMAX];
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t ti = (int64_t)blockIdx.x * SYM_WARPS + w;
  if (ti >= n_touched) return;
  const int s = touched[ti];
  const int e0 = tptr[s], deg = tptr[s + 1] - e0;
  const int L = 3 * (deg + 1);
  const uint64_t tmask = (1ull << bitsT) - 1ull;
  bool nodup = (L <= SYM_LMAX);
  int* c = s_c[w];
  if (nodup) {
    for (int idx = l; idx < L; idx += 32) {
      const int j = idx / 3, n = idx - 3 * j;
      const int t = (j < deg) ? (int)(keys[e0 + j] & tmask) : s;
      c[idx] = tris[3 * (int64_t)t + n];
    }
    __syncwarp();
    bool dup = false;
    for (int idx = l; idx < L; idx += 32) {
      const int me = c[idx];
      int eq = 0;
      for (int x = 0; x < L; ++x) eq += (c[x] == me);
      dup |= (eq > 1);
    }
    nodup = !__any_sync(0xffffffffu, dup);
  }
  for (int idx = l; idx < L; idx += 32) {
    int r = idx;
    if (nodup) {
      const int me = c[idx];
      r = 0;
      for (int x = 0; x < L; ++x) r += (c[x] < me);
    }
    const int j = idx / 3, n = idx - 3 * j;
    if (j < deg) erank[3 * (int64_t)(e0 + j) + n] = r;
    else drank[3 * (int64_t)s + n] = r;
  }
  if (l < 3) {
    const int p = tris[3 * (int64_t)s + l];
    const bool excl = nodup && !force_general && (vcnt[p] == 1);
    slot_excl[3 * (int64_t)s + l] = excl ? 1 : 0;
    tlen[3 * (int64_t)s + l] = excl ? 0 : L;
    if (excl) rowlen[p] = L;
  }
}

// General rows: one merge record per workspace block: key = (row vertex << bitsV) | column vertex,
// payload = workspace block index (assigned by the caller's iota; record index == block index).
__global__ void __launch_bounds__(32 * SYM_WARPS)
k_emit_records(const int* __restrict__ tris, const int* __restrict__ touched, int64_t n_touched,
               const int* __restrict__ tptr, const uint64_t* __restrict__ keys, int bitsT, int bitsV,
               const int* __restrict__ erank, const int* __restrict__ drank, const int64_t* __restrict__ toff,
               const uint8_t* __restrict__ slot_excl, uint64_t* __restrict__ rkeys, uint32_t* __restrict__ rvals) {
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t ti = (int64_t)blockIdx.x * SYM_WARPS + w;
  if (ti >= n_touched) return;
  const int s = touched[ti];
  const int e0 = tptr[s], deg = tptr[s + 1] - e0;
  const int L = 3 * (deg + 1);
  const uint64_t tmask = (1ull << bitsT) - 1ull;
  for (int m = 0; m < 3; ++m) {
    if (slot_excl[3 * (int64_t)s + m]) continue;
    const uint64_t p = (uint64_t)(uint32_t)tris[3 * (int64_t)s + m];
    const int64_t base = toff[3 * (int64_t)s + m];
    for (int idx = l; idx < L; idx += 32) {
      const int j = idx / 3, n = idx - 3 * j;
      const int t = (j < deg) ? (int)(keys[e0 + j] & tmask) : s;
      const int q = tris[3 * (int64_t)t + n];
      const int r = (j < deg) ? erank[3 * (int64_t)(e0 + j) + n] : drank[3 * (int64_t)s + n];
      rkeys[base + r] = (p << bitsV) | (uint32_t)q;
      rvals[base + r] = (uint32_t)(base + r);
    }
  }
}

// Sorted merge records -> run heads, per-row unique counts (integer atomics), first ordinal per row.
__global__ void k_record_heads(const uint64_t* __restrict__ rkeys, int64_t R, int* __restrict__ head) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= R) return;
  head[r] = (r == 0 || rkeys[r] != rkeys[r - 1]) ? 1 : 0;
}
__global__ void k_record_rows(const uint64_t* __restrict__ rkeys, int64_t R, int bitsV,
                              const int* __restrict__ head, const int* __restrict__ ord_incl,
                              int* __restrict__ rowlen, int* __restrict__ rowfirst, int* __restrict__ run_start) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= R) return;
  if (!head[r]) return;
  const int p = (int)(rkeys[r] >> bitsV);
  const int ord = ord_incl[r] - 1;
  run_start[ord] = (int)r;
  atomicAdd(rowlen + p, 1);
  if (r == 0 || (int)(rkeys[r - 1] >> bitsV) != p) rowfirst[p] = ord;
}
// destination block of every run + its column index; run_start[U] = R closes the last run.
__global__ void k_record_dest(const uint64_t* __restrict__ rkeys, int64_t U, int64_t R, int bitsV,
                              int* run_start, const int* __restrict__ rowptr,
                              const int* __restrict__ rowfirst, int* __restrict__ run_dest,
                              int* __restrict__ colind) {
  const int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (u == U) run_start[U] = (int)R;
  if (u >= U) return;
  const uint64_t key = rkeys[run_start[u]];
  const int p = (int)(key >> bitsV);
  const int q = (int)(key & ((1ull << bitsV) - 1ull));
  const int dest = rowptr[p] + ((int)u - rowfirst[p]);
  run_dest[u] = dest;
  colind[dest] = q;
}

// Exclusive rows: column indices + row bases (>= 0: block index into vals; < 0: -(workspace+1)).
__global__ void __launch_bounds__(32 * SYM_WARPS)
k_fill_rows(const int* __restrict__ tris, const int* __restrict__ touched, int64_t n_touched,
            const int* __restrict__ tptr, const uint64_t* __restrict__ keys, int bitsT,
            const int* __restrict__ erank, const int* __restrict__ drank, const int64_t* __restrict__ toff,
            const uint8_t* __restrict__ slot_excl, const int* __restrict__ rowptr,
            int64_t* __restrict__ rowbase /*[3nT]*/, int* __restrict__ colind) {
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t ti = (int64_t)blockIdx.x * SYM_WARPS + w;
  if (ti >= n_touched) return;
  const int s = touched[ti];
  const int e0 = tptr[s], deg = tptr[s + 1] - e0;
  const int L = 3 * (deg + 1);
  const uint64_t tmask = (1ull << bitsT) - 1ull;
  for (int m = 0; m < 3; ++m) {
    const int64_t slot = 3 * (int64_t)s + m;
    if (!slot_excl[slot]) {
      if (l == 0) rowbase[slot] = -(toff[slot] + 1);
      continue;
    }
    const int rp = rowptr[tris[slot]];
    if (l == 0) rowbase[slot] = rp;
    for (int idx = l; idx < L; idx += 32) {
      const int j = idx / 3, n = idx - 3 * j;
      const int t = (j < deg) ? (int)(keys[e0 + j] & tmask) : s;
      const int r = (j < deg) ? erank[3 * (int64_t)(e0 + j) + n] : drank[3 * (int64_t)s + n];
      colind[rp + r] = tris[3 * (int64_t)t + n];
    }
  }
}

// Work partition of K4/K6: chunk c owns the triangles whose first directed entry lies in
// [c*ASM_CHUNK, (c+1)*ASM_CHUNK): chunk_tri[c] = first such triangle (binary search in tptr).
__global__ void k_chunk_bounds(const int* __restrict__ tptr, int64_t nT, int64_t n_chunks,
                               int* __restrict__ chunk_tri) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c > n_chunks) return;
  const int64_t target = c * ASM_CHUNK;
  int64_t lo = 0, hi = nT;  // first s in [0,nT] with tptr[s] >= target
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (tptr[mid] >= target) hi = mid; else lo = mid + 1;
  }
  chunk_tri[c] = (int)lo;
}

// vertex -> touched (triangle, slot) incidence keys: key = vertex, payload = 3s+m
__global__ void k_emit_vslots(const int* __restrict__ tris, const int* __restrict__ touched,
                              int64_t n_touched, uint64_t* __restrict__ vkeys, uint32_t* __restrict__ vvals) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 3 * n_touched) return;
  const int64_t ti = i / 3;
  const int m = (int)(i - 3 * ti);
  const int s = touched[ti];
  vkeys[i] = (uint64_t)(uint32_t)tris[3 * (int64_t)s + m];
  vvals[i] = (uint32_t)(3 * s + m);
}

// ------------------------------------------------------------------------------------------ K4
// Triangle-centric numeric phase.  MODE 0: energy + gradient + Hessian blocks.  MODE 1: energy +
// gradient only.  MODE 2: H.p (K6).  One LANE per directed entry e = (source s -> partner t); one
// WARP per chunk of ~32 entries that starts and ends on a triangle boundary, so a warp owns every
// entry of the triangles it touches and needs no block-level barrier and no atomics.
// The pair is always evaluated in its canonical order (T_a = pairs[k,0]) so that both directed
// copies of a pair compute bit-identical J and take the same FILTER decision.
//
// Per entry the lane forms, with w0 = c00 g0 + c01 g1 and w1 = c01 g0 + c11 g1,
//   off-diagonal blocks  H[p_m, q_n] = g0_pm w0_qn^T + g1_pm w1_qn^T   (q_n = partner vertices):
//     exactly one contribution each -> staged through shared memory row by row and written out
//     by the whole warp in address order (coalesced) to their final place;
//   the diagonal 9x9 contribution (symmetric: 45 unique values) and the 9 gradient / H.p values:
//     staged in shared memory, then summed over the triangle's entries with lane = component,
//     entries in order (deterministic), accumulators carried in registers across rounds.
constexpr int NDIAG = 45;                 // upper triangle of the symmetric 9x9 diagonal block
constexpr int NRED_FULL = NDIAG + 9;      // + gradient of the three own vertices
constexpr int RED_STRIDE = 55;            // odd: conflict-free lane = entry writes
constexpr int OUT_STRIDE = 27;            // odd: conflict-free lane = entry writes

template <typename T>
struct AsmParams {
  const T* pos;
  const int* tris;
  const uint64_t* keys;     // sorted directed keys (source << bitsT | partner)
  const uint32_t* dvals;    // 2k + side
  const int* tptr;          // [nT+1]
  const int* chunk_tri;     // [n_chunks+1]
  const int* erank;         // [2A][3]
  const int* drank;         // [nT][3]
  const int64_t* rowbase;   // [3nT]
  T* vals;                  // final BSR values
  T* tvals;                 // merge workspace values
  T* tslot;                 // [3nT][3] per-slot gradient (MODE 0/1) or H.p (MODE 2) partials
  double* chunk_energy;     // [n_chunks]
  const T* pvec;            // MODE 2: p [nV,3]
  int64_t n_chunks;
  int bitsT;
  int hess_mode;
  double sigma;
};

struct AsmWarpSmem {
  double red[32 * RED_STRIDE];
  double out[32 * OUT_STRIDE];
  unsigned long long rowp[3][32];   // destination row base (element pointer) per entry and row
  int er[32][3];
  int src[32];
};

template <typename T, int MODE>
__global__ void __launch_bounds__(ASM_THREADS)
k_assemble(const AsmParams<T> P) {
  extern __shared__ __align__(16) unsigned char s_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  AsmWarpSmem& S = reinterpret_cast<AsmWarpSmem*>(s_raw)[warp];
  const int64_t c = (int64_t)blockIdx.x * (ASM_THREADS / 32) + warp;
  if (c >= P.n_chunks) return;  // warps are independent: no __syncthreads below
  const int tri_lo = P.chunk_tri[c], tri_hi = P.chunk_tri[c + 1];
  const int e_lo = P.tptr[tri_lo], e_hi = P.tptr[tri_hi];
  const uint64_t tmask = (1ull << P.bitsT) - 1ull;
  constexpr int NRED = (MODE == 0) ? NRED_FULL : 9;
  constexpr int GOFF = (MODE == 0) ? NDIAG : 0;  // first gradient / H.p component

  // lane = component bookkeeping for the reduction: comp0 = lane, comp1 = lane + 32
  int al0 = 0, be0 = 0, al1 = 0, be1 = 0;  // (alpha, beta) of the diagonal components
  if (MODE == 0) {
    int k = 0;
    for (int a = 0; a < 9; ++a)
      for (int b = a; b < 9; ++b, ++k) {
        if (k == lane) { al0 = a; be0 = b; }
        if (k == lane + 32) { al1 = a; be1 = b; }
      }
  }
  double acc0 = 0.0, acc1 = 0.0, e_acc = 0.0;
  int cur = -1;

  auto flush = [&](int s) {
    if (MODE == 0) {
      const int64_t rb0 = P.rowbase[3 * (int64_t)s], rb1 = P.rowbase[3 * (int64_t)s + 1], rb2 = P.rowbase[3 * (int64_t)s + 2];
      const int dr0 = P.drank[3 * (int64_t)s], dr1 = P.drank[3 * (int64_t)s + 1], dr2 = P.drank[3 * (int64_t)s + 2];
      auto put = [&](int a, int b, double v) {  // D[a][b] and its mirror D[b][a]
        const int m = a / 3, i = a - 3 * m, n = b / 3, j = b - 3 * n;
        {
          const int64_t rb = (m == 0) ? rb0 : (m == 1) ? rb1 : rb2;
          const int dr = (n == 0) ? dr0 : (n == 1) ? dr1 : dr2;
          T* rowp = (rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1));
          rowp[9 * (int64_t)dr + 3 * i + j] = (T)v;
        }
        if (a != b) {
          const int64_t rb = (n == 0) ? rb0 : (n == 1) ? rb1 : rb2;
          const int dr = (m == 0) ? dr0 : (m == 1) ? dr1 : dr2;
          T* rowp = (rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1));
          rowp[9 * (int64_t)dr + 3 * j + i] = (T)v;
        }
      };
      put(al0, be0, acc0);
      if (lane + 32 < NDIAG) put(al1, be1, acc1);
      else if (lane + 32 < NRED_FULL) P.tslot[9 * (int64_t)s + (lane + 32 - NDIAG)] = (T)acc1;
    } else {
      if (lane < 9) P.tslot[9 * (int64_t)s + lane] = (T)acc0;
    }
  };

  for (int base = e_lo; base < e_hi; base += 32) {
    const int e = base + lane;
    const bool valid = e < e_hi;
    const int nvalid = min(32, e_hi - base);
    int s = -1;
    double g0[18], g1[18];
    ttg::Coefs cf = {0, 0, 0, 0, 0};
    double hp0 = 0.0, hp1 = 0.0;  // MODE 2: M (J p_loc)
#pragma unroll
    for (int i = 0; i < 18; ++i) { g0[i] = 0.0; g1[i] = 0.0; }
    if (valid) {
      const uint64_t key = P.keys[e];
      s = (int)(key >> P.bitsT);
      const int side = (int)(P.dvals[e] & 1u);
      const int t = (int)(key & tmask);
      const int2 pr = side ? make_int2(t, s) : make_int2(s, t);  // canonical (pairs[k,0], pairs[k,1])
      int va[3], vb[3];
      d3 a[3], b[3];
      gather_pair(P.pos, P.tris, pr.x, pr.y, va, vb, a, b);
      ttg::PairGeom q;
      ttg::pair_intervals(a[0], a[1], a[2], b[0], b[1], b[2], P.sigma, q);  // active by construction
      ttg::pair_derivs(a[0], a[1], a[2], b[0], b[1], b[2], P.sigma, q, g0, g1);
      cf = ttg::pair_coefs(q.tc0, q.tc1, g0, g1, P.hess_mode);
      if (side == 0) {
        const double tt = q.tc0 * q.tc1;
        e_acc += tt * tt;  // Eq. 2, counted once per pair
      }
      if (MODE == 2) {
        double j0 = 0.0, j1 = 0.0;
#pragma unroll
        for (int v = 0; v < 3; ++v) {
          const d3 pa = load_vertex(P.pvec, va[v]);
          const d3 pb = load_vertex(P.pvec, vb[v]);
          j0 += g0[3 * v] * pa.x + g0[3 * v + 1] * pa.y + g0[3 * v + 2] * pa.z;
          j0 += g0[9 + 3 * v] * pb.x + g0[9 + 3 * v + 1] * pb.y + g0[9 + 3 * v + 2] * pb.z;
          j1 += g1[3 * v] * pa.x + g1[3 * v + 1] * pa.y + g1[3 * v + 2] * pa.z;
          j1 += g1[9 + 3 * v] * pb.x + g1[9 + 3 * v + 1] * pb.y + g1[9 + 3 * v + 2] * pb.z;
        }
        hp0 = cf.c00 * j0 + cf.c01 * j1;
        hp1 = cf.c01 * j0 + cf.c11 * j1;
      }
      if (side) {  // make "own" = first nine entries: swap the halves of g0, g1
#pragma unroll
        for (int i = 0; i < 9; ++i) {
          double t0 = g0[i]; g0[i] = g0[9 + i]; g0[9 + i] = t0;
          double t1 = g1[i]; g1[i] = g1[9 + i]; g1[9 + i] = t1;
        }
      }
    }
    // ---- stage the values to be reduced over the triangle: lane = entry ----
    S.src[lane] = s;
    {
      double* red = S.red + lane * RED_STRIDE;
      if (MODE == 0) {
        double d0[9], d1[9];
#pragma unroll
        for (int i = 0; i < 9; ++i) {
          d0[i] = cf.c00 * g0[i] + cf.c01 * g1[i];
          d1[i] = cf.c01 * g0[i] + cf.c11 * g1[i];
        }
        int k = 0;
#pragma unroll
        for (int a = 0; a < 9; ++a)
#pragma unroll
          for (int b = a; b < 9; ++b, ++k) red[k] = g0[a] * d0[b] + g1[a] * d1[b];
      }
#pragma unroll
      for (int i = 0; i < 9; ++i)
        red[GOFF + i] = (MODE == 2) ? (hp0 * g0[i] + hp1 * g1[i]) : (cf.cg0 * g0[i] + cf.cg1 * g1[i]);
    }
    if (MODE == 0) {
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        unsigned long long ptr = 0ull;
        if (valid) {
          const int64_t rb = P.rowbase[3 * (int64_t)s + m];
          ptr = (unsigned long long)((rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1)));
          S.er[lane][m] = P.erank[3 * (int64_t)e + m];
        }
        S.rowp[m][lane] = ptr;
      }
    }
    __syncwarp();
    // ---- reduction over entries, lane = component, fixed order ----
    for (int i = 0; i < nvalid; ++i) {
      const int si = S.src[i];
      if (si != cur) {  // warp-uniform
        if (cur >= 0) flush(cur);
        acc0 = 0.0;
        acc1 = 0.0;
        cur = si;
      }
      if (lane < NRED) acc0 += S.red[i * RED_STRIDE + lane];
      if (NRED > 32 && lane + 32 < NRED) acc1 += S.red[i * RED_STRIDE + lane + 32];
    }
    // ---- off-diagonal blocks, one row of the source triangle at a time ----
    if (MODE == 0) {
      double w0[9], w1[9];  // partner side: entries 9..17
#pragma unroll
      for (int i = 0; i < 9; ++i) {
        w0[i] = cf.c00 * g0[9 + i] + cf.c01 * g1[9 + i];
        w1[i] = cf.c01 * g0[9 + i] + cf.c11 * g1[9 + i];
      }
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        double* o = S.out + lane * OUT_STRIDE;
#pragma unroll
        for (int n = 0; n < 3; ++n)
#pragma unroll
          for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j)
              o[9 * n + 3 * i + j] = g0[3 * m + i] * w0[3 * n + j] + g1[3 * m + i] * w1[3 * n + j];
        __syncwarp();
        const int total = nvalid * 27;
        for (int f = lane; f < total; f += 32) {
          const int ee = f / 27, r = f - 27 * ee;
          const int n = r / 9, q = r - 9 * n;
          T* rowp = reinterpret_cast<T*>(S.rowp[m][ee]);
          rowp[9 * (int64_t)S.er[ee][n] + q] = (T)S.out[f];
        }
        __syncwarp();
      }
    } else {
      __syncwarp();
    }
  }
  if (cur >= 0) flush(cur);
  if (MODE != 2) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_down_sync(0xffffffffu, e_acc, o);
    if (lane == 0) P.chunk_energy[c] = e_acc;
  }
}

// ------------------------------------------------------------------------------------------ K5
// General rows: destination block u = sum of its workspace blocks, in sorted (stable) order.
template <typename T>
__global__ void k_merge(const int* __restrict__ run_start, const int* __restrict__ run_dest,
                        const uint32_t* __restrict__ rvals, int64_t U, const T* __restrict__ tvals,
                        T* __restrict__ vals) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 9 * U) return;
  const int64_t u = i / 9;
  const int comp = (int)(i - 9 * u);
  double acc = 0.0;
  for (int r = run_start[u]; r < run_start[u + 1]; ++r) acc += (double)tvals[9 * (int64_t)rvals[r] + comp];
  vals[9 * (int64_t)run_dest[u] + comp] = (T)acc;
}

// out[v] = sum over touched slots of vertex v of tslot[slot] (sorted incidence, fixed order);
// zero for vertices no active pair touches.
template <typename T>
__global__ void k_gather3(const int* __restrict__ vptr, const uint32_t* __restrict__ vslots, int64_t nV,
                          const T* __restrict__ tslot, T* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 3 * nV) return;
  const int64_t v = i / 3;
  const int comp = (int)(i - 3 * v);
  double acc = 0.0;
  for (int j = vptr[v]; j < vptr[v + 1]; ++j) acc += (double)tslot[3 * (int64_t)vslots[j] + comp];
  out[i] = (T)acc;
}

__global__ void k_iota(uint32_t* __restrict__ v, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) v[i] = (uint32_t)i;
}

__global__ void k_i64_to_i32(const int64_t* __restrict__ in, int64_t n, int* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (int)in[i];
}

}  // namespace ttk
