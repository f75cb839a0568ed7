// tt_kernels.cuh -- sm_100a kernels of the hot path.
//
//   K1  k_classify      a1+a2  : one thread per candidate pair, Moeller intervals, I_c, energy,
//                                ballot bitmask, per-CTA active count and energy partial
//   K2  k_compact       a2'    : order-preserving compaction of active pair ids (ballot/popc)
//   K3* symbolic kernels a4    : directed (triangle -> partner) entries, per-triangle column
//                                ranks, exclusive-row detection, general-row merge records
//   K4  k_assemble_tile a3+a4  : triangle-centric numeric phase, one lane per directed entry, one
//                                warp per round of whole triangles: recompute J analytically,
//                                build each row's run of 3x3 blocks in a shared-memory tile,
//                                sum diagonal rows + gradient in fixed order (no atomics), write
//                                the runs out with TMA bulk copies (k_assemble_long_tile /
//                                k_assemble_long_direct: triangles with more than 32 partners)
//   K5  k_merge / k_gather3    : general rows (vertices shared by several touched triangles)
//   K6  k_entry_pipe    a5     : matrix-free H.p (and the gradient-only call), same rounds
//                                (k_entry_reduce: triangles with more than 32 partners)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tt_geom.cuh"

namespace ttk {
using ttg::d3;

#ifndef TT_CLS_THREADS
#define TT_CLS_THREADS 128         // measured: K1 0.675 ms with 256 threads, 0.645 with 128, 0.633 with 64 (10 M candidates) -- a CTA's
#endif                             // slot is held until its slowest gather returns; 64 costs the mesh configs more partials than it saves
constexpr int CLS_THREADS = TT_CLS_THREADS;   // K1 / K2 CTA size (4 warps -> 4 mask words per CTA)
constexpr int SYM_WARPS = 4;       // warps per CTA in the per-triangle symbolic kernels
constexpr int SYM_LMAX = 1536;     // longest row (in blocks) ranked in shared memory
constexpr int SLOT_PART = (int)0x80000000;  // flag in sinfo.x: the slot is a part of a split triangle

// One vertex = three consecutive values at an address that is only value-aligned: exactly one of
// p, p + 1 is aligned for a two-value load, so a vertex costs two gather requests (one 2-wide, one
// 1-wide; addresses selected, no divergence, nothing read outside the vertex) instead of three.
// K1 is bound by gather requests: 0.69 -> 0.63 ms at 10M candidates.  (Not used in K4 / K6: there the
// selects cost more than the saved request, measured.)
template <typename T> struct Pair2;
template <> struct Pair2<double> { using type = double2; };
template <> struct Pair2<float> { using type = float2; };
template <typename T>
__device__ __forceinline__ void load3(const T* __restrict__ p, double& x, double& y, double& z) {
  using V2 = typename Pair2<T>::type;
  const bool lo = (reinterpret_cast<uintptr_t>(p) & (2 * sizeof(T) - 1)) == 0;
  const V2 q = __ldg(reinterpret_cast<const V2*>(lo ? p : p + 1));
  const T s = __ldg(lo ? p + 2 : p);
  x = (double)(lo ? q.x : s);
  y = (double)(lo ? q.y : q.x);
  z = (double)(lo ? s : q.y);
}
__device__ __forceinline__ int pick3(int i, int v0, int v1, int v2) { return i == 0 ? v0 : (i == 1 ? v1 : v2); }
__device__ __forceinline__ void load3i(const int* __restrict__ p, int (&v)[3]) {  // same, for a triangle's vertex ids
  const bool lo = (reinterpret_cast<uintptr_t>(p) & 7) == 0;
  const int2 q = __ldg(reinterpret_cast<const int2*>(lo ? p : p + 1));
  const int s = __ldg(lo ? p + 2 : p);
  v[0] = lo ? q.x : s;
  v[1] = lo ? q.y : q.x;
  v[2] = lo ? s : q.y;
}
template <typename T>
__device__ __forceinline__ d3 load_vertex(const T* __restrict__ pos, int v) {
  d3 r;
  load3(pos + 3 * (int64_t)v, r.x, r.y, r.z);
  return r;
}

// Gathers the six vertices of candidate (ta, tb) translated by -a0 (local frame: kills the
// cancellation in D.P and keeps fp32 inputs well scaled).  Returns false if the triangles share a
// vertex index ("topologically adjacent").
template <typename T>
__device__ __forceinline__ bool gather_pair(const T* __restrict__ pos, const int* __restrict__ tris,
                                            int ta, int tb, int (&va)[3], int (&vb)[3], d3 (&a)[3],
                                            d3 (&b)[3]) {
  load3i(tris + 3 * (int64_t)ta, va);
  load3i(tris + 3 * (int64_t)tb, vb);
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
#ifndef TT_CLS_MIN_CTAS
#define TT_CLS_MIN_CTAS 6   // 80 registers, 24 warps / SM (more CTAs per SM need fewer registers and spill: measured slower)
#endif
// Per-candidate record written by K1 for the symbolic phase: the recorded branch decisions (ttg::pair_config, 12 bits).
template <typename T>
__global__ void __launch_bounds__(CLS_THREADS, TT_CLS_MIN_CTAS)
k_classify(const T* __restrict__ pos, const int* __restrict__ tris, const int2* __restrict__ pairs,
           int64_t P, double sigma, uint32_t* __restrict__ mask, int* __restrict__ blk_count,
           double* __restrict__ blk_energy, T* __restrict__ e_pp, T* __restrict__ tc_out,
           uint16_t* __restrict__ rec_out, int* __restrict__ deg) {
  __shared__ double s_e[CLS_THREADS / 32];
  __shared__ int s_c[CLS_THREADS / 32];
  const int64_t k = (int64_t)blockIdx.x * CLS_THREADS + threadIdx.x;
  bool active = false;
  double tc0 = 0.0, tc1 = 0.0, en = 0.0;
  unsigned cfg = 0u;
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
        cfg = ttg::pair_config(g);
        if (deg) {
          // Counting sort of the directed entries by source triangle, first half: the histogram (integer
          // reductions without a return value: the RESULT does not depend on the schedule).  The place of an entry
          // inside its triangle's segment is taken by k_compact; K1 runs at 35 % occupancy on a chain of dependent
          // gathers and an atomic whose value it has to wait for costs it 10 % (measured).
          atomicAdd(deg + pr.x, 1);
          atomicAdd(deg + pr.y, 1);
        }
      }
    }
    if (rec_out) rec_out[k] = (uint16_t)cfg;
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

// Fixed-order sum of n doubles (deterministic), scaled, written as T.  Large n: k_sum_stage first
// reduces fixed slices of SUM_SLICE values per CTA, then ONE CTA sums the slice sums.
constexpr int SUM_SLICE = 8192;
__global__ void __launch_bounds__(256) k_sum_stage(const double* __restrict__ part, int64_t n, double* __restrict__ out) {
  __shared__ double s[8];
  const int64_t lo = (int64_t)blockIdx.x * SUM_SLICE, hi = min(lo + (int64_t)SUM_SLICE, n);
  double v = 0.0;
  for (int64_t i = lo + threadIdx.x; i < hi; i += 256) v += part[i];
  const double r = block_sum<256>(v, s);
  if (threadIdx.x == 0) out[blockIdx.x] = r;
}
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
// Order-preserving compaction of the active pair ids (ballot / popc positions + per-CTA offsets) and, in
// the same pass, the COUNTING SORT of the directed entries by source triangle: active pair (s, t) becomes
// the entries s -> t (side 0) and t -> s (side 1); K1 has counted the entries of every triangle (deg), the
// scan of deg is tptr, and an entry takes the next free place of its triangle's segment (integer atomic on
// `fill`, zeroed by the caller).  The order INSIDE a segment is whatever the atomics give; the symbolic
// kernels sort every segment by (partner, side) before anything depends on it, so all results are
// deterministic (two entries with the same key are the same pair listed twice: bit-identical contributions).
//   ent[slot] = (partner triangle, side | recorded config of the canonical pair << 1)
__global__ void __launch_bounds__(CLS_THREADS)
k_compact(const uint32_t* __restrict__ mask, const int* __restrict__ blk_off, int64_t P,
          int* __restrict__ active_ids, const int2* __restrict__ pairs, const uint16_t* __restrict__ rec,
          const int* __restrict__ tptr, uint2* __restrict__ ent, int* __restrict__ fill) {
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
  if ((mine >> l) & 1u) {
    const int64_t a = (int64_t)blk_off[blockIdx.x] + before + __popc(mine & ((1u << l) - 1u));
    __stcs(active_ids + a, (int)k);
    if (ent) {
      // streaming loads / stores for everything that is touched once, so that the 8-byte scattered
      // stores of the entries find their lines still in L2 when the line's other entries arrive
      const int2 pr = __ldcs(pairs + k);
      const unsigned c = (unsigned)__ldcs(rec + k) << 1;
      const int sa = __ldg(tptr + pr.x) + atomicAdd(fill + pr.x, 1);
      const int sb = __ldg(tptr + pr.y) + atomicAdd(fill + pr.y, 1);
      ent[sa] = make_uint2((unsigned)pr.y, c);
      ent[sb] = make_uint2((unsigned)pr.x, c | 1u);
    }
  }
}

// Sort key of a directed entry inside its triangle's segment.
__device__ __forceinline__ unsigned long long entry_key(const uint2 e) {
  return ((unsigned long long)e.x << 1) | (unsigned long long)(e.y & 1u);
}

// ------------------------------------------------------------------------------------------ K3
// Segment pointers from sorted keys: ptr[g] = first entry whose (key >> shift) >= g, g = 0..G.  One thread per
// GROUP, binary search (a thread per ENTRY that fills the groups between its key and its predecessor's walks
// up to G groups alone when the keys are sparse: 147 us on the 1 M-triangle torus, measured, against 10 here).
__global__ void k_segment_ptr(const uint64_t* __restrict__ keys, int64_t n, int shift, int64_t G,
                              int* __restrict__ ptr) {
  const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g > G) return;
  int64_t lo = 0, hi = n;  // first e in [0, n] with (keys[e] >> shift) >= g
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if ((int64_t)(__ldg(keys + mid) >> shift) < g) lo = mid + 1;
    else hi = mid;
  }
  ptr[g] = (int)lo;
}

// Touched triangles count their vertices (integer atomics: the RESULT is order independent).
__global__ void k_vertex_touch(const int* __restrict__ tris, const int* __restrict__ deg, int64_t nT,
                               int* __restrict__ vcnt) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nT) return;
  if (deg[s] > 0) {
#pragma unroll
    for (int m = 0; m < 3; ++m) atomicAdd(vcnt + tris[3 * s + m], 1);
  }
}

// Sorts the n entries of one segment by (partner, side) into (partner_out, dvals_out), one warp: every
// entry counts the keys below it (ties by position: tied entries are identical pairs).  Keys are staged
// in shared memory when they fit (skey, cap entries), else read through L1.
__device__ __forceinline__ void warp_sort_segment(const uint2* __restrict__ ent, int n, unsigned long long* skey, int cap,
                                                  int* __restrict__ partner_out, uint16_t* __restrict__ dvals_out, int lane) {
  const bool staged = n <= cap;
  if (staged) {
    for (int j = lane; j < n; j += 32) skey[j] = entry_key(__ldg(ent + j));
    __syncwarp();
  }
  for (int j = lane; j < n; j += 32) {
    const uint2 me = __ldg(ent + j);
    const unsigned long long key = entry_key(me);
    int r = 0;
    if (staged) {
      for (int x = 0; x < n; ++x) {
        const unsigned long long kx = skey[x];
        r += (kx < key) || (kx == key && x < j);
      }
    } else {
      for (int x = 0; x < n; ++x) {
        const unsigned long long kx = entry_key(__ldg(ent + x));
        r += (kx < key) || (kx == key && x < j);
      }
    }
    partner_out[r] = (int)me.x;
    dvals_out[r] = (uint16_t)me.y;
  }
  __syncwarp();
}

// Per LONG touched triangle s that k_long_prep could not split (one warp; the segment is already sorted):
// candidate columns C = verts(partners in sorted order) ++ verts(s), L = 3 (deg + 1).  Ranks each
// candidate among C by counting (shared memory, all pairs), detects duplicates, decides which of the
// three rows are EXCLUSIVE (vertex used by no other touched triangle, no duplicate column) and records:
//   erank[e][n]   position of partner column (e, n) inside the row       (rank, or identity if dup)
//   drank[ti][n]  position of the diagonal column n
//   rowlen[p]     = L for exclusive rows;  tlen[3ti+m] = L for general rows (their blocks go to
//                 the merge workspace, one merge record each)
// Per-slot arrays (drank, tlen, toff, slot_excl, rowbase, tslot) are indexed by SLOT (here: the triangle's
// only slot): the numeric kernels then need no triangle id to find them.
// layout = rank (columns ascending) when there is no duplicate, else identity (3j+n, diag last).
// Duplicates are detected as in k_round_symbolic: the ranks of L distinct values sum to L (L - 1) / 2.
// Also writes the per-entry vertex ids (everts) of the triangle's entries.
__global__ void __launch_bounds__(32 * SYM_WARPS)
k_tri_symbolic(const int* __restrict__ tris, const int* __restrict__ touched, const int* __restrict__ n_long_dev,
               const int* __restrict__ tfirst, const int4* __restrict__ sinfo, const int* __restrict__ partner,
               const uint16_t* __restrict__ dvals, const int* __restrict__ vcnt, int force_general,
               int* __restrict__ erank /*[2A][3]*/, int* __restrict__ drank /*[n_touched][3]*/, int* __restrict__ rowlen,
               int64_t* __restrict__ tlen /*[3 n_touched]*/, uint8_t* __restrict__ slot_excl /*[3 n_touched]*/,
               const int* __restrict__ long_list, const int4* __restrict__ rdesc, int* __restrict__ vslot1,
               int* __restrict__ everts) {
  __shared__ __align__(8) int s_c[SYM_WARPS][SYM_LMAX];
  constexpr unsigned FULL = 0xffffffffu;
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t n_long = *n_long_dev;
  for (int64_t li = (int64_t)blockIdx.x * SYM_WARPS + w; li < n_long; li += (int64_t)gridDim.x * SYM_WARPS) {
    const int64_t sl = rdesc[long_list[li]].z;
    const int64_t ti = sinfo[sl].x;
    const int s = touched[ti];
    const int e0 = tfirst[ti], deg = tfirst[ti + 1] - e0;
    const int L = 3 * (deg + 1);
    int own[3];
    load3i(tris + 3 * (int64_t)s, own);
    // vertex ids of the canonical pair of every entry, both triangles in recorded (k, p, q) order
    for (int j = l; j < deg; j += 32) {
      const int64_t e = (int64_t)e0 + j;
      int cv[3];
      load3i(tris + 3 * (int64_t)partner[e], cv);
      const unsigned pay = dvals[e];
      const bool side = (pay & 1u) != 0u;
      const unsigned ca = (pay >> 1) & 63u, cb = (pay >> 7) & 63u;
      const int ka = (int)(ca & 3u), pa = (int)((ca >> 2) & 3u), kb = (int)(cb & 3u), pb = (int)((cb >> 2) & 3u);
      const int a0 = side ? cv[0] : own[0], a1 = side ? cv[1] : own[1], a2 = side ? cv[2] : own[2];
      const int b0 = side ? own[0] : cv[0], b1 = side ? own[1] : cv[1], b2 = side ? own[2] : cv[2];
      int2* o = reinterpret_cast<int2*>(everts + 6 * e);
      o[0] = make_int2(pick3(ka, a0, a1, a2), pick3(pa, a0, a1, a2));
      o[1] = make_int2(pick3(3 - ka - pa, a0, a1, a2), pick3(kb, b0, b1, b2));
      o[2] = make_int2(pick3(pb, b0, b1, b2), pick3(3 - kb - pb, b0, b1, b2));
    }
    bool nodup = (L <= SYM_LMAX);  // longer rows: identity layout, general rows
    int* c = s_c[w];
    if (nodup) {
      for (int idx = l; idx < L; idx += 32) {
        const int j = idx / 3, n = idx - 3 * j;
        const int t = (j < deg) ? partner[e0 + j] : s;
        c[idx] = tris[3 * (int64_t)t + n];
      }
      __syncwarp();
      long long sum = 0;
      for (int idx = l; idx < L; idx += 32) {
        const int me = c[idx];
        int r = 0;
        for (int x = 0; x < L; ++x) r += (c[x] < me);
        sum += r;
        const int j = idx / 3, n = idx - 3 * j;
        if (j < deg) erank[3 * (int64_t)(e0 + j) + n] = r;
        else drank[3 * sl + n] = r;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(FULL, sum, o);
      nodup = (2 * sum == (long long)L * (L - 1));
    }
    if (!nodup) {
      for (int idx = l; idx < L; idx += 32) {
        const int j = idx / 3, n = idx - 3 * j;
        if (j < deg) erank[3 * (int64_t)(e0 + j) + n] = idx;
        else drank[3 * sl + n] = idx;
      }
    }
    if (l < 3) {
      const int p = own[l == 0 ? 0 : (l == 1 ? 1 : 2)];
      const bool excl = nodup && !force_general && (vcnt[p] == 1);
      if (vcnt[p] == 1) vslot1[p] = (int)(3 * sl + l);  // the vertex's only slot (k_gather3)
      slot_excl[3 * sl + l] = excl ? 1 : 0;
      tlen[3 * sl + l] = excl ? 0 : L;
      if (excl) rowlen[p] = L;
    }
    __syncwarp();  // s_c is reused by the next triangle
  }
}

// General rows: one merge record per workspace block: key = (row vertex << bitsV) | column vertex,
// payload = workspace block index (assigned by the caller's iota; record index == block index).
// One warp per slot (parts have exclusive rows: nothing to emit).
__global__ void __launch_bounds__(32 * SYM_WARPS)
k_emit_records(const int* __restrict__ tris, const int* __restrict__ touched, int64_t n_slots,
               const int* __restrict__ sfirst, const int4* __restrict__ sinfo, const int* __restrict__ partner, int bitsV,
               const int* __restrict__ erank, const int* __restrict__ drank, const int64_t* __restrict__ toff,
               const uint8_t* __restrict__ slot_excl, uint64_t* __restrict__ rkeys, uint32_t* __restrict__ rvals) {
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t sl = (int64_t)blockIdx.x * SYM_WARPS + w;
  if (sl >= n_slots) return;
  const int4 si = sinfo[sl];
  if (si.x & SLOT_PART) return;
  const int s = touched[si.x];
  const int e0 = sfirst[sl], deg = sfirst[sl + 1] - e0;
  const int L = 3 * (deg + 1);
  for (int m = 0; m < 3; ++m) {
    if (slot_excl[3 * sl + m]) continue;
    const uint64_t p = (uint64_t)(uint32_t)tris[3 * (int64_t)s + m];
    const int64_t base = toff[3 * sl + m];
    for (int idx = l; idx < L; idx += 32) {
      const int j = idx / 3, n = idx - 3 * j;
      const int t = (j < deg) ? partner[e0 + j] : s;
      const int q = tris[3 * (int64_t)t + n];
      const int r = (j < deg) ? erank[3 * (int64_t)(e0 + j) + n] : drank[3 * sl + n];
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

// Long unsplittable triangles: column indices of their exclusive rows + row bases (>= 0: block index into
// vals; < 0: -(workspace + 1)).
__global__ void __launch_bounds__(32 * SYM_WARPS)
k_fill_rows(const int* __restrict__ tris, const int* __restrict__ touched, int64_t n_long,
            const int* __restrict__ sfirst, const int4* __restrict__ sinfo, const int* __restrict__ partner,
            const int* __restrict__ erank, const int* __restrict__ drank, const int64_t* __restrict__ toff,
            const uint8_t* __restrict__ slot_excl, const int* __restrict__ rowptr,
            int64_t* __restrict__ rowbase /*[3 n_slots]*/, int* __restrict__ colind,
            const int* __restrict__ long_list, const int4* __restrict__ rdesc) {
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t li = (int64_t)blockIdx.x * SYM_WARPS + w;
  if (li >= n_long) return;
  const int64_t sl = rdesc[long_list[li]].z;
  const int s = touched[sinfo[sl].x];
  const int e0 = sfirst[sl], deg = sfirst[sl + 1] - e0;
  const int L = 3 * (deg + 1);
  for (int m = 0; m < 3; ++m) {
    const int64_t slot = 3 * sl + m;
    if (!slot_excl[slot]) {
      if (l == 0) rowbase[slot] = -(toff[slot] + 1);
      continue;
    }
    const int rp = rowptr[tris[3 * (int64_t)s + m]];
    if (l == 0) rowbase[slot] = rp;
    for (int idx = l; idx < L; idx += 32) {
      const int j = idx / 3, n = idx - 3 * j;
      const int t = (j < deg) ? partner[e0 + j] : s;
      const int r = (j < deg) ? erank[3 * (int64_t)(e0 + j) + n] : drank[3 * sl + n];
      colind[rp + r] = tris[3 * (int64_t)t + n];
    }
  }
}

// Work partition of K4/K6.  A SLOT is what a warp treats as "one triangle's entries": a whole touched
// triangle, or -- for a triangle with more than RND_MAX_ENT partners whose row layout allows it
// (k_long_prep) -- a PART: a run of consecutive entries of its (partner-sorted) segment that does not
// straddle the position of the diagonal columns.  A ROUND is a run of consecutive slots with at most
// RND_MAX_ENT directed entries (one lane each) and RND_MAX_TRI slots; one warp owns one round.  Parts are
// cut wherever a round fills up, so rounds that meet a splittable long triangle are full.  A long
// triangle that cannot be split is a slot and a round of its own ("long": k_assemble_long*).
// Packing is greedy in touched order, restarted at every bucket of CHK_BUCKET touched triangles so that
// buckets pack in parallel (one thread per bucket; count pass, scan, fill pass).
constexpr int RND_MAX_ENT = 32;
// Slots per round: at most RND_MAX_TRI (the capacity every per-round array is sized for).  The packing LIMIT of one
// symbolic call is 16 or 8, chosen on the device from the mean number of entries per touched triangle: with one or
// two partners per triangle (1-5 M pairs on BASELINE's 2 M-triangle soup) 8 slots fill a third of a round's 32
// lanes; with five or more, rounds fill anyway and K4 runs 8 % faster with its per-slot loops unrolled 8 deep
// (measured; K4 is instantiated for both, K6 and the symbolic kernels do not care).
#ifndef TT_RND_MAX_TRI
#define TT_RND_MAX_TRI 16
#endif
constexpr int RND_MAX_TRI = TT_RND_MAX_TRI;
constexpr int RND_TRI_LOW = 8;
// limit = 16 iff  entries / touched < 3.5
__host__ __device__ inline int round_tri_limit(int64_t n_entries, int64_t n_touched) {
  return (RND_MAX_TRI > RND_TRI_LOW && 2 * n_entries < 7 * n_touched) ? RND_MAX_TRI : RND_TRI_LOW;
}
#ifndef TT_CHK_BUCKET
#define TT_CHK_BUCKET 128
#endif
constexpr int CHK_BUCKET = TT_CHK_BUCKET;

// Layout order of the triangles' entry segments.  K4 / K6 give one warp to a ROUND of consecutive slots with at most
// 32 directed entries, and a round costs the same whether 20 or 32 of its lanes work: what counts is the NUMBER of
// rounds.  Packing the triangles in id order fills 80-85 % of the lanes once triangles have 10-25 partners (two
// neighbours of 20 do not fit one round); nothing ties the segments to id order, though -- rows are addressed
// through rowbase -- so every bucket of ORD_BUCKET consecutive triangle ids is re-ordered here by best-fit-decreasing
// bin packing of the degrees into rounds of 32 (one thread per bucket), and the segments, the touched list, the
// slots and the rounds follow that order.  Simulated on the soup's measured degrees: 18 % fewer rounds at 20 M
// pairs, 11 % at 50 M, none below a mean degree of ~7 (there the 8-slot limit binds, not the 32 entries): such
// buckets keep their id order.  Triangles with more than 32 partners go first (their parts fill rounds anyway).
//   order[pos] = triangle id at layout position pos;  degp[pos] = its degree (degp[nT] = 0)
constexpr int ORD_BUCKET = 128;
__global__ void __launch_bounds__(64)
k_bucket_order(const int* __restrict__ deg, int64_t nT, const int64_t* __restrict__ n_active_dev, int* __restrict__ order,
               int* __restrict__ degp) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n_buckets = (nT + ORD_BUCKET - 1) / ORD_BUCKET;
  if (b == n_buckets) degp[nT] = 0;  // closes the scan (one extra thread)
  if (2 * *n_active_dev < 7 * nT) {  // fewer than 7 entries per triangle overall: id order, as a coalesced copy
    for (int64_t t = b; t < nT; t += (int64_t)gridDim.x * blockDim.x) {
      order[t] = (int)t;
      degp[t] = deg[t];
    }
    return;
  }
  if (b >= n_buckets) return;
  const int64_t t0 = b * ORD_BUCKET;
  const int n = (int)min((int64_t)ORD_BUCKET, nT - t0);
  short d[ORD_BUCKET];
  int sum = 0, touched = 0;
  for (int i = 0; i < n; ++i) {
    const int v = deg[t0 + i];
    d[i] = (short)min(v, 32767);
    sum += v;
    touched += v > 0;
  }
  if (sum < 7 * touched || n < 4) {  // few partners per triangle (or nothing to pack): id order
    for (int i = 0; i < n; ++i) {
      order[t0 + i] = (int)(t0 + i);
      degp[t0 + i] = deg[t0 + i];
    }
    return;
  }
  // stable counting sort by degree class (long first, then 32 .. 0)
  unsigned char srt[ORD_BUCKET];
  {
    int cnt[34];
    for (int k = 0; k < 34; ++k) cnt[k] = 0;
    for (int i = 0; i < n; ++i) cnt[33 - min((int)d[i], 33)]++;   // class 0 = long, 1 = 32, ..., 33 = 0
    int acc = 0;
    for (int k = 0; k < 34; ++k) { const int c = cnt[k]; cnt[k] = acc; acc += c; }
    for (int i = 0; i < n; ++i) srt[cnt[33 - min((int)d[i], 33)]++] = (unsigned char)i;
  }
  // best fit decreasing into rounds of RND_MAX_ENT entries and RND_TRI_LOW slots
  unsigned char rnd_of[ORD_BUCKET], room[ORD_BUCKET], cnt_r[ORD_BUCKET];
  short head[RND_MAX_ENT], nxt[ORD_BUCKET];   // open rounds by remaining room (singly linked)
  for (int r = 0; r < RND_MAX_ENT; ++r) head[r] = -1;
  int n_rounds = 0;
  for (int k = 0; k < n; ++k) {
    const int i = srt[k], di = d[i];
    if (di > RND_MAX_ENT || di == 0) {  // long triangles first, untouched ones last: rounds of their own in this order
      rnd_of[i] = (unsigned char)n_rounds;
      room[n_rounds] = 0;
      cnt_r[n_rounds] = RND_TRI_LOW;
      ++n_rounds;
      continue;
    }
    int r = di;
    while (r < RND_MAX_ENT && head[r] < 0) ++r;
    int q;
    if (r < RND_MAX_ENT) {  // the open round with the least room that still takes it
      q = head[r];
      head[r] = nxt[q];
    } else {
      q = n_rounds++;
      room[q] = RND_MAX_ENT;
      cnt_r[q] = 0;
    }
    rnd_of[i] = (unsigned char)q;
    room[q] = (unsigned char)(room[q] - di);
    cnt_r[q]++;
    if (room[q] > 0 && cnt_r[q] < RND_TRI_LOW) {
      nxt[q] = head[room[q]];
      head[room[q]] = (short)q;
    }
  }
  // emit: rounds in creation order, members in placement order (stable counting sort by round)
  {
    short start[ORD_BUCKET];
    for (int q = 0; q < n_rounds; ++q) start[q] = 0;
    for (int i = 0; i < n; ++i) start[rnd_of[i]]++;
    short acc = 0;
    for (int q = 0; q < n_rounds; ++q) { const short c = start[q]; start[q] = acc; acc += c; }
    for (int k = 0; k < n; ++k) {
      const int i = srt[k];
      const int pos = start[rnd_of[i]]++;
      order[t0 + pos] = (int)(t0 + i);
      degp[t0 + pos] = deg[t0 + i];
    }
  }
}
// segment starts by triangle id from the scan in layout order
__global__ void k_scatter_tptr(const int* __restrict__ tptrp, const int* __restrict__ order, int64_t nT, int* __restrict__ tptr) {
  const int64_t pos = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (pos < nT) tptr[order[pos]] = tptrp[pos];
  if (pos == nT) tptr[nT] = tptrp[nT];
}

struct PackCount {  // per-bucket counts, scanned together
  int rounds, longs, slots, splits, parts;
};
struct PackAdd {
  __host__ __device__ PackCount operator()(const PackCount& a, const PackCount& b) const {
    return PackCount{a.rounds + b.rounds, a.longs + b.longs, a.slots + b.slots, a.splits + b.splits, a.parts + b.parts};
  }
};
// sinfo[slot] = (touched index | SLOT_PART, unit offset of the part inside its triangle's row run, part ordinal
// or -1, the triangle's id).  A unit is a group of 3 columns: entry j of a split triangle is unit j + (j >= pos_d), the
// diagonal columns are unit pos_d.

// tfirst[i] = first directed entry of touched triangle i; tfirst[n_touched] = n_dir
__global__ void k_touched_first(const int* __restrict__ touched, const int* __restrict__ n_touched_dev,
                                const int* __restrict__ tptr, int64_t nT, int* __restrict__ tfirst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n_touched = *n_touched_dev;  // still on the device: the grid covers its bound
  if (i < n_touched) tfirst[i] = tptr[touched[i]];
  if (i == n_touched) tfirst[i] = tptr[nT];  // = number of directed entries
}

// Long triangles (more than RND_MAX_ENT partners), one warp each: sorts the segment by (partner, side)
// and decides whether the triangle can be SPLIT into parts.  It can when its three rows are exclusive and
// the vertex-id intervals [min, max] of its partners (in sorted order) and of the triangle itself are
// pairwise disjoint and ascending: the sorted columns of the row are then the partners' (sorted) triples
// one after the other, with the triangle's own triple in between at unit pos_d = number of partners
// below it -- so any run of consecutive entries owns a CONTIGUOUS piece of every row run, and the column
// ranks need no counting.  (Always true in a soup, where a triangle's vertex ids are 3t, 3t+1, 3t+2.)
//   tsplit[ti] = pos_d, or -1 (not splittable: k_tri_symbolic + the long assembly kernels)
__device__ __forceinline__ int min3i(int a, int b, int c) { return min(a, min(b, c)); }
__device__ __forceinline__ int max3i(int a, int b, int c) { return max(a, max(b, c)); }

__global__ void __launch_bounds__(32 * SYM_WARPS)
k_long_prep(const int* __restrict__ tris, const int* __restrict__ touched, const int* __restrict__ n_touched_dev,
            const int* __restrict__ tfirst, const uint2* __restrict__ ent, const int* __restrict__ vcnt,
            int force_general, int* partner, uint16_t* dvals, int* __restrict__ tsplit) {
  __shared__ unsigned long long s_key[SYM_WARPS][SYM_LMAX / 2];
  constexpr unsigned FULL = 0xffffffffu;
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int64_t n_touched = *n_touched_dev;
  const int64_t stride = (int64_t)gridDim.x * SYM_WARPS * 32;
  for (int64_t base = ((int64_t)blockIdx.x * SYM_WARPS + w) * 32; base < n_touched; base += stride) {
    const int64_t mine = base + l;
    const int dmine = (mine < n_touched) ? __ldg(tfirst + mine + 1) - __ldg(tfirst + mine) : 0;
    unsigned todo = __ballot_sync(FULL, dmine > RND_MAX_ENT);
    while (todo) {
      const int b = __ffs(todo) - 1;
      todo &= todo - 1;
      const int64_t ti = base + b;
      const int s = __ldg(touched + ti);
      const int e0 = __ldg(tfirst + ti), deg = __ldg(tfirst + ti + 1) - e0;
      warp_sort_segment(ent + e0, deg, s_key[w], SYM_LMAX / 2, partner + e0, dvals + e0, l);
      int own[3];
      load3i(tris + 3 * (int64_t)s, own);
      const int mn_s = min3i(own[0], own[1], own[2]), mx_s = max3i(own[0], own[1], own[2]);
      bool ok = !force_general && __ldg(vcnt + own[0]) == 1 && __ldg(vcnt + own[1]) == 1 && __ldg(vcnt + own[2]) == 1;
      int pos = 0;
      for (int j = l; j < deg; j += 32) {
        int cv[3];
        load3i(tris + 3 * (int64_t)partner[e0 + j], cv);
        const int mn = min3i(cv[0], cv[1], cv[2]), mx = max3i(cv[0], cv[1], cv[2]);
        if (j + 1 < deg) {
          int nv[3];
          load3i(tris + 3 * (int64_t)partner[e0 + j + 1], nv);
          ok = ok && (mx < min3i(nv[0], nv[1], nv[2]));
        }
        ok = ok && ((mx < mn_s) || (mx_s < mn));
        pos += (mx < mn_s) ? 1 : 0;
      }
      ok = __all_sync(FULL, ok);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) pos += __shfl_xor_sync(FULL, pos, o);
      if (l == 0) tsplit[ti] = ok ? pos : -1;
      __syncwarp();  // s_key is reused by the next triangle
    }
  }
}

// FILL = false: bucket_cnt[b] = counts of bucket b.
// FILL = true : round descriptors (first entry, entries, first slot, slots), slot tables, the list of
//               long (unsplittable) rounds and the list of split triangles, at the offsets bucket_off[b].
template <bool FILL>
__global__ void k_chunk_pack(const int* __restrict__ touched, const int* __restrict__ tfirst, const int* __restrict__ n_touched_dev,
                             const int* __restrict__ tsplit, PackCount* __restrict__ bucket_cnt,
                             const PackCount* __restrict__ bucket_off, int4* __restrict__ rdesc,
                             int* __restrict__ long_list, int* __restrict__ sfirst, int4* __restrict__ sinfo,
                             int4* __restrict__ split_list) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n_touched = *n_touched_dev;  // still on the device: the grid covers its bound
  const int64_t n_buckets = (n_touched + CHK_BUCKET - 1) / CHK_BUCKET;
  if (b >= n_buckets) return;             // the counts of the buckets beyond stay zero
  const int64_t i0 = b * CHK_BUCKET, i1 = min(i0 + (int64_t)CHK_BUCKET, n_touched);
  const int max_tri = round_tri_limit((int64_t)tfirst[n_touched], n_touched);
  PackCount base = PackCount{0, 0, 0, 0, 0};
  if (FILL) base = bucket_off[b];
  int nch = 0, nlong = 0, nslot = 0, nsplit = 0, npart = 0, ent = 0, tri = 0;
  int e_i = tfirst[i0];
  int r_e0 = e_i, r_s0 = 0;               // the open round: first entry, first slot (relative to the bucket)
  auto close_round = [&](int e_end) {
    if (FILL && nch > 0) rdesc[base.rounds + nch - 1] = make_int4(r_e0, e_end - r_e0, base.slots + r_s0, nslot - r_s0);
  };
  auto open_round = [&](int e_begin) {
    close_round(e_begin);
    r_e0 = e_begin;
    r_s0 = nslot;
    ++nch;
    ent = 0;
    tri = 0;
  };
  auto add_slot = [&](int e_begin, int cnt, int ti_flag, int u0, int pidx) {
    if (FILL) {
      sfirst[base.slots + nslot] = e_begin;
      sinfo[base.slots + nslot] = make_int4(ti_flag, u0, pidx, touched[ti_flag & ~SLOT_PART]);
    }
    ++nslot;
    ent += cnt;
    tri += 1;
  };
  for (int64_t i = i0; i < i1; ++i) {
    const int e_next = tfirst[i + 1];
    const int d = e_next - e_i;
    if (d <= RND_MAX_ENT) {
      if (tri == 0 || ent + d > RND_MAX_ENT || tri + 1 > max_tri) open_round(e_i);
      add_slot(e_i, d, (int)i, 0, -1);
    } else {
      const int sp = tsplit[i];
      if (sp < 0) {  // a round of its own
        open_round(e_i);
        if (FILL) long_list[base.longs + nlong] = base.rounds + nch - 1;
        ++nlong;
        add_slot(e_i, d, (int)i, 0, -1);
        tri = max_tri;  // closes the round: the next slot opens a new one
      } else {
        const int first_slot = nslot;
        if (FILL) split_list[base.splits + nsplit] = make_int4(base.slots + nslot, 0, (int)i, base.parts + npart);
#pragma unroll 1
        for (int seg = 0; seg < 2; ++seg) {  // entries below / above the diagonal columns
          int j = seg ? sp : 0;
          const int j1 = seg ? d : sp;
          while (j < j1) {
            if (tri == 0 || ent >= RND_MAX_ENT || tri + 1 > max_tri) open_round(e_i + j);
            const int take = min(j1 - j, RND_MAX_ENT - ent);
            add_slot(e_i + j, take, (int)i | SLOT_PART, j + seg, base.parts + npart);
            ++npart;
            j += take;
          }
        }
        if (FILL) split_list[base.splits + nsplit].y = nslot - first_slot;
        ++nsplit;
      }
    }
    e_i = e_next;
  }
  close_round(e_i);
  if (FILL && b == n_buckets - 1) sfirst[base.slots + nslot] = e_i;  // sentinel: number of directed entries
  if (!FILL) bucket_cnt[b] = PackCount{nch, nlong, nslot, nsplit, npart};
}

// vertex -> slot incidence keys: key = vertex, payload = 3 slot + m.  Only the slot that holds a triangle's
// summed gradient / H.p partial takes part: whole slots and the FIRST part of a split triangle
// (k_split_finish adds the other parts into it); the others get the key nV, which sorts past every vertex.
__global__ void k_emit_vslots(const int* __restrict__ tris, const int* __restrict__ touched, int64_t n_slots,
                              const int4* __restrict__ sinfo, const int* __restrict__ tsplit, int64_t nV,
                              uint64_t* __restrict__ vkeys, uint32_t* __restrict__ vvals) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 3 * n_slots) return;
  const int64_t sl = i / 3;
  const int m = (int)(i - 3 * sl);
  const int4 si = sinfo[sl];
  const int ti = si.x & ~SLOT_PART;
  bool holder = true;
  if (si.x & SLOT_PART) holder = (si.y == 0) || (si.y == 1 && tsplit[ti] == 0);
  vkeys[i] = holder ? (uint64_t)(uint32_t)tris[3 * (int64_t)touched[ti] + m] : (uint64_t)nV;
  vvals[i] = (uint32_t)i;
}

// ------------------------------------------------------------------------------------------ K4
// Triangle-centric numeric phase.  One LANE per directed entry e = (source s -> partner t); one
// WARP per round (whole triangles, <= 32 entries), warps fully independent (no __syncthreads, no
// atomics).  The pair is always evaluated in its canonical order (T_a = pairs[k,0]) so that both
// directed copies of a pair compute bit-identical J and take the same FILTER decision.
//
// k_assemble_tile (energy + gradient + Hessian blocks).  Row m of triangle s (vertex p_m) owns ONE
// contiguous run of L = 3 (deg + 1) blocks in its destination (vals for exclusive rows, the merge
// workspace otherwise).  For m = 0, 1, 2 the warp builds the runs of all its triangles for that
// row in a shared-memory tile laid out exactly like global memory,
//   off-diagonal block (p_m, q_n), one contribution:  a g0_q^T + b g1_q^T,
//       a = c00 g0_pm + c01 g1_pm,  b = c01 g0_pm + c11 g1_pm            (M symmetric),
//   diagonal-row blocks (p_m, p_n) and the gradient of p_m: staged per entry, summed over the
//       triangle's entries with lane = component in entry order (deterministic),
// and hands every run to the TMA engine (cp.async.bulk shared -> global, 16-byte aligned body;
// the <= 15 unaligned head / tail bytes by plain stores).  Address generation and full-line
// writes are the copy engine's; the SM issues ~60 shared stores per entry and row.
//
// The grid is PERSISTENT (8 one-warp CTAs per SM: the kernel needs 255 registers); a warp walks
// rounds c, c + G, c + 2G, ... with every gather of a round off its critical path:
//   descriptor three rounds ahead, vertex ids two, payload / ranks / row destinations one (requested
//   after the register peak of the derivative code); the positions of round c + G are pulled into
//   L2 at the top of round c (prefetch.global.L2: no registers, no scoreboard) and loaded into
//   registers at the end of round c, when J is dead.
// cp.async (LDGSTS) is NOT used for the positions: cp.async.wait_group and
// cp.async.bulk.wait_group.read both compile to DEPBAR on scoreboard SB0, so every wait for the
// copy engine would also wait for the gathers in flight (measured: +40 % kernel time).
// The staging area of the diagonal / gradient products aliases the row tile (12.5 KB of shared
// memory per warp); the measured limiter is the L1 data pipe (shared-memory wavefronts of staging,
// tile writes and the engine's reads: 62 % busy), not HBM (49 %) or instruction issue (31 %).
// C = the arithmetic type of the derivative code: double in every kernel of the hot path (reading A12; the
// fp32 instantiation was measured -- it misses the 1e-4 gradient bar on config 3 and buys 14 % on K4 -- and
// is not used); TT_HESS_EXACT instantiates it with second-order information (tt_exact.cuh).
template <typename C>
struct Entry {
  C g0[18], g1[18];        // own triangle's 9 DOF first, partner's 9 after; vertices in RECORDED order (k, p, q)
  ttg::Coefs<C> cf;
  C en;                    // Eq. 2 energy if this is the canonical copy (side 0), else 0
  int po[3], pp[3];        // recorded order -> index 0..2 inside the own / partner triangle
};

template <typename T>
struct AsmParams {
  const T* pos;
  const uint16_t* dvals;    // side | recorded config << 1 (ttg::pair_config)
  const int* everts;        // [2A][6] vertex ids of the canonical pair, both triangles in recorded order
  const int4* rdesc;        // [n_chunks] round descriptor: first entry, entries, first touched index, triangles
  const int* tfirst;        // [n_slots+1] first entry of every slot
  const int* long_list;     // [n_long] round ids of the long triangles
  const int* erank;         // [2A][3]
  const int* drank;         // [n_slots][3]; a part: [0] = -1 - part ordinal
  const int64_t* rowbase;   // [3 n_slots]
  T* vals;                  // final BSR values
  T* tvals;                 // merge workspace values
  T* tslot;                 // [3 n_slots][3] per-slot gradient (K4) or H.p (K6) partials
  double* chunk_energy;     // [n_chunks]
  double* dpart;            // [n_parts][NDIAG] diagonal partial sums of the parts of split triangles
  const T* pvec;            // K6: p [nV,3]
  int64_t n_chunks;
  int64_t n_long;
  int hess_mode;
  double sigma;
};

// ---- round-based symbolic kernels (one warp per round, lane = directed entry) -------------------
// Same results as k_tri_symbolic / k_ent_verts / k_fill_rows, which remain for LONG triangles (more
// than RND_MAX_ENT partners): a warp owns a round of whole triangles, so every gather is one lane
// wide and 32 entries deep instead of one warp per (on average 5-entry) triangle.
constexpr int RSYM_WARPS = 4;


// Segment sort by (partner, side), column ranks (erank / drank), duplicate detection, exclusive rows,
// row lengths and the per-entry vertex ids (everts) of every non-long round.  Persistent grid: a warp
// walks rounds c, c + G, ... (the number of rounds is still on the device when this kernel is enqueued).
// Lane = slot for the per-slot work, lane = directed entry for the per-entry work.
//   whole slot: its segment is sorted here.  Ranks: if the vertex-id intervals of the (sorted) partners and
//               of the triangle are pairwise disjoint and ascending, the rank of column n of entry j is
//               3 (j + [j >= pos_d]) + (rank of the vertex inside its own triple) -- no counting; if any
//               slot of the round fails that test the round falls back to counting (all pairs).
//   part slot : sorted and tested by k_long_prep; ranks are relative to the part's own run:
//               3 i + local rank, i = position inside the part.
__global__ void __launch_bounds__(32 * RSYM_WARPS)
k_round_symbolic(const int* __restrict__ tris, const int* __restrict__ touched, const int4* __restrict__ rdesc,
                 const int* __restrict__ n_chunks_dev, const int* __restrict__ tfirst, const int* __restrict__ sfirst,
                 const int4* __restrict__ sinfo, const int* __restrict__ tsplit, const uint2* __restrict__ ent,
                 const int* __restrict__ vcnt, int force_general, int* partner /*in (parts) / out*/,
                 uint16_t* dvals /*in (parts) / out*/, int* __restrict__ erank, int* __restrict__ drank,
                 int* __restrict__ rowlen, int64_t* __restrict__ tlen, uint8_t* __restrict__ slot_excl,
                 int* __restrict__ everts, int* __restrict__ vslot1) {
  __shared__ int s_cand[RSYM_WARPS][3 * RND_MAX_ENT];  // partner vertex ids of entry i at [3 i + n]
  __shared__ int s_own[RSYM_WARPS][3 * RND_MAX_TRI];   // own vertex ids of slot tt at [3 tt + n]
  __shared__ int s_first[RSYM_WARPS][RND_MAX_TRI + 1];
  __shared__ int s_dup[RSYM_WARPS][RND_MAX_TRI];
  __shared__ int s_dacc[RSYM_WARPS][3 * RND_MAX_TRI];  // per own column: partner columns below it
  __shared__ int s_rsum[RSYM_WARPS][RND_MAX_TRI];      // per slot: sum of the partner columns' ranks
  __shared__ int s_posd[RSYM_WARPS][RND_MAX_TRI];      // per slot: entries below the diagonal columns (fast path)
  __shared__ unsigned long long s_key[RSYM_WARPS][RND_MAX_ENT];
  __shared__ uint2 s_ent[RSYM_WARPS][RND_MAX_ENT];
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int* cand = s_cand[warp];
  int* own = s_own[warp];
  int* first = s_first[warp];
  int* dupf = s_dup[warp];
  int* dacc = s_dacc[warp];
  int* rsum = s_rsum[warp];
  int* posd = s_posd[warp];
  unsigned long long* skey = s_key[warp];
  uint2* sent = s_ent[warp];
  const int64_t n_chunks = *n_chunks_dev;
  const int64_t stride = (int64_t)gridDim.x * RSYM_WARPS;
  // The head of a round is a chain of dependent loads (descriptor -> slot table -> vertex ids); the descriptor
  // and the slot rows of the NEXT round are requested while this one is worked on, so that a round starts
  // one load (the triangles' vertex ids) away from its data instead of three.
  const int4 dzero = make_int4(0, 0, 0, 0);
  int64_t c = (int64_t)blockIdx.x * RSYM_WARPS + warp;
  int4 d = (c < n_chunks) ? __ldg(rdesc + c) : dzero;
  int4 psi = make_int4(0, 0, -1, 0);
  int pf = 0, pl = 0;
  auto fetch_slots = [&](const int4 dd) {  // slot rows of a round (lane = slot); nothing for a long round
    psi = make_int4(0, 0, -1, 0);
    pf = pl = 0;
    if (dd.y <= RND_MAX_ENT && lane < dd.w) {
      psi = __ldg(sinfo + dd.z + lane);
      pf = __ldg(sfirst + dd.z + lane);
      pl = __ldg(sfirst + dd.z + lane + 1);
    }
  };
  fetch_slots(d);
  for (; c < n_chunks; c += stride) {
    const int4 d_next = (c + stride < n_chunks) ? __ldg(rdesc + c + stride) : dzero;
    const int e_lo = d.x, nent = d.y, s_lo = d.z, nsl = d.w;
    if (nent > RND_MAX_ENT) {  // long triangle: k_tri_symbolic
      d = d_next;
      fetch_slots(d);
      continue;
    }
    // ---- lane = slot ----
    int f = 0, l = 0, ov[3] = {0, 0, 0};
    const int4 si = psi;
    if (lane < nsl) {
      f = pf - e_lo;
      l = pl - e_lo;
      load3i(tris + 3 * (int64_t)si.w, ov);
#pragma unroll
      for (int n = 0; n < 3; ++n) own[3 * lane + n] = ov[n];
      first[lane] = f;
      dupf[lane] = 0;
      rsum[lane] = 0;
      posd[lane] = 0;
      dacc[3 * lane] = dacc[3 * lane + 1] = dacc[3 * lane + 2] = 0;
    }
    const bool slot_is_part = (si.x & SLOT_PART) != 0;
    if (lane == 0) first[nsl] = nent;
    const unsigned heads = __reduce_or_sync(FULL, (lane < nsl) ? (1u << f) : 0u);
    const unsigned partmask = __ballot_sync(FULL, lane < nsl && slot_is_part);  // bit tt: slot tt is a part
    // ---- lane = entry ----
    const bool valid = lane < nent;
    const int my_ti = __popc(heads & (0xffffffffu >> (31 - lane))) - 1;
    const bool in_part = valid && ((partmask >> my_ti) & 1u);
    uint2 me = make_uint2(0u, 0u);
    if (valid) {
      const int64_t e = (int64_t)e_lo + lane;
      if (in_part) me = make_uint2((unsigned)partner[e], (unsigned)dvals[e]);  // sorted by k_long_prep
      else me = __ldg(ent + e);                                                  // as the counting sort left them
    }
    const unsigned long long key = entry_key(me);
    skey[lane] = key;
    __syncwarp();
    int myf = 0, deg = 0;
    int mo[3] = {0, 0, 0};  // own vertex ids of the entry's triangle
    if (valid) {
      myf = first[my_ti];
      deg = first[my_ti + 1] - myf;
#pragma unroll
      for (int n = 0; n < 3; ++n) mo[n] = own[3 * my_ti + n];
    }
    const int sortdeg = in_part ? 0 : deg;
    const int maxdeg = __reduce_max_sync(FULL, sortdeg);
    // ---- sort every whole slot's segment by (partner, side): position = number of keys below (ties by lane) ----
    {
      int pos = in_part ? lane - myf : 0;
      for (int k = 0; k < maxdeg; ++k) {
        if (k < sortdeg) {
          const unsigned long long kx = skey[myf + k];
          pos += (kx < key) || (kx == key && myf + k < lane);
        }
      }
      if (valid) sent[myf + pos] = me;
      __syncwarp();
      if (valid) me = sent[lane];
    }
    int cv[3] = {0, 0, 0};
    const unsigned pay = me.y;
    if (valid) {
      const int64_t e = (int64_t)e_lo + lane;
      if (!in_part) {
        partner[e] = (int)me.x;
        dvals[e] = (uint16_t)me.y;
      }
      load3i(tris + 3 * (int64_t)me.x, cv);
#pragma unroll
      for (int n = 0; n < 3; ++n) cand[3 * lane + n] = cv[n];
    }
    // ---- fast path test: disjoint ascending vertex-id intervals ----
    const int mn = min3i(cv[0], cv[1], cv[2]), mx = max3i(cv[0], cv[1], cv[2]);
    const int mn_s = min3i(mo[0], mo[1], mo[2]), mx_s = max3i(mo[0], mo[1], mo[2]);
    const int mn_next = __shfl_down_sync(FULL, mn, 1);
    const bool last_of_slot = valid && (lane == myf + deg - 1);
    bool ordered = true;
    if (valid && !in_part) ordered = (last_of_slot || mx < mn_next) && ((mx < mn_s) || (mx_s < mn));
    const bool fast = __all_sync(FULL, ordered);
    const bool below = valid && (mx < mn_s);
    const unsigned below_mask = __ballot_sync(FULL, below);
    __syncwarp();
    const int lr0 = (cv[1] < cv[0]) + (cv[2] < cv[0]), lr1 = (cv[0] < cv[1]) + (cv[2] < cv[1]), lr2 = (cv[0] < cv[2]) + (cv[1] < cv[2]);
    int r[3] = {0, 0, 0};
    int dr[3] = {0, 0, 0};
    if (fast) {
      if (valid) {
        const unsigned seg = (deg >= 32) ? 0xffffffffu : (((1u << deg) - 1u) << myf);
        const int pd = __popc(below_mask & seg);       // entries of my slot below the diagonal columns
        const int j = lane - myf;
        const int unit = in_part ? j : j + (j >= pd ? 1 : 0);
        r[0] = 3 * unit + lr0;
        r[1] = 3 * unit + lr1;
        r[2] = 3 * unit + lr2;
        if (j == 0) posd[my_ti] = pd;
      }
      __syncwarp();
      if (lane < nsl) {
        const int pd = (l > f) ? posd[lane] : 0;
#pragma unroll
        for (int n = 0; n < 3; ++n) dr[n] = 3 * pd + (ov[0] < ov[n]) + (ov[1] < ov[n]) + (ov[2] < ov[n]);
      }
    } else {
      // Rank of a column = number of smaller columns among the triangle's L = 3 (deg + 1) candidates.
      // Duplicates: the ranks of L distinct values sum to L (L - 1) / 2 and every tied pair lowers the sum
      // by one, so one integer per triangle (shared-memory atomics: the RESULT is order independent)
      // replaces all equality counting.  The diagonal columns are ranked by the entries' lanes too:
      // each adds how many of its three columns lie below each own column.  (Part slots keep their own.)
      const int cdeg = in_part ? 0 : deg;
      const int cmax = __reduce_max_sync(FULL, cdeg);
      for (int k = 0; k < cmax; ++k) {
        if (k < cdeg) {
          const int* o = cand + 3 * (myf + k);
          const int o0 = o[0], o1 = o[1], o2 = o[2];
#pragma unroll
          for (int n = 0; n < 3; ++n) r[n] += (o0 < cv[n]) + (o1 < cv[n]) + (o2 < cv[n]);
        }
      }
      if (valid && !in_part) {
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          r[n] += (mo[0] < cv[n]) + (mo[1] < cv[n]) + (mo[2] < cv[n]);
          atomicAdd(&dacc[3 * my_ti + n], (cv[0] < mo[n]) + (cv[1] < mo[n]) + (cv[2] < mo[n]));
        }
        atomicAdd(&rsum[my_ti], r[0] + r[1] + r[2]);
      }
      if (in_part) {
        const int j = lane - myf;
        r[0] = 3 * j + lr0;
        r[1] = 3 * j + lr1;
        r[2] = 3 * j + lr2;
      }
      __syncwarp();
      if (lane < nsl && !slot_is_part) {
        int tot = rsum[lane];
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          dr[n] = dacc[3 * lane + n] + (ov[0] < ov[n]) + (ov[1] < ov[n]) + (ov[2] < ov[n]);
          tot += dr[n];
        }
        const int L = 3 * (l - f + 1);
        dupf[lane] = (2 * tot != L * (L - 1)) ? 1 : 0;
      }
      __syncwarp();
    }
    if (valid) {
      const int64_t e = (int64_t)e_lo + lane;
      const bool nodup = dupf[my_ti] == 0;
      const int j = lane - myf;
#pragma unroll
      for (int n = 0; n < 3; ++n) erank[3 * e + n] = nodup ? r[n] : 3 * j + n;
      // vertex ids of the canonical pair, both triangles in recorded (k, p, q) order
      const bool side = (pay & 1u) != 0u;
      const unsigned ca = (pay >> 1) & 63u, cb = (pay >> 7) & 63u;
      const int ka = (int)(ca & 3u), pa = (int)((ca >> 2) & 3u), kb = (int)(cb & 3u), pb = (int)((cb >> 2) & 3u);
      const int a0 = side ? cv[0] : mo[0], a1 = side ? cv[1] : mo[1], a2 = side ? cv[2] : mo[2];
      const int b0 = side ? mo[0] : cv[0], b1 = side ? mo[1] : cv[1], b2 = side ? mo[2] : cv[2];
      int2* o = reinterpret_cast<int2*>(everts + 6 * e);
      o[0] = make_int2(pick3(ka, a0, a1, a2), pick3(pa, a0, a1, a2));
      o[1] = make_int2(pick3(3 - ka - pa, a0, a1, a2), pick3(kb, b0, b1, b2));
      o[2] = make_int2(pick3(pb, b0, b1, b2), pick3(3 - kb - pb, b0, b1, b2));
    }
    if (lane < nsl) {
      const int64_t sl = (int64_t)s_lo + lane;
      if (!slot_is_part) {
        const bool nodup = dupf[lane] == 0;
        const int dg = l - f, L = 3 * (dg + 1);
#pragma unroll
        for (int n = 0; n < 3; ++n) drank[3 * sl + n] = nodup ? dr[n] : 3 * dg + n;
#pragma unroll
        for (int m = 0; m < 3; ++m) {
          const bool single = __ldg(vcnt + ov[m]) == 1;
          const bool excl = nodup && !force_general && single;
          if (single) vslot1[ov[m]] = (int)(3 * sl + m);  // the vertex's only slot (k_gather3)
          slot_excl[3 * sl + m] = excl ? 1 : 0;
          tlen[3 * sl + m] = excl ? 0 : L;
          if (excl) rowlen[ov[m]] = L;
        }
      } else {  // part of a split triangle: exclusive rows by construction; the triangle's first part owns its rows
        const int ti = si.x & ~SLOT_PART;
        const int pd = __ldg(tsplit + ti);
        const bool first_part = (si.y == 0) || (si.y == 1 && pd == 0);
        drank[3 * sl] = -1 - si.z;   // part ordinal (diagonal partial sums: k_split_finish)
        drank[3 * sl + 1] = 0;
        drank[3 * sl + 2] = 0;
        const int L = 3 * (__ldg(tfirst + ti + 1) - __ldg(tfirst + ti) + 1);
#pragma unroll
        for (int m = 0; m < 3; ++m) {
          slot_excl[3 * sl + m] = 1;
          tlen[3 * sl + m] = 0;
          if (first_part) {
            vslot1[ov[m]] = (int)(3 * sl + m);
            rowlen[ov[m]] = L;
          }
        }
      }
    }
    __syncwarp();  // shared memory is reused by the next round
    d = d_next;
    fetch_slots(d);
  }
}

// Column indices of the exclusive rows + row bases of every non-long round (after the rowptr scan).
// The three rows of a slot have the SAME column run: it is built once in shared memory (ranks are
// positions in the run) and written out three times with consecutive lanes on consecutive addresses,
// instead of nine scattered 4-byte stores per entry.  A whole slot's run has deg + 1 units of 3 columns
// (the last unit in the staging area is the diagonal's); a part's run has one unit per entry and starts
// 3 u0 blocks into the triangle's rows; the first part of a split triangle also writes the diagonal columns.
__global__ void __launch_bounds__(32 * RSYM_WARPS)
k_round_fill(const int* __restrict__ tris, const int* __restrict__ touched, const int4* __restrict__ rdesc,
             int64_t n_chunks, const int* __restrict__ sfirst, const int4* __restrict__ sinfo,
             const int* __restrict__ tsplit, const int* __restrict__ partner,
             const int* __restrict__ erank, const int* __restrict__ drank, const int64_t* __restrict__ toff,
             const uint8_t* __restrict__ slot_excl, const int* __restrict__ rowptr,
             int64_t* __restrict__ rowbase, int* __restrict__ colind) {
  constexpr int UNITS = RND_MAX_ENT + RND_MAX_TRI;
  __shared__ int s_rp[RSYM_WARPS][3 * RND_MAX_TRI];       // first block of the run of row m of slot tt, or -1
  __shared__ int s_ci[RSYM_WARPS][3 * UNITS];             // column runs of the round's slots, back to back
  __shared__ int s_ub[RSYM_WARPS][RND_MAX_TRI];           // first unit of slot tt in s_ci
  __shared__ unsigned char s_utt[RSYM_WARPS][UNITS];      // unit -> slot
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t c = (int64_t)blockIdx.x * RSYM_WARPS + warp;
  if (c >= n_chunks) return;
  const int4 d = __ldg(rdesc + c);
  const int e_lo = d.x, nent = d.y, s_lo = d.z, nsl = d.w;
  if (nent > RND_MAX_ENT) return;  // long triangle: k_fill_rows
  int* rps = s_rp[warp];
  int* ci = s_ci[warp];
  int* ubase = s_ub[warp];
  unsigned char* utt = s_utt[warp];
  // entry lanes: partner columns and ranks (independent of the slot lanes' loads)
  int cv[3] = {0, 0, 0}, er[3] = {0, 0, 0};
  if (lane < nent) {
    const int64_t e = (int64_t)e_lo + lane;
    const int t = __ldg(partner + e);
    load3i(tris + 3 * (int64_t)t, cv);
    load3i(erank + 3 * e, er);
  }
  // slot lanes
  int f = 0, l = 0;
  int4 si = make_int4(0, 0, -1, 0);
  if (lane < nsl) {
    si = __ldg(sinfo + s_lo + lane);
    f = __ldg(sfirst + s_lo + lane) - e_lo;
    l = __ldg(sfirst + s_lo + lane + 1) - e_lo;
  }
  const bool is_part = (si.x & SLOT_PART) != 0;
  const unsigned wholemask = __ballot_sync(FULL, lane < nsl && !is_part);
  const int ub = f + __popc(wholemask & ((1u << lane) - 1u));   // every whole slot before adds one (diagonal) unit
  const unsigned heads = __reduce_or_sync(FULL, (lane < nsl) ? (1u << f) : 0u);
  const int my_ti = __popc(heads & (0xffffffffu >> (31 - lane))) - 1;
  if (lane < nsl) {
    const int64_t sl = (int64_t)s_lo + lane;
    const int ti = si.x & ~SLOT_PART;
    int ov[3];
    load3i(tris + 3 * (int64_t)si.w, ov);  // sinfo carries the triangle's id: one load less in the chain
    ubase[lane] = ub;
    if (!is_part) {
      utt[ub + (l - f)] = (unsigned char)lane;  // the diagonal's unit closes the run
#pragma unroll
      for (int n = 0; n < 3; ++n) ci[3 * ub + __ldg(drank + 3 * sl + n)] = ov[n];
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const bool excl = slot_excl[3 * sl + m] != 0;
        const int rp = excl ? __ldg(rowptr + ov[m]) : -1;
        rps[3 * lane + m] = rp;
        rowbase[3 * sl + m] = excl ? (int64_t)rp : -(toff[3 * sl + m] + 1);
      }
    } else {
      const int pd = __ldg(tsplit + ti);
      const bool first_part = (si.y == 0) || (si.y == 1 && pd == 0);
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const int row0 = __ldg(rowptr + ov[m]);
        const int rp = row0 + 3 * si.y;
        rps[3 * lane + m] = rp;
        rowbase[3 * sl + m] = (int64_t)rp;
        if (first_part) {
#pragma unroll
          for (int n = 0; n < 3; ++n) colind[row0 + 3 * pd + (ov[0] < ov[n]) + (ov[1] < ov[n]) + (ov[2] < ov[n])] = ov[n];
        }
      }
    }
  }
  __syncwarp();
  // first entry of my slot, by shuffle from the slot lane
  const int myf = __shfl_sync(FULL, f, my_ti < 0 ? 0 : my_ti);
  if (lane < nent) {
    const int u = ubase[my_ti];
    utt[u + (lane - myf)] = (unsigned char)my_ti;
    const int base = 3 * u;
#pragma unroll
    for (int n = 0; n < 3; ++n) ci[base + er[n]] = cv[n];
  }
  __syncwarp();
  const int total = 3 * (nent + __popc(wholemask));
  for (int idx = lane; idx < total; idx += 32) {
    const int tt = utt[idx / 3];
    const int off = idx - 3 * ubase[tt];
    const int v = ci[idx];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      const int rp = rps[3 * tt + m];
      if (rp >= 0) colind[rp + off] = v;
    }
  }
}

template <typename T, typename C>
__device__ __forceinline__ void load_pos18(const T* __restrict__ pos, const int (&ids)[6], C (&x)[18]) {
#pragma unroll
  for (int v = 0; v < 6; ++v) {
    const T* p = pos + 3 * (int64_t)ids[v];
    x[3 * v] = (C)__ldg(p);
    x[3 * v + 1] = (C)__ldg(p + 1);
    x[3 * v + 2] = (C)__ldg(p + 2);
  }
}

// J by the straight-line code on gathered positions x = [a_k, a_p, a_q, b_k, b_p, b_q] (raw),
// coefficients, energy; swaps halves so that "own" is first.
template <typename C, bool PROJ = true>
__device__ __forceinline__ void eval_core(const C (&x)[18], unsigned pay, C sigma, int hess_mode, Entry<C>& E) {
  using V = ttg::v3<C>;
  const bool side = (pay & 1u) != 0u;
  const unsigned ca = (pay >> 1) & 63u, cb = (pay >> 7) & 63u;
  int pa[3], pb[3];
  pa[0] = (int)(ca & 3u); pa[1] = (int)((ca >> 2) & 3u); pa[2] = 3 - pa[0] - pa[1];
  pb[0] = (int)(cb & 3u); pb[1] = (int)((cb >> 2) & 3u); pb[2] = 3 - pb[0] - pb[1];
  // local frame: translate by -a_k (kills the cancellation in D.E, keeps fp32 inputs well scaled)
  const V o = ttg::mk<C>(x[0], x[1], x[2]);
  const V ak = ttg::mk<C>(C(0), C(0), C(0));
  const V ap = ttg::mk<C>(x[3], x[4], x[5]) - o, aq = ttg::mk<C>(x[6], x[7], x[8]) - o;
  const V bk = ttg::mk<C>(x[9], x[10], x[11]) - o, bp = ttg::mk<C>(x[12], x[13], x[14]) - o, bq = ttg::mk<C>(x[15], x[16], x[17]) - o;
  C tc0, tc1;
  ttg::pair_derivs_recorded<C>(ak, ap, aq, bk, bp, bq, sigma, ca >> 4, cb >> 4, tc0, tc1, E.g0, E.g1);
  E.cf = ttg::pair_coefs<C, PROJ>(tc0, tc1, E.g0, E.g1, hess_mode);
  const C tt = tc0 * tc1;
  E.en = side ? C(0) : tt * tt;  // Eq. 2, counted once per pair
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    E.po[m] = side ? pb[m] : pa[m];
    E.pp[m] = side ? pa[m] : pb[m];
  }
  if (side) {
#pragma unroll
    for (int i = 0; i < 9; ++i) {
      const C t0 = E.g0[i]; E.g0[i] = E.g0[9 + i]; E.g0[9 + i] = t0;
      const C t1 = E.g1[i]; E.g1[i] = E.g1[9 + i]; E.g1[9 + i] = t1;
    }
  }
}

// Brings the own half of J back to the triangle's own vertex order (selects on the recorded
// permutation: no shared-memory round trip, the L1 data pipe is the kernel's busiest unit), and the
// partner's block ranks into recorded order.
template <typename C>
__device__ __forceinline__ void unpermute_own(Entry<C>& E, int (&er)[3]) {
  C t0[9], t1[9];
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    t0[i] = E.g0[i];
    t1[i] = E.g1[i];
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {  // own vertex i = recorded position r with po[r] == i
    const bool p0 = E.po[0] == i, p1 = E.po[1] == i;
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
      E.g0[3 * i + cc] = p0 ? t0[cc] : (p1 ? t0[3 + cc] : t0[6 + cc]);
      E.g1[3 * i + cc] = p0 ? t1[cc] : (p1 ? t1[3 + cc] : t1[6 + cc]);
    }
  }
  const int e0 = er[0], e1 = er[1], e2 = er[2];
#pragma unroll
  for (int r = 0; r < 3; ++r) er[r] = (E.pp[r] == 0) ? e0 : ((E.pp[r] == 1) ? e1 : e2);
}

__device__ __forceinline__ void bulk_s2g(void* gdst, const void* ssrc, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
               "r"((uint32_t)__cvta_generic_to_shared(ssrc)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
template <int N>  // at most N of this thread's most recent groups may still be reading shared memory
__device__ __forceinline__ void bulk_wait_read_n() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- cp.async (LDGSTS): global -> shared gathers that hold no registers while in flight ---------
template <typename T>
__device__ __forceinline__ void cp_async_elem(T* sdst, const T* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(sdst);
  if (sizeof(T) == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

#ifndef TT_TILE_WARPS
#define TT_TILE_WARPS 1
#endif
#ifndef TT_TILE_MAXNREG
#define TT_TILE_MAXNREG 255               // 8 warps / SM.  Measured: 200 / 184 / 168 registers (10 / 11 / 12 warps) spill
#endif                                    // 400-700 bytes per thread and run 20-60 % slower (profiles/r1_step_breakdown.md)
#ifndef TT_RED_UNR
#define TT_RED_UNR 8                      // entries per triangle whose staged values are loaded up front
#endif
constexpr int RED_UNR = TT_RED_UNR;
#ifndef TT_RED_UNR1
#define TT_RED_UNR1 6                     // the same for the one-pass sums (four chains: fewer values each)
#endif
constexpr int RED_UNR1 = TT_RED_UNR1;
#ifndef TT_RED_UNR1_WIDE
#define TT_RED_UNR1_WIDE 3             // measured at 1 / 2 / 5 M pairs: 6 -> 0.374 / 0.629 / 1.234 ms, 4 -> 0.364 / 0.615 / 1.231, 3 -> 0.359 / 0.609 / 1.231, 2 -> 0.355 / 0.609 / 1.239
#endif
#ifndef TT_TILE_ONEPASS
#define TT_TILE_ONEPASS 1
#endif
#ifndef TT_TILE_NBUF
#define TT_TILE_NBUF 2                    // row tiles per warp: with two, a row is built while the copy engine reads the previous one
#endif
constexpr int TILE_WARPS = TT_TILE_WARPS; // warps per CTA (independent; a CTA is only a packaging unit)
constexpr int NDIAG = 45;                 // upper triangle of the symmetric 9x9 diagonal block, row-major packed
constexpr int NSTG = NDIAG + 9;           // + gradient of the three own vertices
constexpr int STG_PASS = NSTG / 2;        // the 54 per-entry values are staged in two passes of 27
constexpr int STG_STRIDE = STG_PASS;      // 27 doubles: odd, so lane = entry writes are conflict-free
constexpr int STG1_STRIDE = NSTG + 1;     // one-pass staging (all 54 values of an entry at once): 55 doubles, odd
constexpr int LONG_STRIDE = 31;           // k_assemble_long: 27 + 3 staged values per entry, odd stride

template <typename T, int MT>  // MT: slots per round this instantiation of K4 is built for
struct TileCfg {
  static constexpr int RUN_UNIT = 27 * (int)sizeof(T);  // bytes one entry (or the diagonal) adds to a row run
  static constexpr int TILE_BYTES = RUN_UNIT * (RND_MAX_ENT + MT) + 32 * MT;
  static constexpr int STAGE_BYTES = 32 * STG_STRIDE * (int)sizeof(double);
  // fp64 with 16 slots per round: two tiles per warp would not leave room for 8 warps per SM
  static constexpr int NBUF = (MT > RND_TRI_LOW && sizeof(T) == 8) ? 1 : TT_TILE_NBUF;
  // All 54 values of an entry are staged at once and summed in one loop (four independent chains instead of two, half
  // the shuffles and warp barriers; the 36 registers of the diagonal factors are dead before the sums start).  The
  // staging area spans the tile buffer(s), which are made large enough for it.
  static constexpr bool ONEPASS = (TT_TILE_ONEPASS != 0);
  static constexpr int STAGE1_PART = ((32 * STG1_STRIDE * (int)sizeof(double) / NBUF) + 15) & ~15;
  static constexpr int UNION0 = TILE_BYTES > STAGE_BYTES ? TILE_BYTES : STAGE_BYTES;
  static constexpr int UNION_BYTES = (ONEPASS && STAGE1_PART > UNION0) ? STAGE1_PART : UNION0;
  static_assert(UNION_BYTES % 16 == 0, "tile buffers must stay 16-byte aligned");
};

// Shared memory of one warp.  `tile` holds, in turn, (1) the per-entry staging area of the
// diagonal / gradient products and (2) the row tile the copy engine reads: the two never live at
// the same time (the per-triangle sums move to `dsum` in between).
template <typename T, int MT>
struct alignas(16) TileWarpSmem {
  unsigned char tile[TileCfg<T, MT>::NBUF * TileCfg<T, MT>::UNION_BYTES];
  double dsum[MT][NSTG];                  // per-triangle sums: 45 diagonal-block values + 9 gradient values
  int run_off[MT];                        // byte offset of the triangle's run in the tile (current row)
  int diag_off[MT][3];                    // byte offset of its diagonal block n in the tile (current row)
};
// Pulls the (at most two) 32-byte sectors of each of six vertices into L2.
template <typename T>
__device__ __forceinline__ void prefetch_pos_l2(const T* __restrict__ pos, const int (&ids)[6]) {
#pragma unroll
  for (int v = 0; v < 6; ++v) {
    const T* p = pos + 3 * (int64_t)ids[v];
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
    if ((reinterpret_cast<uintptr_t>(p) & 31) + 3 * sizeof(T) > 32)  // the vertex straddles two sectors
      asm volatile("prefetch.global.L2 [%0];" ::"l"(p + 2));
  }
}
struct alignas(16) LongWarpSmem {
  double stage[32 * LONG_STRIDE];
};

// Operands of a round that depend only on its descriptor.  Vertex ids travel two rounds ahead
// (their positions are requested one round ahead), everything else one round ahead.
struct RoundOps {
  unsigned pay;      // lane = entry
  int er[3];
  int e0, e1;        // lane = triangle
  int64_t rb[3];
  int dr[3];
};
__device__ __forceinline__ int round_entries(const int4 d) { return d.y > RND_MAX_ENT ? 0 : d.y; }  // long rounds: none here

template <typename T>
__device__ __forceinline__ void load_round_ids(const AsmParams<T>& P, const int4 d, int lane, int (&ids)[6]) {
#pragma unroll
  for (int i = 0; i < 6; ++i) ids[i] = 0;
  if (lane < round_entries(d)) {
    const int2* v = reinterpret_cast<const int2*>(P.everts + 6 * ((int64_t)d.x + lane));
    const int2 v0 = __ldg(v), v1 = __ldg(v + 1), v2 = __ldg(v + 2);
    ids[0] = v0.x; ids[1] = v0.y; ids[2] = v1.x; ids[3] = v1.y; ids[4] = v2.x; ids[5] = v2.y;
  }
}
template <typename T>
__device__ __forceinline__ void load_round_ops(const AsmParams<T>& P, const int4 d, int lane, RoundOps& R) {
  R.pay = 0u;
  R.er[0] = R.er[1] = R.er[2] = 0;
  R.e0 = R.e1 = 0;
  R.rb[0] = R.rb[1] = R.rb[2] = 0;
  R.dr[0] = R.dr[1] = R.dr[2] = 0;
  if (lane < round_entries(d)) {
    const int64_t e = (int64_t)d.x + lane;
    R.pay = (unsigned)__ldg(P.dvals + e);
#pragma unroll
    for (int n = 0; n < 3; ++n) R.er[n] = __ldg(P.erank + 3 * e + n);
  }
  if (d.y <= RND_MAX_ENT && lane < d.w) {
    const int64_t ti = (int64_t)d.z + lane;
    R.e0 = __ldg(P.tfirst + ti);
    R.e1 = __ldg(P.tfirst + ti + 1);
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      R.rb[m] = __ldg(P.rowbase + 3 * ti + m);
      R.dr[m] = __ldg(P.drank + 3 * ti + m);
    }
  }
}

// PROJ: TT_HESS_PSDPROJ compiled in (the other modes run the leaner instantiation).  PARTS: some slots are parts of
// split triangles (more than 32 partners); without any -- up to ~15 M pairs on BASELINE's 2 M-triangle soup -- the
// instantiation without their code runs: the kernel sits at 254 of 255 registers and the few selects and the ballot
// of the part path cost it 3 % (measured, profiles/r2_step_breakdown.md).
#ifdef TT_K4_PROFILE
__device__ unsigned long long tt_k4_prof[16];
#define K4_MARK(i) { const long long t_ = clock64(); prof[i] += t_ - tprev; tprev = t_; }
#else
#define K4_MARK(i)
#endif
template <typename T, bool PROJ, bool PARTS, int MT>
__global__ void __maxnreg__(TT_TILE_MAXNREG)
k_assemble_tile(const AsmParams<T> P) {
  extern __shared__ __align__(16) unsigned char s_raw[];
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int RUN_UNIT = TileCfg<T, MT>::RUN_UNIT;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int NBUF = TileCfg<T, MT>::NBUF, UNION_BYTES = TileCfg<T, MT>::UNION_BYTES;
  TileWarpSmem<T, MT>& S = reinterpret_cast<TileWarpSmem<T, MT>*>(s_raw)[warp];
  int krow = 0;  // rows handed to the copy engine so far: row k lives in tile buffer k % NBUF
  const int64_t G = (int64_t)gridDim.x * TILE_WARPS;
  int64_t c = (int64_t)blockIdx.x * TILE_WARPS + warp;
  if (c >= P.n_chunks) return;
  const int cn = (lane < 27) ? lane / 9 : 0, cq = (lane < 27) ? lane % 9 : 0;
  const int4 dzero = make_int4(0, 0, 0, 0);

  // ---- prologue: this warp's first round ----
  int4 d_cur = __ldg(P.rdesc + c);
  int4 d_nxt = (c + G < P.n_chunks) ? __ldg(P.rdesc + c + G) : dzero;
  int4 d_nn = (c + 2 * G < P.n_chunks) ? __ldg(P.rdesc + c + 2 * G) : dzero;
  RoundOps cur;
  load_round_ops(P, d_cur, lane, cur);
  int ids_nxt[6];
  double x[18];  // J and the coefficients always in fp64 (reading A12; measured: fp32 J misses the 1e-4 bar on config 3)
  {
    int ids_cur[6];
    load_round_ids(P, d_cur, lane, ids_cur);
#pragma unroll
    for (int i = 0; i < 18; ++i) x[i] = 0.0;
    if (lane < round_entries(d_cur)) load_pos18(P.pos, ids_cur, x);
  }
  load_round_ids(P, d_nxt, lane, ids_nxt);

#ifdef TT_K4_PROFILE
  long long prof[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  long long tprev = clock64();
#endif
  while (true) {
    const bool has_next = c + G < P.n_chunks;
    const int e_lo = d_cur.x, nent = d_cur.y, t_lo = d_cur.z, ntri = d_cur.w;
    const bool is_long = nent > RND_MAX_ENT;  // k_assemble_long's
    const bool valid = !is_long && lane < nent;

    // positions of the NEXT round: pulled into L2 now (no registers, no scoreboard), loaded into
    // registers at the end of this round, when the derivative registers are free again
    if (lane < round_entries(d_nxt)) prefetch_pos_l2(P.pos, ids_nxt);

    // ---- lane = entry: J, coefficients ----
    Entry<double> E;
#pragma unroll
    for (int i = 0; i < 18; ++i) { E.g0[i] = 0.0; E.g1[i] = 0.0; }
    E.cf = {0.0, 0.0, 0.0, 0.0, 0.0};
    E.en = 0.0;
    int er[3] = {cur.er[0], cur.er[1], cur.er[2]};
    if (valid) eval_core<double, PROJ>(x, cur.pay, P.sigma, P.hess_mode, E);
    K4_MARK(0)
    // ---- operands of round c + G, vertex ids of c + 2G, descriptor of c + 3G: requested after the
    //      register peak of the derivative code, consumed a round later ----
    RoundOps nxt;
    load_round_ops(P, d_nxt, lane, nxt);
    int ids_nn[6];
    load_round_ids(P, d_nn, lane, ids_nn);
    const int4 d_nnn = (c + 3 * G < P.n_chunks) ? __ldg(P.rdesc + c + 3 * G) : dzero;
    // the staging area aliases the tile buffer of this round's first row: the copy engine must have read the row that
    // used it last (every lane commits one group per row, so "all but the NBUF - 1 newest groups" means exactly that)
    constexpr bool ONEPASS = TileCfg<T, MT>::ONEPASS;  // the staging area spans the tile buffer(s)
    double* const stage = reinterpret_cast<double*>(S.tile + (ONEPASS ? 0 : (krow % NBUF) * UNION_BYTES));
    bulk_wait_read_n<ONEPASS ? 0 : NBUF - 1>();
    __syncwarp();
    if (valid) {
      unpermute_own(E, er);
    }
    K4_MARK(1)

    if (!is_long) {
      // lane = triangle: tile slots (16-byte slots, prefix sum over the round's triangles)
      const bool part_slot = PARTS && cur.dr[0] < 0;  // a part of a split triangle: no diagonal blocks in its runs
      const int run_bytes = RUN_UNIT * (cur.e1 - cur.e0 + (part_slot ? 0 : 1));
      int slot_off;
      {
        int incl = (lane < ntri) ? (((run_bytes + 15) & ~15) + 16) : 0;
        const int mine = incl;
#pragma unroll
        for (int o = 1; o < MT; o <<= 1) {
          const int v = __shfl_up_sync(FULL, incl, o);
          if (lane >= o) incl += v;
        }
        slot_off = incl - mine;
      }
      // bit i of heads: entry i is the first of its triangle; my_ti: triangle of entry `lane`
      const unsigned heads = __reduce_or_sync(FULL, (lane < ntri) ? (1u << (cur.e0 - e_lo)) : 0u);
      const int my_ti = __popc(heads & (0xffffffffu >> (31 - lane))) - 1;
      const int my_first = (lane < ntri) ? cur.e0 - e_lo : nent;  // first entry of triangle `lane`; nent past the last

      // ---- diagonal 9x9 (symmetric: 45 unique) + gradient: stage per entry, sum per triangle ----
      double d0[9], d1[9];
#pragma unroll
      for (int i = 0; i < 9; ++i) {
        d0[i] = E.cf.c00 * E.g0[i] + E.cf.c01 * E.g1[i];
        d1[i] = E.cf.c01 * E.g0[i] + E.cf.c11 * E.g1[i];
      }
      K4_MARK(2)
      if constexpr (ONEPASS) {
        if (valid) {
          double* st = stage + lane * STG1_STRIDE;
          int k = 0;
#pragma unroll
          for (int r = 0; r < 9; ++r)
#pragma unroll
            for (int q = r; q < 9; ++q, ++k) st[k] = E.g0[r] * d0[q] + E.g1[r] * d1[q];
#pragma unroll
          for (int i = 0; i < 9; ++i) st[NDIAG + i] = E.cf.cg0 * E.g0[i] + E.cf.cg1 * E.g1[i];
        }
        __syncwarp();
        K4_MARK(3)
        // per-triangle sums: lane = components (lane, lane + 27), entries in ascending order (deterministic); two
        // triangles at a time: four independent load -> add chains in flight
        for (int tt = 0; tt < ntri; tt += 2) {
          const int a0 = __shfl_sync(FULL, my_first, tt), a1 = __shfl_sync(FULL, my_first, tt + 1);
          const int b1 = __shfl_sync(FULL, my_first, tt + 2);
          const int dA = a1 - a0, dB = b1 - a1, dn = max(dA, dB);
          if (lane < STG_PASS) {
            const double* pA = stage + a0 * STG1_STRIDE + lane;
            const double* pB = stage + a1 * STG1_STRIDE + lane;
            constexpr int RU1 = (MT > RND_TRI_LOW) ? TT_RED_UNR1_WIDE : RED_UNR1;  // 16-slot rounds: triangles with few entries
            double vA0[RU1], vA1[RU1], vB0[RU1], vB1[RU1];
#pragma unroll
            for (int j = 0; j < RU1; ++j) {
              vA0[j] = (j < dA) ? pA[j * STG1_STRIDE] : 0.0;
              vA1[j] = (j < dA) ? pA[j * STG1_STRIDE + STG_PASS] : 0.0;
              vB0[j] = (j < dB) ? pB[j * STG1_STRIDE] : 0.0;
              vB1[j] = (j < dB) ? pB[j * STG1_STRIDE + STG_PASS] : 0.0;
            }
            double accA0 = vA0[0], accA1 = vA1[0], accB0 = vB0[0], accB1 = vB1[0];
#pragma unroll
            for (int j = 1; j < RU1; ++j) {
              accA0 += vA0[j];
              accA1 += vA1[j];
              accB0 += vB0[j];
              accB1 += vB1[j];
            }
            for (int j = RU1; j < dn; ++j) {
              if (j < dA) {
                accA0 += pA[j * STG1_STRIDE];
                accA1 += pA[j * STG1_STRIDE + STG_PASS];
              }
              if (j < dB) {
                accB0 += pB[j * STG1_STRIDE];
                accB1 += pB[j * STG1_STRIDE + STG_PASS];
              }
            }
            S.dsum[tt][lane] = accA0;
            S.dsum[tt][STG_PASS + lane] = accA1;
            if (dB > 0) {
              S.dsum[tt + 1][lane] = accB0;
              S.dsum[tt + 1][STG_PASS + lane] = accB1;
            }
            if (lane >= NDIAG - STG_PASS) {  // gradient of the triangle's three vertices
              T* ts = P.tslot + 9 * ((int64_t)t_lo + tt) + (lane - (NDIAG - STG_PASS));
              ts[0] = (T)accA1;
              if (dB > 0) ts[9] = (T)accB1;
            }
          }
        }
        __syncwarp();
        K4_MARK(4)
      } else
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (valid) {
          double* st = stage + lane * STG_STRIDE - h * STG_PASS;
          int k = 0;
#pragma unroll
          for (int r = 0; r < 9; ++r)
#pragma unroll
            for (int q = r; q < 9; ++q, ++k)
              if (k >= h * STG_PASS && k < (h + 1) * STG_PASS) st[k] = E.g0[r] * d0[q] + E.g1[r] * d1[q];
#pragma unroll
          for (int i = 0; i < 9; ++i)
            if (NDIAG + i >= h * STG_PASS && NDIAG + i < (h + 1) * STG_PASS)
              st[NDIAG + i] = E.cf.cg0 * E.g0[i] + E.cf.cg1 * E.g1[i];
        }
        __syncwarp();
        K4_MARK(3)
        // per-triangle sums, lane = component, entries in ascending order (deterministic); two
        // triangles at a time so that two independent load -> add chains are in flight.  The loops
        // are warp-uniform: lanes >= STG_PASS only take part in the shuffles.
        for (int tt = 0; tt < ntri; tt += 2) {
          const int a0 = __shfl_sync(FULL, my_first, tt), a1 = __shfl_sync(FULL, my_first, tt + 1);
          const int b1 = __shfl_sync(FULL, my_first, tt + 2);
          const int dA = a1 - a0, dB = b1 - a1, dn = max(dA, dB);
          if (lane < STG_PASS) {
            const double* pA = stage + a0 * STG_STRIDE + lane;
            const double* pB = stage + a1 * STG_STRIDE + lane;
            // the first RED_UNR entries of both triangles are loaded before any add (one shared-memory
            // latency per pair of triangles, not one per entry); longer triangles finish in a loop
            double vA[RED_UNR], vB[RED_UNR];
#pragma unroll
            for (int j = 0; j < RED_UNR; ++j) {
              vA[j] = (j < dA) ? pA[j * STG_STRIDE] : 0.0;
              vB[j] = (j < dB) ? pB[j * STG_STRIDE] : 0.0;
            }
            double accA = vA[0], accB = vB[0];
#pragma unroll
            for (int j = 1; j < RED_UNR; ++j) {
              accA += vA[j];
              accB += vB[j];
            }
#pragma unroll 2
            for (int j = RED_UNR; j < dn; ++j) {
              if (j < dA) accA += pA[j * STG_STRIDE];
              if (j < dB) accB += pB[j * STG_STRIDE];
            }
            S.dsum[tt][h * STG_PASS + lane] = accA;
            if (dB > 0) S.dsum[tt + 1][h * STG_PASS + lane] = accB;
            if (h == 1 && lane >= NDIAG - STG_PASS) {  // gradient of the triangle's three vertices
              T* ts = P.tslot + 9 * ((int64_t)t_lo + tt) + (lane - (NDIAG - STG_PASS));
              ts[0] = (T)accA;
              if (dB > 0) ts[9] = (T)accB;
            }
          }
        }
        __syncwarp();
        K4_MARK(4)
      }

      if (PARTS) {  // parts hand their diagonal partial sums to k_split_finish
        const int pidx = (lane < ntri && part_slot) ? (-1 - cur.dr[0]) : -1;
        if (__ballot_sync(FULL, pidx >= 0)) {
          for (int tt = 0; tt < ntri; ++tt) {
            const int px = __shfl_sync(FULL, pidx, tt);
            if (px >= 0)
              for (int k = lane; k < NDIAG; k += 32) P.dpart[(int64_t)NDIAG * px + k] = S.dsum[tt][k];
          }
        }
      }
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const unsigned long long g =
            (unsigned long long)((cur.rb[m] >= 0) ? (P.vals + 9 * cur.rb[m]) : (P.tvals + 9 * (-cur.rb[m] - 1)));
        const int my_off = slot_off + (int)(g & 15ull);
        // the copy engine must have read the row that used this buffer last
        unsigned char* const tb = S.tile + (krow % NBUF) * UNION_BYTES;
        ++krow;
        if (m > 0) {
          bulk_wait_read_n<NBUF - 1>();
          __syncwarp();
        }
        if (lane < ntri) {
          S.run_off[lane] = my_off;
#pragma unroll
          for (int n = 0; n < 3; ++n) S.diag_off[lane][n] = part_slot ? -1 : my_off + 9 * (int)sizeof(T) * cur.dr[n];
        }
        __syncwarp();
        if (valid) {
          // The two outer products of a block run in the OUTPUT precision (fp32 variant: FFMA on the rounded J,
          // 1e-7 relative per block against a 1e-3 tolerance); J, the coefficients, the staged diagonal /
          // gradient products and every sum over pairs stay fp64 -- reading A12.  (Staging in fp32 was measured:
          // 54 more F2F conversions per entry, K4 2.45 -> 2.70 ms.)
          T at[3], bt[3];
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            at[i] = (T)(E.cf.c00 * E.g0[3 * m + i] + E.cf.c01 * E.g1[3 * m + i]);
            bt[i] = (T)(E.cf.c01 * E.g0[3 * m + i] + E.cf.c11 * E.g1[3 * m + i]);
          }
          T* run = reinterpret_cast<T*>(tb + S.run_off[my_ti]);
#pragma unroll
          for (int n = 0; n < 3; ++n) {
            T* blk = run + 9 * er[n];
            T p0[3], p1[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
              p0[j] = (T)E.g0[9 + 3 * n + j];
              p1[j] = (T)E.g1[9 + 3 * n + j];
            }
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
              for (int j = 0; j < 3; ++j) blk[3 * i + j] = at[i] * p0[j] + bt[i] * p1[j];
          }
        }
        K4_MARK(5)
        // diagonal-row blocks (p_m, p_n): lane = element (n, i, j), from the packed upper triangle
        if (lane < 27) {
          const int r_ = 3 * m + cq / 3, c_ = 3 * cn + cq % 3;
          const int lo = min(r_, c_), hi = max(r_, c_);
          const int uidx = lo * 9 - (lo * (lo - 1)) / 2 + (hi - lo);
          int off[MT];
          T val[MT];
#pragma unroll
          for (int tt = 0; tt < MT; ++tt) {  // slots past ntri hold stale but readable data
            off[tt] = S.diag_off[tt][cn];
            val[tt] = (T)S.dsum[tt][uidx];
          }
#pragma unroll
          for (int tt = 0; tt < MT; ++tt)
            if (tt < ntri && (!PARTS || off[tt] >= 0)) *reinterpret_cast<T*>(tb + off[tt] + cq * (int)sizeof(T)) = val[tt];
        }
        // positions of the next round (L2 hits): requested as soon as this round's J is dead
        if (m == 2 && lane < round_entries(d_nxt)) load_pos18(P.pos, ids_nxt, x);
        K4_MARK(6)
        fence_async_smem();
        __syncwarp();
        // ---- lane = triangle: hand the run to the copy engine ----
        if (lane < ntri) {
          const unsigned char* src = tb + my_off;
          int head = (int)((16ull - (g & 15ull)) & 15ull);
          head = min(head, run_bytes);
          const int body = (run_bytes - head) & ~15;
          if (sizeof(T) == 8) {  // blocks are 8-byte aligned: at most one value before and one after the body
            if (head > 0) *reinterpret_cast<T*>(g) = *reinterpret_cast<const T*>(src);
            if (body > 0) bulk_s2g(reinterpret_cast<void*>(g + head), src + head, (uint32_t)body);
            if (head + body < run_bytes)
              *reinterpret_cast<T*>(g + head + body) = *reinterpret_cast<const T*>(src + head + body);
          } else {
            for (int o = 0; o < head; o += (int)sizeof(T)) *reinterpret_cast<T*>(g + o) = *reinterpret_cast<const T*>(src + o);
            if (body > 0) bulk_s2g(reinterpret_cast<void*>(g + head), src + head, (uint32_t)body);
            for (int o = head + body; o < run_bytes; o += (int)sizeof(T))
              *reinterpret_cast<T*>(g + o) = *reinterpret_cast<const T*>(src + o);
          }
        }
        bulk_commit();  // by every lane, so that all lanes count the same groups
        K4_MARK(7)
      }
    }
    if (is_long && lane < round_entries(d_nxt)) load_pos18(P.pos, ids_nxt, x);
    double e_acc = (double)E.en;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_down_sync(FULL, e_acc, o);
    if (lane == 0) P.chunk_energy[c] = e_acc;  // 0 for a long round: k_assemble_long overwrites it
    K4_MARK(8)
    if (!has_next) break;
    c += G;
    d_cur = d_nxt;
    d_nxt = d_nn;
    d_nn = d_nnn;
    cur = nxt;
#pragma unroll
    for (int i = 0; i < 6; ++i) ids_nxt[i] = ids_nn[i];
  }
  bulk_wait_all();  // shared memory must outlive the engine's reads
#ifdef TT_K4_PROFILE
  if (lane == 0) for (int i = 0; i < 10; ++i) atomicAdd(&tt_k4_prof[i], (unsigned long long)prof[i]);
#endif
}

// Long triangles with at most LONG_TILE_MAX partners (a round of their own): one warp per triangle.
// A row of the triangle is ONE run of 3 (deg + 1) blocks; it is built in a shared-memory tile and
// handed to the copy engine like the runs of k_assemble_tile.  The tile holds one row, so the warp
// makes three passes over the triangle's entries (m = 0, 1, 2).  CACHE = true (deg <= LONG_CACHE_MAX):
// pass 0 leaves J and the coefficients of every entry in shared memory (lane-private columns) and
// passes 1, 2 reload them; CACHE = false: J is re-evaluated in every pass (the derivative code is
// ~20 % of an entry's cost; three tiles or a larger cache would not fit).  The diagonal blocks and
// the gradient of row m are summed in registers: lane-private partial sums over the groups of 32
// entries, then a reduce-scatter butterfly (fixed tree: deterministic) that leaves value L in lane L.
// Launched after k_assemble_tile on the same stream (it overwrites that round's energy slot).
constexpr int LONG_TILE_MAX = 127;
constexpr int LONG_CACHE_MAX = 64;
constexpr int JC_N = 41;  // g0[18], g1[18], c00, c11, c01, cg0, cg1
template <typename T, bool CACHE>
struct alignas(16) LongTileSmem {
  unsigned char tile[27 * sizeof(T) * ((CACHE ? LONG_CACHE_MAX : LONG_TILE_MAX) + 1) + 16];
  double jc[CACHE ? JC_N * LONG_CACHE_MAX : 1];  // value k of entry (group gi, lane) at [(gi * JC_N + k) * 32 + lane]
};

// v[0..32) per lane -> lane L returns the warp sum of v[L]
__device__ __forceinline__ double warp_reduce_scatter32(double (&v)[32], int lane) {
  constexpr unsigned FULL = 0xffffffffu;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const bool up = (lane & o) != 0;
#pragma unroll
    for (int i = 0; i < o; ++i) {
      const double send = up ? v[i] : v[i + o];
      const double keep = up ? v[i + o] : v[i];
      v[i] = keep + __shfl_xor_sync(FULL, send, o);
    }
  }
  return v[0];
}

template <typename T, bool CACHE>
__global__ void __launch_bounds__(32)
k_assemble_long_tile(const AsmParams<T> P) {
  extern __shared__ __align__(16) unsigned char s_raw[];
  constexpr unsigned FULL = 0xffffffffu;
  LongTileSmem<T, CACHE>& S = *reinterpret_cast<LongTileSmem<T, CACHE>*>(s_raw);
  const int lane = threadIdx.x;
  const int64_t li = blockIdx.x;
  if (li >= P.n_long) return;
  const int c = __ldg(P.long_list + li);
  const int4 d = __ldg(P.rdesc + c);
  if (CACHE ? (d.y > LONG_CACHE_MAX) : (d.y <= LONG_CACHE_MAX || d.y > LONG_TILE_MAX)) return;  // another kernel's
  const int64_t ti = d.z;
  const int e_lo = d.x, e_hi = d.x + d.y;
  const int run_bytes = 27 * (int)sizeof(T) * (d.y + 1);
  double e_acc = 0.0;
#pragma unroll 1
  for (int m = 0; m < 3; ++m) {
    const int64_t rb = __ldg(P.rowbase + 3 * ti + m);
    const int my_dr = (lane < 27) ? __ldg(P.drank + 3 * ti + lane / 9) : 0;
    const unsigned long long g = (unsigned long long)((rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1)));
    unsigned char* const run = S.tile + (int)(g & 15ull);
    double acc[32];  // diagonal-row blocks (p_m, p_n) at [9 n + 3 i + j], gradient of p_m at [27 + i]
#pragma unroll
    for (int k = 0; k < 32; ++k) acc[k] = 0.0;
    if (m > 0) {  // the copy engine must have read the previous row
      bulk_wait_read();
      __syncwarp();
    }
    int gi = 0;
    for (int base = e_lo; base < e_hi; base += 32, ++gi) {
      if (base + lane < e_hi) {
        const int64_t e = (int64_t)base + lane;
        int er[3];
#pragma unroll
        for (int n = 0; n < 3; ++n) er[n] = __ldg(P.erank + 3 * e + n);
        Entry<double> E;
        double* const jc = S.jc + gi * JC_N * 32 + lane;
        if (!CACHE || m == 0) {
          int ids[6];
          {
            const int2* iv = reinterpret_cast<const int2*>(P.everts + 6 * e);
            const int2 v0 = __ldg(iv), v1 = __ldg(iv + 1), v2 = __ldg(iv + 2);
            ids[0] = v0.x; ids[1] = v0.y; ids[2] = v1.x; ids[3] = v1.y; ids[4] = v2.x; ids[5] = v2.y;
          }
          double x[18];
          load_pos18(P.pos, ids, x);
          eval_core(x, (unsigned)__ldg(P.dvals + e), P.sigma, P.hess_mode, E);
          if (m == 0) e_acc += E.en;
          unpermute_own(E, er);
          if (CACHE) {
#pragma unroll
            for (int k = 0; k < 18; ++k) {
              jc[k * 32] = E.g0[k];
              jc[(18 + k) * 32] = E.g1[k];
            }
            jc[36 * 32] = E.cf.c00; jc[37 * 32] = E.cf.c11; jc[38 * 32] = E.cf.c01;
            jc[39 * 32] = E.cf.cg0; jc[40 * 32] = E.cf.cg1;
          }
        } else {
#pragma unroll
          for (int k = 0; k < 18; ++k) {
            E.g0[k] = jc[k * 32];
            E.g1[k] = jc[(18 + k) * 32];
          }
          E.cf.c00 = jc[36 * 32]; E.cf.c11 = jc[37 * 32]; E.cf.c01 = jc[38 * 32];
          E.cf.cg0 = jc[39 * 32]; E.cf.cg1 = jc[40 * 32];
          // er must follow the recorded -> partner order again (pp is not cached: redo the selects)
          const unsigned pay = (unsigned)__ldg(P.dvals + e);
          const bool side = (pay & 1u) != 0u;
          const unsigned cp = side ? ((pay >> 1) & 63u) : ((pay >> 7) & 63u);  // partner triangle's config
          int pp[3];
          pp[0] = (int)(cp & 3u); pp[1] = (int)((cp >> 2) & 3u); pp[2] = 3 - pp[0] - pp[1];
          const int e0 = er[0], e1 = er[1], e2 = er[2];
#pragma unroll
          for (int r = 0; r < 3; ++r) er[r] = (pp[r] == 0) ? e0 : ((pp[r] == 1) ? e1 : e2);
        }
        double a[3], b[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {  // own row m: dynamic m, selected from the three static rows
          const double g0m = (m == 0) ? E.g0[i] : ((m == 1) ? E.g0[3 + i] : E.g0[6 + i]);
          const double g1m = (m == 0) ? E.g1[i] : ((m == 1) ? E.g1[3 + i] : E.g1[6 + i]);
          a[i] = E.cf.c00 * g0m + E.cf.c01 * g1m;
          b[i] = E.cf.c01 * g0m + E.cf.c11 * g1m;
          acc[27 + i] += E.cf.cg0 * g0m + E.cf.cg1 * g1m;
        }
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          T* blk = reinterpret_cast<T*>(run) + 9 * er[n];
#pragma unroll
          for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
              blk[3 * i + j] = (T)(a[i] * E.g0[9 + 3 * n + j] + b[i] * E.g1[9 + 3 * n + j]);
              acc[9 * n + 3 * i + j] += a[i] * E.g0[3 * n + j] + b[i] * E.g1[3 * n + j];
            }
        }
      }
    }
    const double tot = warp_reduce_scatter32(acc, lane);  // lane L: sum of value L
    if (lane < 27) reinterpret_cast<T*>(run)[9 * my_dr + lane % 9] = (T)tot;
    else if (lane < 30) P.tslot[9 * ti + 3 * m + (lane - 27)] = (T)tot;
    fence_async_smem();
    __syncwarp();
    if (lane == 0) {
      int head = (int)((16ull - (g & 15ull)) & 15ull);
      head = min(head, run_bytes);
      const int body = (run_bytes - head) & ~15;
      for (int o = 0; o < head; o += (int)sizeof(T)) *reinterpret_cast<T*>(g + o) = *reinterpret_cast<const T*>(run + o);
      if (body > 0) bulk_s2g(reinterpret_cast<void*>(g + head), run + head, (uint32_t)body);
      for (int o = head + body; o < run_bytes; o += (int)sizeof(T))
        *reinterpret_cast<T*>(g + o) = *reinterpret_cast<const T*>(run + o);
      bulk_commit();
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_down_sync(FULL, e_acc, o);
  if (lane == 0) P.chunk_energy[c] = e_acc;
  bulk_wait_all();  // shared memory must outlive the engine's reads
}

// Triangles with more than LONG_TILE_MAX partners: one warp per triangle, entries in groups of 32,
// off-diagonal blocks stored directly, diagonal rows and gradient carried across groups.
// Launched after k_assemble_tile on the same stream (it overwrites that round's energy slot).
template <typename T>
__global__ void __launch_bounds__(32 * TILE_WARPS)
k_assemble_long_direct(const AsmParams<T> P) {
  extern __shared__ __align__(16) unsigned char s_raw[];
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  LongWarpSmem& S = reinterpret_cast<LongWarpSmem*>(s_raw)[warp];
  const int64_t li = (int64_t)blockIdx.x * TILE_WARPS + warp;
  if (li >= P.n_long) return;
  const int c = __ldg(P.long_list + li);
  const int4 d = __ldg(P.rdesc + c);
  if (d.y <= LONG_TILE_MAX) return;  // k_assemble_long_tile's
  const int64_t ti = d.z;
  const int e_lo = d.x, e_hi = d.x + d.y;
  T* rowp[3];
  int dr[3];
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    const int64_t rb = __ldg(P.rowbase + 3 * ti + m);
    rowp[m] = (rb >= 0) ? (P.vals + 9 * rb) : (P.tvals + 9 * (-rb - 1));
    dr[m] = __ldg(P.drank + 3 * ti + m);
  }
  const int cn = (lane < 27) ? lane / 9 : 0, cq = (lane < 27) ? lane % 9 : 0;
  double acc[3] = {0.0, 0.0, 0.0}, e_acc = 0.0;
  for (int base = e_lo; base < e_hi; base += 32) {
    const int nvalid = min(32, e_hi - base);
    const bool valid = lane < nvalid;
    Entry<double> E;
    int er[3] = {0, 0, 0};
    if (valid) {
      const int64_t e = (int64_t)base + lane;
      int ids[6];
#pragma unroll
      for (int i = 0; i < 6; ++i) ids[i] = __ldg(P.everts + 6 * e + i);
#pragma unroll
      for (int n = 0; n < 3; ++n) er[n] = __ldg(P.erank + 3 * e + n);
      double x[18];
      load_pos18(P.pos, ids, x);
      eval_core(x, (unsigned)__ldg(P.dvals + e), P.sigma, P.hess_mode, E);
      e_acc += E.en;
      unpermute_own(E, er);
    }
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      if (valid) {
        double a[3], b[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          a[i] = E.cf.c00 * E.g0[3 * m + i] + E.cf.c01 * E.g1[3 * m + i];
          b[i] = E.cf.c01 * E.g0[3 * m + i] + E.cf.c11 * E.g1[3 * m + i];
        }
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          T* blk = rowp[m] + 9 * (int64_t)er[n];
#pragma unroll
          for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) blk[3 * i + j] = (T)(a[i] * E.g0[9 + 3 * n + j] + b[i] * E.g1[9 + 3 * n + j]);
        }
        double* st = S.stage + lane * LONG_STRIDE;
#pragma unroll
        for (int n = 0; n < 3; ++n)
#pragma unroll
          for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) st[9 * n + 3 * i + j] = a[i] * E.g0[3 * n + j] + b[i] * E.g1[3 * n + j];
#pragma unroll
        for (int i = 0; i < 3; ++i) st[27 + i] = E.cf.cg0 * E.g0[3 * m + i] + E.cf.cg1 * E.g1[3 * m + i];
      }
      __syncwarp();
      if (lane < 30)
        for (int i = 0; i < nvalid; ++i) acc[m] += S.stage[i * LONG_STRIDE + lane];
      __syncwarp();
    }
  }
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    if (lane < 27) rowp[m][9 * (int64_t)dr[cn] + cq] = (T)acc[m];
    else if (lane < 30) P.tslot[9 * ti + 3 * m + (lane - 27)] = (T)acc[m];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_down_sync(FULL, e_acc, o);
  if (lane == 0) P.chunk_energy[c] = e_acc;
}

// ------------------------------------------------------------------------------------------ K6
// MODE 1: energy + gradient only.  MODE 2: matrix-free H.p:  y_s = sum_j (J^T M (J p_loc))_own.
// Same rounds as K4, lane = directed entry.  A lane brings its 9 own-vertex values back to the
// triangle's own vertex order (selects on the recorded permutation) and the per-triangle sums are
// a SEGMENTED warp scan over the lanes (shuffles, fixed tree order: deterministic); the last lane
// of each triangle writes its 9 sums.  No shared memory, no atomics.  A long triangle is a round of
// its own and simply takes several groups of 32 entries, carried in registers.
constexpr int RED_THREADS = 128;
#ifndef TT_RED_MIN_CTAS
#define TT_RED_MIN_CTAS 3
#endif
template <typename T, int MODE>
__global__ void __launch_bounds__(RED_THREADS, TT_RED_MIN_CTAS)
k_entry_reduce(const AsmParams<T> P, const int* __restrict__ round_list, int64_t n_rounds) {
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t ci = (int64_t)blockIdx.x * (RED_THREADS / 32) + warp;
  if (ci >= n_rounds) return;
  const int64_t c = round_list ? (int64_t)__ldg(round_list + ci) : ci;
  const int4 d = __ldg(P.rdesc + c);
  const int e_lo = d.x, e_hi = d.x + d.y;
  const bool is_long = d.y > RND_MAX_ENT;
  unsigned heads = 1u;  // bit i: entry i opens a triangle
  if (!is_long) {
    const int f = (lane < d.w) ? __ldg(P.tfirst + d.z + lane) - e_lo : 0;
    heads = __reduce_or_sync(FULL, (lane < d.w) ? (1u << f) : 0u);
  }
  const unsigned below = heads & (0xffffffffu >> (31 - lane));  // heads at or below this lane
  const int segf = 31 - __clz((int)below);                      // first lane of this lane's triangle
  double carry[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) carry[k] = 0.0;
  double e_acc = 0.0;
  for (int base = e_lo; base < e_hi; base += 32) {
    const int nvalid = min(32, e_hi - base);
    double v[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) v[k] = 0.0;
    if (lane < nvalid) {
      const int64_t e = (int64_t)base + lane;
      int ids[6];
      {
        const int2* iv = reinterpret_cast<const int2*>(P.everts + 6 * e);
        const int2 v0 = __ldg(iv), v1 = __ldg(iv + 1), v2 = __ldg(iv + 2);
        ids[0] = v0.x; ids[1] = v0.y; ids[2] = v1.x; ids[3] = v1.y; ids[4] = v2.x; ids[5] = v2.y;
      }
      double x[18];
      load_pos18(P.pos, ids, x);
      const unsigned pay = (unsigned)__ldg(P.dvals + e);
      Entry<double> E;
      eval_core(x, pay, P.sigma, P.hess_mode, E);
      e_acc += E.en;
      double u0 = E.cf.cg0, u1 = E.cf.cg1;  // MODE 1: Eq. 3
      if (MODE == 2) {
        const bool side = (pay & 1u) != 0u;
        const int pid[6] = {side ? ids[3] : ids[0], side ? ids[4] : ids[1], side ? ids[5] : ids[2],
                            side ? ids[0] : ids[3], side ? ids[1] : ids[4], side ? ids[2] : ids[5]};
        double pv[18];  // p of (own, partner) vertices, recorded order
        load_pos18(P.pvec, pid, pv);
        double j0 = 0.0, j1 = 0.0;
#pragma unroll
        for (int i = 0; i < 18; ++i) {
          j0 = fma(E.g0[i], pv[i], j0);
          j1 = fma(E.g1[i], pv[i], j1);
        }
        u0 = E.cf.c00 * j0 + E.cf.c01 * j1;  // M (J p_loc)
        u1 = E.cf.c01 * j0 + E.cf.c11 * j1;
      }
      double yr[9];  // own half, recorded order
#pragma unroll
      for (int i = 0; i < 9; ++i) yr[i] = u0 * E.g0[i] + u1 * E.g1[i];
#pragma unroll
      for (int i = 0; i < 3; ++i)  // own vertex i = recorded position r with po[r] == i
#pragma unroll
        for (int cc = 0; cc < 3; ++cc)
          v[3 * i + cc] = (E.po[0] == i) ? yr[cc] : ((E.po[1] == i) ? yr[3 + cc] : yr[6 + cc]);
    }
    // segmented inclusive scan over the lanes (segments = triangles)
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const bool take = (lane - o) >= segf;
#pragma unroll
      for (int k = 0; k < 9; ++k) {
        const double up = __shfl_up_sync(FULL, v[k], o);
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
  if (MODE == 1) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_down_sync(FULL, e_acc, o);
    if (lane == 0) P.chunk_energy[c] = e_acc;
  }
}

// Pipelined form of the same kernel for the ordinary (non-long) rounds: persistent grid, a warp
// walks rounds c, c + G, ...  Positions (and p) of the NEXT round travel global -> shared with
// cp.async (LDGSTS: no registers held while in flight) into lane-private slots, vertex ids one
// round further ahead and descriptors two, so that the three dependent gathers of a round
// (descriptor -> vertex ids -> positions) are all off the critical path.
// One-warp CTAs: the kernel needs ~216 registers, and 9 x 32 x 216 fit the register file where 2 CTAs of 4 warps stop
// at 8 warps (0.942 -> 0.893 ms at 10 M pairs, measured; asking ptxas for 9 CTAs makes it cap the kernel at 168
// registers and spill: 1.30 ms -- so the bound below stays at 8 and the occupancy query finds the ninth).
#ifndef TT_PIPE_WARPS
#define TT_PIPE_WARPS 1
#endif
#ifndef TT_PIPE_MIN_CTAS
#define TT_PIPE_MIN_CTAS 8
#endif
constexpr int PIPE_WARPS = TT_PIPE_WARPS;
#ifndef TT_K6_SMEM_SUM
#define TT_K6_SMEM_SUM 1
#endif
template <typename T, int MODE>
struct PipeWarpSmem {
  T xp[2][9 * 32];                          // partner triangle's positions, lane-private slots [k * 32 + lane]
  T xo[2][9 * RND_MAX_TRI];                 // own triangle's positions, ONE copy per triangle (head lane's order)
  T pp[MODE == 2 ? 9 * 32 : 1];             // p of the partner's vertices
  T po[MODE == 2 ? 9 * RND_MAX_TRI : 1];    // p of the own vertices, one copy per triangle
  double stgf[sizeof(T) == 8 ? 1 : 9 * 32];  // staging of the per-entry results (fp64 aliases xp[buf], dead by then)
  int fst[RND_MAX_TRI + 2];                 // first entry of every triangle of the round, nent behind the last
};

struct PipeOps {
  int ids[6];      // lane = entry: canonical pair, recorded order
  unsigned pay;
  int f;           // lane = triangle: first entry of the triangle (ABSOLUTE: the round's first entry d.x is subtracted
                   // where f is used, rounds later -- subtracting it here made the load's first use immediate and left
                   // its latency exposed: 14 % of K6's stall samples sat on that one subtraction)
};
template <typename T>
__device__ __forceinline__ void load_pipe_ops(const AsmParams<T>& P, const int4 d, int lane, PipeOps& R) {
#pragma unroll
  for (int i = 0; i < 6; ++i) R.ids[i] = 0;
  R.pay = 0u;
  R.f = 0;
  if (d.y > RND_MAX_ENT) return;  // long round: k_entry_reduce's
  if (lane < d.y) {
    const int64_t e = (int64_t)d.x + lane;
    const int2* v = reinterpret_cast<const int2*>(P.everts + 6 * e);
    const int2 v0 = __ldg(v), v1 = __ldg(v + 1), v2 = __ldg(v + 2);
    R.ids[0] = v0.x; R.ids[1] = v0.y; R.ids[2] = v1.x; R.ids[3] = v1.y; R.ids[4] = v2.x; R.ids[5] = v2.y;
    R.pay = (unsigned)__ldg(P.dvals + e);
  }
  if (lane < d.w) R.f = __ldg(P.tfirst + d.z + lane);
}
__device__ __forceinline__ void own_first_ids(const PipeOps& R, int (&pid)[6]) {
  const bool side = (R.pay & 1u) != 0u;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    pid[i] = side ? R.ids[3 + i] : R.ids[i];
    pid[3 + i] = side ? R.ids[i] : R.ids[3 + i];
  }
}

// Where a lane finds its triangle's shared (own-vertex) slots: triangle index inside the round and,
// for each of its three own vertices in ITS recorded order, the position in the head lane's order.
struct OwnMap {
  int ti;
  int rp[3];
};

// The gathers of one round.  Every entry needs its partner's three vertices (lane-private slots),
// but the entries of one triangle all need the SAME three own vertices: only the triangle's first
// lane (head) requests them, once, and the others read the head's copy.  K6 is bound by the number
// of gather requests the L1 accepts (measured: dropping the own-vertex requests of the non-head
// lanes is worth 20 % of the kernel), not by bytes.
template <typename T>
__device__ __forceinline__ OwnMap issue_round_gather(const T* __restrict__ src, const PipeOps& o, const int4 d,
                                                     int lane, T* part, T* own) {
  constexpr unsigned FULL = 0xffffffffu;
  const bool ok = d.y <= RND_MAX_ENT;
  const bool valid = ok && lane < d.y;
  const unsigned heads = __reduce_or_sync(FULL, (ok && lane < d.w) ? (1u << (o.f - d.x)) : 0u) | 1u;
  const unsigned below = heads & (0xffffffffu >> (31 - lane));
  const int head_lane = 31 - __clz((int)below);
  int pid[6];
  own_first_ids(o, pid);
  OwnMap m;
  m.ti = __popc(below) - 1;
  const int h0 = __shfl_sync(FULL, pid[0], head_lane), h1 = __shfl_sync(FULL, pid[1], head_lane);
#pragma unroll
  for (int r = 0; r < 3; ++r) m.rp[r] = (pid[r] == h0) ? 0 : ((pid[r] == h1) ? 1 : 2);
  if (valid) {
#pragma unroll
    for (int v = 0; v < 3; ++v) {
      const T* g = src + 3 * (int64_t)pid[3 + v];
#pragma unroll
      for (int k = 0; k < 3; ++k) cp_async_elem(part + (3 * v + k) * 32 + lane, g + k);
    }
    if (lane == head_lane && m.ti < RND_MAX_TRI) {
#pragma unroll
      for (int v = 0; v < 3; ++v) {
        const T* g = src + 3 * (int64_t)pid[v];
#pragma unroll
        for (int k = 0; k < 3; ++k) cp_async_elem(own + 9 * m.ti + 3 * v + k, g + k);
      }
    }
  }
  return m;
}
// own-first values [own r = 0..2 | partner] of a lane, from the round's two areas
template <typename T>
__device__ __forceinline__ void read_round_gather(const T* part, const T* own, const OwnMap& m, int lane,
                                                  double (&v)[18]) {
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int k = 0; k < 3; ++k) v[3 * r + k] = (double)own[9 * m.ti + 3 * m.rp[r] + k];
#pragma unroll
  for (int i = 0; i < 9; ++i) v[9 + i] = (double)part[i * 32 + lane];
}

template <typename T, int MODE>
__global__ void __launch_bounds__(32 * PIPE_WARPS, TT_PIPE_MIN_CTAS)
k_entry_pipe(const AsmParams<T> P) {
  extern __shared__ __align__(16) unsigned char s_raw[];
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  PipeWarpSmem<T, MODE>& S = reinterpret_cast<PipeWarpSmem<T, MODE>*>(s_raw)[warp];
  const int64_t G = (int64_t)gridDim.x * PIPE_WARPS;
  int64_t c = (int64_t)blockIdx.x * PIPE_WARPS + warp;
  if (c >= P.n_chunks) return;
  const int4 dzero = make_int4(0, 0, 0, 0);
  // ---- prologue ----
  int4 d_cur = __ldg(P.rdesc + c);
  int4 d_nxt = (c + G < P.n_chunks) ? __ldg(P.rdesc + c + G) : dzero;
  int4 d_nn = (c + 2 * G < P.n_chunks) ? __ldg(P.rdesc + c + 2 * G) : dzero;
  PipeOps cur, nxt;
  load_pipe_ops(P, d_cur, lane, cur);
  load_pipe_ops(P, d_nxt, lane, nxt);
  OwnMap m_cur = issue_round_gather(P.pos, cur, d_cur, lane, S.xp[0], S.xo[0]);
  cp_async_commit();
  if (MODE == 2) {
    issue_round_gather(P.pvec, cur, d_cur, lane, S.pp, S.po);
    cp_async_commit();
  }
  int buf = 0;
  while (true) {
    const bool has_next = c + G < P.n_chunks;
    // ---- top of round c: ids two rounds ahead, descriptor three, positions of the next round ----
    PipeOps nn;
    load_pipe_ops(P, d_nn, lane, nn);
    const int4 d_nnn = (c + 3 * G < P.n_chunks) ? __ldg(P.rdesc + c + 3 * G) : dzero;
    const OwnMap m_nxt = issue_round_gather(P.pos, nxt, d_nxt, lane, S.xp[buf ^ 1], S.xo[buf ^ 1]);
    cp_async_commit();
    const int nent = d_cur.y;
    const bool is_long = nent > RND_MAX_ENT;  // k_entry_reduce's (launched over long_list)
    const bool valid = !is_long && lane < nent;
    const bool tri_lane = !is_long && lane < d_cur.w;
    if (MODE == 2) cp_async_wait<2>(); else cp_async_wait<1>();  // positions of THIS round have landed
    __syncwarp();                                                 // ... including the head lanes' copies
    double v[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) v[k] = 0.0;
    double e_acc = 0.0;
    Entry<double> E;
    if (valid) {
      double xf[18], x[18];
      read_round_gather(S.xp[buf], S.xo[buf], m_cur, lane, xf);
      const bool side = (cur.pay & 1u) != 0u;  // eval_core wants the canonical order (T_a first)
#pragma unroll
      for (int k = 0; k < 9; ++k) {
        x[k] = side ? xf[9 + k] : xf[k];
        x[9 + k] = side ? xf[k] : xf[9 + k];
      }
      eval_core(x, cur.pay, P.sigma, P.hess_mode, E);
      e_acc = E.en;
    }
    double u0 = 0.0, u1 = 0.0;
    if (MODE == 2) {
      cp_async_wait<1>();  // p of THIS round
      __syncwarp();
    }
    if (valid) {
      u0 = E.cf.cg0;  // MODE 1: Eq. 3
      u1 = E.cf.cg1;
      if (MODE == 2) {
        double pv[18];
        read_round_gather(S.pp, S.po, m_cur, lane, pv);
        double j0 = 0.0, j1 = 0.0;
#pragma unroll
        for (int i = 0; i < 18; ++i) {
          j0 = fma(E.g0[i], pv[i], j0);
          j1 = fma(E.g1[i], pv[i], j1);
        }
        u0 = E.cf.c00 * j0 + E.cf.c01 * j1;  // M (J p_loc)
        u1 = E.cf.c01 * j0 + E.cf.c11 * j1;
      }
      double yr[9];
#pragma unroll
      for (int i = 0; i < 9; ++i) yr[i] = u0 * E.g0[i] + u1 * E.g1[i];
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int cc = 0; cc < 3; ++cc)
          v[3 * i + cc] = (E.po[0] == i) ? yr[cc] : ((E.po[1] == i) ? yr[3 + cc] : yr[6 + cc]);
    }
    if (MODE == 2) {
      __syncwarp();  // every lane has read the shared p slots of this round: p of the next round
      issue_round_gather(P.pvec, nxt, d_nxt, lane, S.pp, S.po);
      cp_async_commit();
    }
    if (!is_long) {
#if TT_K6_SMEM_SUM
      // per-triangle sums through shared memory: every entry stages its 9 values, then lane = (triangle, component)
      // adds the triangle's entries in ascending order (a segmented shuffle scan of 9 doubles costs 5 x 9 x 3
      // instructions per lane; this is a third of it)
      double* const stg = (sizeof(T) == 8) ? reinterpret_cast<double*>(S.xp[buf]) : S.stgf;
      const int ntri = d_cur.w;
      __syncwarp();  // every lane has read its positions out of xp[buf]
      if (tri_lane) S.fst[lane] = cur.f - d_cur.x;
      if (lane == 0) S.fst[ntri] = nent;
      if (valid) {
#pragma unroll
        for (int k = 0; k < 9; ++k) stg[9 * lane + k] = v[k];
      }
      __syncwarp();
      for (int i = lane; i < 9 * ntri; i += 32) {
        const int t = i / 9, k = i - 9 * t;
        const int a = S.fst[t], b = S.fst[t + 1];
        const double* q = stg + 9 * a + k;
        double acc0 = 0.0, acc1 = 0.0;
        int e = a;
        for (; e + 1 < b; e += 2, q += 18) {
          acc0 += q[0];
          acc1 += q[9];
        }
        if (e < b) acc0 += q[0];
        P.tslot[9 * ((int64_t)d_cur.z + t) + k] = (T)(acc0 + acc1);
      }
      __syncwarp();  // the next round's gathers land in xp[buf]
#else
      const unsigned heads = __reduce_or_sync(FULL, tri_lane ? (1u << (cur.f - d_cur.x)) : 0u) | 1u;  // bit i: entry i opens a triangle
      const unsigned below = heads & (0xffffffffu >> (31 - lane));
      const int segf = 31 - __clz((int)below);
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const bool take = (lane - o) >= segf;
#pragma unroll
        for (int k = 0; k < 9; ++k) {
          const double up = __shfl_up_sync(FULL, v[k], o);
          if (take) v[k] += up;
        }
      }
      const bool last = valid && (lane == nent - 1 || ((heads >> 1) >> lane) & 1u);
      if (last) {
        const int64_t ti = (int64_t)d_cur.z + __popc(below) - 1;
#pragma unroll
        for (int k = 0; k < 9; ++k) P.tslot[9 * ti + k] = (T)v[k];
      }
#endif
      if (MODE == 1) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_down_sync(FULL, e_acc, o);
        if (lane == 0) P.chunk_energy[c] = e_acc;
      }
    }
    if (!has_next) break;
    c += G;
    d_cur = d_nxt;
    d_nxt = d_nn;
    d_nn = d_nnn;
    cur = nxt;
    nxt = nn;
    m_cur = m_nxt;
    buf ^= 1;
  }
  cp_async_wait<0>();
}

// Split triangles (one warp each), after K4 / K6: adds the parts' gradient (or H.p) partials into the
// triangle's first slot -- the one k_gather3 reads -- and, with HESS, sums the parts' diagonal partial sums
// (fixed order) and writes the triangle's nine diagonal blocks (rows exclusive by construction).
template <typename T, bool HESS>
__global__ void __launch_bounds__(128)
k_split_finish(const int4* __restrict__ split_list, int64_t n_split, const int* __restrict__ tris,
               const int* __restrict__ touched, const int* __restrict__ tsplit, const int* __restrict__ rowptr,
               const double* __restrict__ dpart, T* tslot, T* __restrict__ vals) {
  __shared__ double s_d[4][NDIAG];
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t i = (int64_t)blockIdx.x * 4 + w;
  if (i >= n_split) return;
  const int4 sp = __ldg(split_list + i);  // first slot, parts, touched index, first part ordinal
  if (lane < 9) {
    double a = 0.0;
    for (int k = 0; k < sp.y; ++k) a += (double)tslot[9 * ((int64_t)sp.x + k) + lane];
    tslot[9 * (int64_t)sp.x + lane] = (T)a;
  }
  if (HESS) {
    for (int k = lane; k < NDIAG; k += 32) {
      double a = 0.0;
      for (int q = 0; q < sp.y; ++q) a += __ldg(dpart + (int64_t)NDIAG * (sp.w + q) + k);
      s_d[w][k] = a;
    }
    __syncwarp();
    int ov[3];
    load3i(tris + 3 * (int64_t)__ldg(touched + sp.z), ov);
    const int pd = __ldg(tsplit + sp.z);
    if (lane < 27) {
      const int n = lane / 9, q = lane % 9;
      const int on = pick3(n, ov[0], ov[1], ov[2]);
      const int lr = (ov[0] < on) + (ov[1] < on) + (ov[2] < on);
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const int r_ = 3 * m + q / 3, c_ = 3 * n + q % 3;
        const int lo = min(r_, c_), hi = max(r_, c_);
        const int uidx = lo * 9 - (lo * (lo - 1)) / 2 + (hi - lo);
        vals[9 * ((int64_t)__ldg(rowptr + ov[m]) + 3 * pd + lr) + q] = (T)s_d[w][uidx];
      }
    }
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

// out[v] = sum over the touched slots of vertex v of tslot[slot]; zero for vertices no active pair
// touches.  A vertex with a single slot (always, in a soup) reads it through vslot1; the sorted
// vertex -> slot incidence (vptr / vslots, fixed order) is built only when some vertex has several.
template <typename T>
__global__ void k_gather3(const int* __restrict__ vcnt, const int* __restrict__ vslot1, const int* __restrict__ vptr,
                          const uint32_t* __restrict__ vslots, int64_t nV, const T* __restrict__ tslot,
                          T* __restrict__ out) {
  const int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // one thread per vertex: 3 consecutive values
  if (v >= nV) return;
  const int n = __ldg(vcnt + v);
  T r0 = (T)0, r1 = (T)0, r2 = (T)0;
  if (n == 1) {
    const T* t = tslot + 3 * (int64_t)__ldg(vslot1 + v);
    r0 = t[0]; r1 = t[1]; r2 = t[2];
  } else if (n > 1) {
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    for (int j = vptr[v]; j < vptr[v + 1]; ++j) {
      const T* t = tslot + 3 * (int64_t)vslots[j];
      a0 += (double)t[0]; a1 += (double)t[1]; a2 += (double)t[2];
    }
    r0 = (T)a0; r1 = (T)a1; r2 = (T)a2;
  }
  out[3 * v] = r0;
  out[3 * v + 1] = r1;
  out[3 * v + 2] = r2;
}

// Order-independent 64-bit checksum of n 32-bit words (each word mixed with its index, integer adds:
// associative and commutative, so the result does not depend on the schedule).  tt_hess_symbolic
// takes it of `pos`; the numeric phase and H.p re-take it and refuse to replay the recorded branch
// decisions at positions that have moved (TT_ERR_STATE).
__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  return z ^ (z >> 31);
}
__global__ void __launch_bounds__(256) k_checksum(const uint32_t* __restrict__ w, int64_t n, unsigned long long* __restrict__ out) {
  unsigned long long acc = 0ull;
  const int64_t stride = (int64_t)gridDim.x * 256;
  const int64_t n4 = ((reinterpret_cast<uintptr_t>(w) & 15) == 0) ? n / 4 : 0;  // 16-byte body when aligned
  const uint4* w4 = reinterpret_cast<const uint4*>(w);
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n4; i += stride) {
    const uint4 v = __ldg(w4 + i);
    const unsigned long long k = (unsigned long long)i * 0x9e3779b97f4a7c15ull;
    acc += mix64((((unsigned long long)v.y << 32) | v.x) ^ k) + mix64((((unsigned long long)v.w << 32) | v.z) ^ ~k);
  }
  for (int64_t i = 4 * n4 + (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += stride)
    acc += mix64((unsigned long long)__ldg(w + i) ^ ((unsigned long long)i * 0xd1b54a32d192ed03ull));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0 && acc) atomicAdd(out, acc);
}

// TT_FLAG_VALIDATE_INDICES: counts the entries of an index array outside [0, bound)
__global__ void k_count_out_of_range(const int* __restrict__ idx, int64_t n, int64_t bound, int* __restrict__ bad) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n && (idx[i] < 0 || (int64_t)idx[i] >= bound)) atomicAdd(bad, 1);
}

__global__ void k_i64_to_i32(const int64_t* __restrict__ in, int64_t n, int* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (int)in[i];
}

}  // namespace ttk
