// tt_lib.cu -- C ABI of libtt.so (include/tt.h): context, workspace, launch logic.
// Kernels: tt_kernels.cuh; per-pair arithmetic: tt_geom.cuh.  Scans / radix sorts / select of the
// symbolic phase use CUB (ships with the CUDA toolkit); everything the paper defines runs in the
// hand-written kernels.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>

#include <cub/cub.cuh>

#include "../../include/tt.h"
#include "tt_broad.cuh"
#include "tt_kernels.cuh"
#include "tt_probe.cuh"
#include "tt_solve.cuh"
#include "tt_exact.cuh"
#include "tt_membrane.cuh"

// ---- tt_energy_static: the scratch of the allocation-free energy entry point (include/tt.h) -----------------------
// File-scope device memory, held by every GPU that loads the library until the process exits: the per-CTA energy
// partials of K1, the slice sums of the two-level final sum, and the per-CTA active counts, for at most
// TT_STATIC_MAX_PAIRS candidates.  In HOST code the name below is a host-side stand-in, not a device address: tt_create
// asks for the address once per context, with the context's device current (cudaGetSymbolAddress), and the kernels are
// handed that pointer.  Every call shares the array and leaves its contents behind; nothing in it has to start at zero
// (every slot a call reads it has written itself), and calls that overlap on the GPU race on it.
constexpr int64_t TT_STATIC_MAX_BLK = TT_STATIC_MAX_PAIRS / ttk::CLS_THREADS;                     // 131072 CTAs of K1
constexpr int64_t TT_STATIC_MAX_STAGE = (TT_STATIC_MAX_BLK + ttk::SUM_SLICE - 1) / ttk::SUM_SLICE;  // 16 slice sums
constexpr int64_t TT_STATIC_DOUBLES = TT_STATIC_MAX_BLK + TT_STATIC_MAX_STAGE + TT_STATIC_MAX_BLK / 2;  // counts: int32
static_assert(TT_STATIC_MAX_PAIRS % ttk::CLS_THREADS == 0 && TT_STATIC_MAX_BLK % 2 == 0, "scratch layout");
static __device__ __align__(256) double tt_static_scratch[TT_STATIC_DOUBLES];  // 1.5 MB + 128 B

namespace {

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  ~DevBuf() { release(); }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    bytes = 0;
  }
  // grow-only; contents are NOT preserved across a grow
  cudaError_t ensure(size_t need) {
    if (need <= bytes) return cudaSuccess;
    release();
    size_t want = need + need / 8 + 256;
    cudaError_t e = cudaMalloc(&p, want);
    if (e != cudaSuccess) {
      p = nullptr;
      (void)cudaGetLastError();
      e = cudaMalloc(&p, need);
      want = need;
    }
    if (e == cudaSuccess) bytes = want;
    return e;
  }
  template <typename U> U* as() const { return reinterpret_cast<U*>(p); }
};

struct Signature {
  const void* pos = nullptr;
  const int32_t* tris = nullptr;
  const int32_t* pairs = nullptr;
  int64_t nV = -1, nT = -1, P = -1;
  bool valid = false;
  bool matches(const tt_problem* q) const {
    return valid && pos == q->pos && tris == q->tris && pairs == q->pairs && nV == q->n_verts &&
           nT == q->n_tris && P == q->n_pairs;
  }
};

}  // namespace

struct tt_ctx {
  tt_options opt;
  std::string err;
  int64_t launches = 0;
  // classification
  DevBuf mask, blk_count, blk_off, blk_energy, counts, energy, rec, sum_stage;
  // active set + directed entries
  DevBuf active_ids, ent_in, partner, dvals, tptr, zero_blk, touched, order, degp, tptrp;
  // per-triangle symbolic
  DevBuf erank, drank, tlen, toff, slot_excl, rowbase;
  int* vcnt_p = nullptr;    // views into zero_blk (one memset per symbolic call)
  int* rowlen_p = nullptr;
  // merge path
  DevBuf rkeys[2], rvals[2], head, ord, rowfirst, run_start, run_dest;
  // pattern
  DevBuf rowptr64, rowptr, colind;
  // numeric
  DevBuf everts, rdesc, tfirst, sfirst, sinfo, tsplit, split_list, dpart, bucket_cnt, bucket_off, long_list, asm_energy, tvals, tslot, vkeys[2], vvals[2], vptr, vslot1;
  DevBuf cub_tmp;
  DevBuf pcg_r, pcg_p, pcg_q, pcg_part[2], pcg_sc, pcg_hist;  // tt_pcg_solve workspace
  DevBuf nw_g, nw_d, nw_x, nw_vals, nw_minv, nw_sc;            // tt_newton_step workspace
  // membrane (tt_membrane_build): vertex -> neighbour adjacency, rest lengths
  DevBuf mb_keys[2], mb_ptr, mb_adj, mb_rest, mb_part, mb_num;
  int64_t mb_nV = -1, mb_half = 0;
  double mb_k = 0.0;
  double* static_scratch = nullptr;  // device address of tt_static_scratch on opt.device (tt_create)
  DevBuf possig;  // [2] u64: checksum of pos at tt_hess_symbolic, and at the last numeric / H.p call
  // broad phase (tt_broad_phase): boxes, grid, (cell, triangle) records, pair keys, result
  DevBuf bp_box, bp_part, bp_grid, bp_cnt, bp_off, bp_keys[2], bp_vals[2], bp_pcnt, bp_poff, bp_pkeys[2], bp_pairs;
  int64_t bp_n_pairs = -1;
  // host-API mirrors
  DevBuf h_pos, h_tris, h_pairs, h_p, o_vals, o_grad, o_energy, o_y;
  // cached symbolic state
  Signature sig;
  int64_t A = 0, n_dir = 0, n_touched = 0, R = 0, U = 0, nnzb = 0, n_chunks = 0, n_long = 0, rows_excl = 0, rows_gen = 0;
  int64_t n_slots = 0, n_split = 0, n_parts = 0;
  int bitsT = 1, bitsV = 1, sms = 148;
  int tile_grid[2][2] = {{0, 0}, {0, 0}};  // persistent grid of k_assemble_tile<double / float, MT = 8 / 16>
  int tri_limit = 8;          // slots-per-round limit the last symbolic call packed with (ttk::round_tri_limit)
  int pipe_grid[2][2] = {{0, 0}, {0, 0}};  // persistent grid of k_entry_pipe<double / float, MODE 1 / 2>
  uint64_t* rkeys_sorted = nullptr;
  uint32_t* rvals_sorted = nullptr;
  uint32_t* vvals_sorted = nullptr;
  int64_t host_nnzb = 0;
  // device-side timing of the three big kernels (events recorded on the caller's stream)
  // (a ring of EV_RING launches per kernel: tt_kernel_ms reads the latest, tt_kernel_ms_mean all of them)
  static constexpr int EV_RING = 64;
  cudaEvent_t evr[3][EV_RING][2] = {};
  int64_t ev_n[3] = {0, 0, 0};   // launches recorded since the last reset
  // host-buffer entry point: copies that do not feed the next kernel travel on a second stream
  cudaStream_t side = nullptr;
  cudaEvent_t ev_in = nullptr, ev_p = nullptr, ev_num = nullptr, ev_side = nullptr, ev_sig = nullptr;
  unsigned long long* h_sig = nullptr;  // pinned [2]: the two position checksums, read back without stalling the stream
};

namespace {

tt_status fail(tt_ctx* c, tt_status s, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  if (c) c->err = buf;
  return s;
}

#define TT_CUDA(call)                                                                            \
  do {                                                                                           \
    cudaError_t e_ = (call);                                                                     \
    if (e_ != cudaSuccess) {                                                                     \
      (void)cudaGetLastError();                                                                  \
      return fail(ctx, e_ == cudaErrorMemoryAllocation ? TT_ERR_NOMEM : TT_ERR_CUDA,             \
                  "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_));            \
    }                                                                                            \
  } while (0)

#define TT_LAUNCH_CHECK()                                                                        \
  do {                                                                                           \
    ctx->launches++;                                                                             \
    TT_CUDA(cudaGetLastError());                                                                 \
  } while (0)

inline int ceil_log2(int64_t n) {
  int b = 1;
  while ((int64_t(1) << b) < n) ++b;
  return b;
}
inline unsigned grid_for(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

struct CastI64 {
  __host__ __device__ int64_t operator()(int v) const { return (int64_t)v; }
};

tt_status check_problem(tt_ctx* ctx, const tt_problem* q) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (!q) return fail(ctx, TT_ERR_INVALID_ARG, "problem is NULL");
  if (q->n_verts < 0 || q->n_tris < 0 || q->n_pairs < 0) return fail(ctx, TT_ERR_INVALID_ARG, "negative size");
  if (q->n_verts >= (int64_t(1) << 31) / 3 || q->n_tris >= (int64_t(1) << 31) / 3 || q->n_pairs >= (int64_t(1) << 30))
    return fail(ctx, TT_ERR_INVALID_ARG, "sizes exceed int32 indexing (nV, nT < 2^31/3, P < 2^30)");
  if ((q->n_verts > 0 && !q->pos) || (q->n_tris > 0 && !q->tris) || (q->n_pairs > 0 && !q->pairs))
    return fail(ctx, TT_ERR_INVALID_ARG, "NULL array with non-zero size");
  return TT_OK;
}

// TT_FLAG_VALIDATE_INDICES: tris < nV and (if given) pairs < nT, checked on the device
tt_status validate_indices(tt_ctx* ctx, const int32_t* tris, int64_t nT, int64_t nV, const int32_t* pairs, int64_t P,
                           cudaStream_t st) {
  if (!(ctx->opt.flags & TT_FLAG_VALIDATE_INDICES)) return TT_OK;
  TT_CUDA(ctx->counts.ensure(sizeof(int64_t) * 16));
  int* d_bad = reinterpret_cast<int*>(ctx->counts.as<int64_t>() + 8);
  TT_CUDA(cudaMemsetAsync(d_bad, 0, 2 * sizeof(int), st));
  if (nT > 0) {
    ttk::k_count_out_of_range<<<grid_for(3 * nT, 256), 256, 0, st>>>(tris, 3 * nT, nV, d_bad);
    TT_LAUNCH_CHECK();
  }
  if (pairs && P > 0) {
    ttk::k_count_out_of_range<<<grid_for(2 * P, 256), 256, 0, st>>>(pairs, 2 * P, nT, d_bad + 1);
    TT_LAUNCH_CHECK();
  }
  int bad[2] = {0, 0};
  TT_CUDA(cudaMemcpyAsync(bad, d_bad, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaStreamSynchronize(st));
  if (bad[0] || bad[1])
    return fail(ctx, TT_ERR_INVALID_ARG, "%d vertex indices of tris outside [0, %lld), %d triangle indices of pairs outside [0, %lld)",
                bad[0], (long long)nV, bad[1], (long long)nT);
  return TT_OK;
}

// checksum of pos -> possig[slot] (enqueued on st)
tt_status pos_checksum(tt_ctx* ctx, const tt_problem* q, int slot, cudaStream_t st) {
  TT_CUDA(ctx->possig.ensure(sizeof(unsigned long long) * 2));
  unsigned long long* d = ctx->possig.as<unsigned long long>() + slot;
  TT_CUDA(cudaMemsetAsync(d, 0, sizeof(unsigned long long), st));
  const int64_t words = 3 * q->n_verts * (ctx->opt.dtype == TT_F64 ? 2 : 1);
  if (words > 0) {
    const int64_t want = (words / 4 + 255) / 256;
    ttk::k_checksum<<<(unsigned)(want < 148 * 8 ? (want > 0 ? want : 1) : 148 * 8), 256, 0, st>>>((const uint32_t*)q->pos, words, d);
    TT_LAUNCH_CHECK();
  }
  return TT_OK;
}
// The position check of the numeric / H.p calls, in two halves so that the GPU never waits for the host:
//   begin: enqueue the checksum of the current positions and its read-back into pinned memory, record an event;
//   (the caller then enqueues its kernels)
//   end:   wait for THAT EVENT only and compare with the checksum tt_hess_symbolic took -> TT_ERR_STATE.
// If the positions have moved, the kernels that were enqueued in between replay stale branch decisions: they
// cannot fault (every index is fixed by the symbolic phase) and the call returns the error, so its outputs are
// simply not valid -- as for any failed call.
tt_status check_positions_begin(tt_ctx* ctx, const tt_problem* q, cudaStream_t st) {
  if (ctx->opt.flags & TT_FLAG_NO_STATE_CHECK) return TT_OK;
  tt_status s = pos_checksum(ctx, q, 1, st);
  if (s != TT_OK) return s;
  TT_CUDA(cudaMemcpyAsync(ctx->h_sig, ctx->possig.p, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaEventRecord(ctx->ev_sig, st));
  return TT_OK;
}
tt_status check_positions_end(tt_ctx* ctx, const char* who) {
  if (ctx->opt.flags & TT_FLAG_NO_STATE_CHECK) return TT_OK;
  TT_CUDA(cudaEventSynchronize(ctx->ev_sig));
  if (ctx->h_sig[0] != ctx->h_sig[1])
    return fail(ctx, TT_ERR_STATE, "%s: positions changed since tt_hess_symbolic (the cached active set and branch decisions are stale): call tt_hess_symbolic again", who);
  return TT_OK;
}
// the same in one piece, for callers that must know before they enqueue anything (tt_pcg_solve)
tt_status check_positions(tt_ctx* ctx, const tt_problem* q, const char* who, cudaStream_t st) {
  tt_status s = check_positions_begin(ctx, q, st);
  if (s != TT_OK) return s;
  return check_positions_end(ctx, who);
}

// exclusive sum of n ints (+ grand total in out[n]); `in` must have n+1 entries with in[n] == 0
tt_status scan_i32(tt_ctx* ctx, const int* in, int* out, int64_t n_plus_1, cudaStream_t st) {
  size_t tmp = 0;
  TT_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tmp, in, out, n_plus_1, st));
  TT_CUDA(ctx->cub_tmp.ensure(tmp));
  TT_CUDA(cub::DeviceScan::ExclusiveSum(ctx->cub_tmp.p, tmp, in, out, n_plus_1, st));
  ctx->launches += 2;  // CUB scan: init + scan kernel
  return TT_OK;
}
tt_status scan_i64(tt_ctx* ctx, const int64_t* in, int64_t* out, int64_t n_plus_1, cudaStream_t st) {
  size_t tmp = 0;
  TT_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tmp, in, out, n_plus_1, st));
  TT_CUDA(ctx->cub_tmp.ensure(tmp));
  TT_CUDA(cub::DeviceScan::ExclusiveSum(ctx->cub_tmp.p, tmp, in, out, n_plus_1, st));
  ctx->launches += 2;  // CUB scan: init + scan kernel
  return TT_OK;
}
tt_status scan_i32_to_i64(tt_ctx* ctx, const int* in, int64_t* out, int64_t n_plus_1, cudaStream_t st) {
  cub::TransformInputIterator<int64_t, CastI64, const int*> it(in, CastI64());
  size_t tmp = 0;
  TT_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tmp, it, out, n_plus_1, st));
  TT_CUDA(ctx->cub_tmp.ensure(tmp));
  TT_CUDA(cub::DeviceScan::ExclusiveSum(ctx->cub_tmp.p, tmp, it, out, n_plus_1, st));
  ctx->launches += 2;  // CUB scan: init + scan kernel
  return TT_OK;
}
tt_status incl_scan_i32(tt_ctx* ctx, const int* in, int* out, int64_t n, cudaStream_t st) {
  size_t tmp = 0;
  TT_CUDA(cub::DeviceScan::InclusiveSum(nullptr, tmp, in, out, n, st));
  TT_CUDA(ctx->cub_tmp.ensure(tmp));
  TT_CUDA(cub::DeviceScan::InclusiveSum(ctx->cub_tmp.p, tmp, in, out, n, st));
  ctx->launches += 2;  // CUB scan: init + scan kernel
  return TT_OK;
}
// stable LSD radix sort of (key, payload) on bits [0, end_bit); result pointers returned
template <typename V>
tt_status sort_pairs(tt_ctx* ctx, DevBuf (&kb)[2], DevBuf (&vb)[2], int64_t n, int begin_bit, int end_bit,
                     uint64_t** k_out, V** v_out, cudaStream_t st) {
  cub::DoubleBuffer<uint64_t> dk(kb[0].as<uint64_t>(), kb[1].as<uint64_t>());
  cub::DoubleBuffer<V> dv(vb[0].as<V>(), vb[1].as<V>());
  size_t tmp = 0;
  TT_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tmp, dk, dv, n, begin_bit, end_bit, st));
  TT_CUDA(ctx->cub_tmp.ensure(tmp));
  TT_CUDA(cub::DeviceRadixSort::SortPairs(ctx->cub_tmp.p, tmp, dk, dv, n, begin_bit, end_bit, st));
  ctx->launches += 2 + (end_bit - begin_bit + 7) / 8;  // CUB onesweep sort: histogram + exclusive sum + one kernel per 8-bit pass
  *k_out = dk.Current();
  *v_out = dv.Current();
  return TT_OK;
}

// ---- K1 (+ sums): shared by tt_energy and tt_hess_symbolic -------------------------------------
template <typename T>
tt_status run_classify(tt_ctx* ctx, const tt_problem* q, T* e_pp, T* tc, bool record, int* deg, cudaStream_t st, int64_t* nblk_out) {
  const int64_t P = q->n_pairs;
  const int64_t nblk = (P + ttk::CLS_THREADS - 1) / ttk::CLS_THREADS;
  *nblk_out = nblk;
  TT_CUDA(ctx->mask.ensure(sizeof(uint32_t) * (size_t)(nblk * (ttk::CLS_THREADS / 32) + 1)));
  TT_CUDA(ctx->blk_count.ensure(sizeof(int) * (size_t)(nblk + 1)));
  TT_CUDA(ctx->blk_off.ensure(sizeof(int) * (size_t)(nblk + 1)));
  TT_CUDA(ctx->blk_energy.ensure(sizeof(double) * (size_t)(nblk + 1)));
  TT_CUDA(ctx->counts.ensure(sizeof(int64_t) * 16));
  TT_CUDA(ctx->energy.ensure(sizeof(double) * 2));
  if (record) TT_CUDA(ctx->rec.ensure(sizeof(uint16_t) * (size_t)(P + 2)));
  TT_CUDA(cudaMemsetAsync(ctx->blk_count.as<int>() + nblk, 0, sizeof(int), st));
  if (nblk > 0) {
    cudaEvent_t* ev_k1 = ctx->evr[0][ctx->ev_n[0] % tt_ctx::EV_RING];
    TT_CUDA(cudaEventRecord(ev_k1[0], st));
    ttk::k_classify<T><<<(unsigned)nblk, ttk::CLS_THREADS, 0, st>>>(
        (const T*)q->pos, q->tris, (const int2*)q->pairs, P, ctx->opt.tc_scale, ctx->mask.as<uint32_t>(),
        ctx->blk_count.as<int>(), ctx->blk_energy.as<double>(), e_pp, tc, record ? ctx->rec.as<uint16_t>() : nullptr, deg);
    TT_LAUNCH_CHECK();
    TT_CUDA(cudaEventRecord(ev_k1[1], st));
    ctx->ev_n[0]++;
  }
  tt_status s = scan_i32(ctx, ctx->blk_count.as<int>(), ctx->blk_off.as<int>(), nblk + 1, st);
  if (s != TT_OK) return s;
  return TT_OK;
}

// deterministic sum of n partials -> out[0] (two levels above SUM_SLICE values)
template <typename T>
tt_status sum_partials(tt_ctx* ctx, const double* part, int64_t n, T* out, cudaStream_t st) {
  using namespace ttk;
  if (n > 4 * SUM_SLICE) {
    const int64_t ns = (n + SUM_SLICE - 1) / SUM_SLICE;
    TT_CUDA(ctx->sum_stage.ensure(sizeof(double) * (size_t)ns));
    k_sum_stage<<<(unsigned)ns, 256, 0, st>>>(part, n, ctx->sum_stage.as<double>());
    TT_LAUNCH_CHECK();
    part = ctx->sum_stage.as<double>();
    n = ns;
  }
  k_sum_partials<T><<<1, 1024, 0, st>>>(part, n, 1.0, out);
  TT_LAUNCH_CHECK();
  return TT_OK;
}

template <typename T>
tt_status energy_impl(tt_ctx* ctx, const tt_problem* q, void* energy_sum, void* e_pp, uint32_t* active_mask,
                      void* tc, int64_t* n_active, cudaStream_t st) {
  int64_t nblk = 0;
  tt_status s = validate_indices(ctx, q->tris, q->n_tris, q->n_verts, q->pairs, q->n_pairs, st);
  if (s != TT_OK) return s;
  s = run_classify<T>(ctx, q, (T*)e_pp, (T*)tc, false, nullptr, st, &nblk);
  if (s != TT_OK) return s;
  s = sum_partials<T>(ctx, ctx->blk_energy.as<double>(), nblk, (T*)energy_sum, st);
  if (s != TT_OK) return s;
  if (n_active) {
    ttk::k_set_count<<<1, 32, 0, st>>>(ctx->blk_off.as<int>(), ctx->blk_count.as<int>(), nblk, n_active, nullptr);
    TT_LAUNCH_CHECK();
  }
  if (active_mask && q->n_pairs > 0)
    TT_CUDA(cudaMemcpyAsync(active_mask, ctx->mask.p, sizeof(uint32_t) * (size_t)((q->n_pairs + 31) / 32),
                            cudaMemcpyDeviceToDevice, st));
  return TT_OK;
}

// ---- tt_energy_static: K1's energy / active count with the scratch in tt_static_scratch; allocates nothing ---------
// The variant of k_classify that keeps only what the total needs: same gather, same Moeller intervals, same per-pair
// energy, same CTA size and the same fixed-order CTA tree, so its per-CTA partials are the ones k_classify writes and
// the two-level final sum below is sum_partials' -- the result is bit-identical to tt_energy's.
template <typename T>
__global__ void __launch_bounds__(ttk::CLS_THREADS, TT_CLS_MIN_CTAS)
k_energy_static(const T* __restrict__ pos, const int* __restrict__ tris, const int2* __restrict__ pairs, int64_t P,
                double sigma, double* __restrict__ blk_energy, int* __restrict__ blk_count) {
  using namespace ttk;
  __shared__ double s_e[CLS_THREADS / 32];
  __shared__ int s_c[CLS_THREADS / 32];
  const int64_t k = (int64_t)blockIdx.x * CLS_THREADS + threadIdx.x;
  bool active = false;
  double en = 0.0;
  if (k < P) {
    const int2 pr = __ldg(pairs + k);
    int va[3], vb[3];
    d3 a[3], b[3];
    if (gather_pair(pos, tris, pr.x, pr.y, va, vb, a, b)) {
      ttg::PairGeom g;
      active = ttg::pair_intervals(a[0], a[1], a[2], b[0], b[1], b[2], sigma, g);
      if (active) {
        const double pr2 = g.tc0 * g.tc1;
        en = pr2 * pr2;  // Eq. 2
      }
    }
  }
  const uint32_t bal = __ballot_sync(0xffffffffu, active);
  if ((threadIdx.x & 31) == 0) s_c[threadIdx.x >> 5] = __popc(bal);
  const double e = block_sum<CLS_THREADS>(en, s_e);  // its barrier also orders s_c
  if (threadIdx.x == 0) {
    int c = 0;
#pragma unroll
    for (int i = 0; i < CLS_THREADS / 32; ++i) c += s_c[i];
    blk_count[blockIdx.x] = c;
    blk_energy[blockIdx.x] = e;
  }
}
// one CTA: n_active = sum of the per-CTA counts (integers: any order gives the same result)
__global__ void __launch_bounds__(1024) k_count_static(const int* __restrict__ blk_count, int64_t n, int64_t* __restrict__ out) {
  __shared__ long long s[32];
  long long v = 0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) v += blk_count[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    v = s[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (threadIdx.x == 0) out[0] = (int64_t)v;
  }
}
template <typename T>
tt_status energy_static_impl(tt_ctx* ctx, const tt_problem* q, void* energy_sum, int64_t* n_active, cudaStream_t st) {
  using namespace ttk;
  const int64_t P = q->n_pairs;
  const int64_t nblk = (P + CLS_THREADS - 1) / CLS_THREADS;
  double* blk_energy = ctx->static_scratch;
  double* stage = blk_energy + TT_STATIC_MAX_BLK;
  int* blk_count = reinterpret_cast<int*>(stage + TT_STATIC_MAX_STAGE);
  if (nblk > 0) {
    k_energy_static<T><<<(unsigned)nblk, CLS_THREADS, 0, st>>>((const T*)q->pos, q->tris, (const int2*)q->pairs, P, ctx->opt.tc_scale,
                                                                blk_energy, blk_count);
    TT_LAUNCH_CHECK();
  }
  const double* part = blk_energy;
  int64_t n = nblk;
  if (n > 4 * SUM_SLICE) {  // the same two levels as sum_partials
    const int64_t ns = (n + SUM_SLICE - 1) / SUM_SLICE;
    k_sum_stage<<<(unsigned)ns, 256, 0, st>>>(part, n, stage);
    TT_LAUNCH_CHECK();
    part = stage;
    n = ns;
  }
  k_sum_partials<T><<<1, 1024, 0, st>>>(part, n, 1.0, (T*)energy_sum);
  TT_LAUNCH_CHECK();
  if (n_active) {
    k_count_static<<<1, 1024, 0, st>>>(blk_count, nblk, n_active);
    TT_LAUNCH_CHECK();
  }
  return TT_OK;
}

// 0 beyond 3 * n_touched (still on the device): the scan of the general-row lengths runs over the host-known bound
struct MaskedLen {
  const int64_t* tlen;
  const int* n_slots;
  __host__ __device__ int64_t operator()(int64_t i) const { return i < 3 * (int64_t)(*n_slots) ? tlen[i] : 0; }
};
struct DegFlag {
  const int* deg;
  __host__ __device__ int operator()(int t) const { return deg[t] > 0 ? 1 : 0; }
};

template <typename T>
tt_status symbolic_impl(tt_ctx* ctx, const tt_problem* q, int64_t* nnzb_host, int64_t* n_active_host,
                        cudaStream_t st) {
  using namespace ttk;
  ctx->sig.valid = false;
  const int64_t P = q->n_pairs, nT = q->n_tris, nV = q->n_verts;
  int64_t nblk = 0;
  tt_status s = validate_indices(ctx, q->tris, nT, nV, q->pairs, P, st);
  if (s != TT_OK) return s;
  s = pos_checksum(ctx, q, 0, st);
  if (s != TT_OK) return s;
  ctx->bitsV = ceil_log2(nV > 1 ? nV : 2);
  const int bitsV = ctx->bitsV;
  // Everything up to the pattern sizes is enqueued WITHOUT a host round trip: buffers and grids use the
  // bounds  directed entries <= 2 P,  touched triangles <= min(nT, 2 P),  slots <= touched + entries / 8
  // (a part ends where its segment ends -- twice per split triangle, which has > 32 entries -- or where a
  // round is full -- once per 32 entries),  and the kernels read the true counts from device memory.
  // One synchronisation (below) then brings all counts to the host.
  const int64_t n_ub = 2 * P;
  const int64_t touched_ub = nT < n_ub ? nT : n_ub;
  const int64_t slots_ub = touched_ub + n_ub / 8 + 8;
  // ---- one zeroed block: deg [nT+1], vcnt [nV+1], rowlen [nV+1], fill [nT+1] ----
  const size_t zints = (size_t)(nT + 1) + 2 * (size_t)(nV + 1) + (size_t)(nT + 1);
  TT_CUDA(ctx->zero_blk.ensure(sizeof(int) * zints));
  TT_CUDA(cudaMemsetAsync(ctx->zero_blk.p, 0, sizeof(int) * zints, st));
  int* deg = ctx->zero_blk.as<int>();
  int* vcnt = deg + (nT + 1);
  int* rowlen = vcnt + (nV + 1);
  int* fill = rowlen + (nV + 1);
  ctx->vcnt_p = vcnt;
  ctx->rowlen_p = rowlen;
  // ---- K1: classification, recorded decisions, degree histogram ----
  s = run_classify<T>(ctx, q, nullptr, nullptr, true, deg, st, &nblk);
  if (s != TT_OK) return s;
  int64_t* d_counts = ctx->counts.as<int64_t>();
  k_set_count<<<1, 32, 0, st>>>(ctx->blk_off.as<int>(), ctx->blk_count.as<int>(), nblk, d_counts, nullptr);
  TT_LAUNCH_CHECK();
  // ---- layout order of the entry segments (k_bucket_order), segment starts in that order, then by triangle id ----
  TT_CUDA(ctx->tptr.ensure(sizeof(int) * (size_t)(nT + 2)));
  TT_CUDA(ctx->order.ensure(sizeof(int) * (size_t)(nT + 2)));
  TT_CUDA(ctx->degp.ensure(sizeof(int) * (size_t)(nT + 2)));
  TT_CUDA(ctx->tptrp.ensure(sizeof(int) * (size_t)(nT + 2)));
  {
    const int64_t n_ord = (nT + ORD_BUCKET - 1) / ORD_BUCKET + 1;   // + the thread that closes degp
    k_bucket_order<<<grid_for(n_ord, 64), 64, 0, st>>>(deg, nT, d_counts, ctx->order.as<int>(), ctx->degp.as<int>());
    TT_LAUNCH_CHECK();
  }
  s = scan_i32(ctx, ctx->degp.as<int>(), ctx->tptrp.as<int>(), nT + 1, st);  // tptrp[nT] = directed entries = 2 A
  if (s != TT_OK) return s;
  k_scatter_tptr<<<grid_for(nT + 1, 256), 256, 0, st>>>(ctx->tptrp.as<int>(), ctx->order.as<int>(), nT, ctx->tptr.as<int>());
  TT_LAUNCH_CHECK();
  // ---- K2: compaction + counting-sort scatter of the directed entries by source triangle ----
  TT_CUDA(ctx->active_ids.ensure(sizeof(int) * (size_t)(P + 1)));
  TT_CUDA(ctx->ent_in.ensure(sizeof(uint2) * (size_t)(n_ub + 1)));
  TT_CUDA(ctx->partner.ensure(sizeof(int) * (size_t)(n_ub + 1)));
  TT_CUDA(ctx->dvals.ensure(sizeof(uint16_t) * (size_t)(n_ub + 2)));
  if (nblk > 0) {
    k_compact<<<(unsigned)nblk, CLS_THREADS, 0, st>>>(ctx->mask.as<uint32_t>(), ctx->blk_off.as<int>(), P, ctx->active_ids.as<int>(),
                                                      (const int2*)q->pairs, ctx->rec.as<uint16_t>(), ctx->tptr.as<int>(),
                                                      ctx->ent_in.as<uint2>(), fill);
    TT_LAUNCH_CHECK();
  }
  // ---- touched triangles, vertex use counts, the work partition (slots, rounds) shared by the symbolic
  //      round kernels, K4 and K6 ----
  TT_CUDA(ctx->touched.ensure(sizeof(int) * (size_t)(nT + 1)));
  TT_CUDA(ctx->tfirst.ensure(sizeof(int) * (size_t)(touched_ub + 2)));
  TT_CUDA(ctx->tsplit.ensure(sizeof(int) * (size_t)(touched_ub + 1)));
  TT_CUDA(ctx->sfirst.ensure(sizeof(int) * (size_t)(slots_ub + 2)));
  TT_CUDA(ctx->sinfo.ensure(sizeof(int4) * (size_t)(slots_ub + 1)));
  TT_CUDA(ctx->rdesc.ensure(sizeof(int4) * (size_t)(slots_ub + 1)));
  TT_CUDA(ctx->long_list.ensure(sizeof(int) * (size_t)(n_ub / (RND_MAX_ENT + 1) + 2)));
  TT_CUDA(ctx->split_list.ensure(sizeof(int4) * (size_t)(n_ub / (RND_MAX_ENT + 1) + 2)));
  const int64_t buckets_ub = (touched_ub + CHK_BUCKET - 1) / CHK_BUCKET;
  TT_CUDA(ctx->bucket_cnt.ensure(sizeof(PackCount) * (size_t)(buckets_ub + 1)));
  TT_CUDA(ctx->bucket_off.ensure(sizeof(PackCount) * (size_t)(buckets_ub + 1)));
  TT_CUDA(ctx->erank.ensure(sizeof(int) * (size_t)(3 * n_ub + 3)));
  TT_CUDA(ctx->everts.ensure(sizeof(int) * 6 * (size_t)(n_ub + 1)));
  TT_CUDA(ctx->drank.ensure(sizeof(int) * (size_t)(3 * slots_ub + 3)));
  TT_CUDA(ctx->tlen.ensure(sizeof(int64_t) * (size_t)(3 * slots_ub + 1)));
  TT_CUDA(ctx->toff.ensure(sizeof(int64_t) * (size_t)(3 * slots_ub + 2)));
  TT_CUDA(ctx->slot_excl.ensure((size_t)(3 * slots_ub + 1)));
  TT_CUDA(ctx->rowbase.ensure(sizeof(int64_t) * (size_t)(3 * slots_ub + 1)));
  TT_CUDA(ctx->vslot1.ensure(sizeof(int) * (size_t)(nV + 1)));
  TT_CUDA(ctx->rowptr64.ensure(sizeof(int64_t) * (size_t)(nV + 1)));
  TT_CUDA(ctx->rowptr.ensure(sizeof(int) * (size_t)(nV + 1)));
  int* d_num = reinterpret_cast<int*>(d_counts + 1);                              // n_touched
  PackCount* d_tot = ctx->bucket_off.as<PackCount>() + buckets_ub;                // totals of the scan
  TT_CUDA(cudaMemsetAsync(d_num, 0, sizeof(int), st));
  TT_CUDA(cudaMemsetAsync(ctx->bucket_cnt.p, 0, sizeof(PackCount) * (size_t)(buckets_ub + 1), st));
  const int force_general = (ctx->opt.flags & TT_FLAG_FORCE_GENERAL_ROWS) ? 1 : 0;
  if (touched_ub > 0) {
    k_vertex_touch<<<grid_for(nT, 256), 256, 0, st>>>(q->tris, deg, nT, vcnt);
    TT_LAUNCH_CHECK();
    // touched triangles in LAYOUT order: the ids at the positions whose degree is not zero
    cub::CountingInputIterator<int> iota(0);
    cub::TransformInputIterator<int, DegFlag, cub::CountingInputIterator<int>> flags(iota, DegFlag{ctx->degp.as<int>()});
    const int* ord = ctx->order.as<int>();
    size_t tmp = 0;
    TT_CUDA(cub::DeviceSelect::Flagged(nullptr, tmp, ord, flags, ctx->touched.as<int>(), d_num, (int)nT, st));
    TT_CUDA(ctx->cub_tmp.ensure(tmp));
    TT_CUDA(cub::DeviceSelect::Flagged(ctx->cub_tmp.p, tmp, ord, flags, ctx->touched.as<int>(), d_num, (int)nT, st));
    ctx->launches += 2;  // CUB select: init + sweep kernel
    k_touched_first<<<grid_for(touched_ub + 1, 256), 256, 0, st>>>(ctx->touched.as<int>(), d_num, ctx->tptr.as<int>(), nT,
                                                                   ctx->tfirst.as<int>());
    TT_LAUNCH_CHECK();
    const int64_t prep_pers = (int64_t)ctx->sms * 8;
    const int64_t prep_full = (touched_ub + 32 * SYM_WARPS - 1) / (32 * SYM_WARPS);
    if (n_ub > RND_MAX_ENT) {  // long triangles: segment sort + can it be split into parts?
      k_long_prep<<<(unsigned)(prep_full < prep_pers ? prep_full : prep_pers), 32 * SYM_WARPS, 0, st>>>(
          q->tris, ctx->touched.as<int>(), d_num, ctx->tfirst.as<int>(), ctx->ent_in.as<uint2>(), vcnt, force_general,
          ctx->partner.as<int>(), ctx->dvals.as<uint16_t>(), ctx->tsplit.as<int>());
      TT_LAUNCH_CHECK();
    }
    k_chunk_pack<false><<<grid_for(buckets_ub, 128), 128, 0, st>>>(ctx->touched.as<int>(), ctx->tfirst.as<int>(), d_num, ctx->tsplit.as<int>(),
                                                                  ctx->bucket_cnt.as<PackCount>(), nullptr, nullptr, nullptr,
                                                                  nullptr, nullptr, nullptr);
    TT_LAUNCH_CHECK();
    {
      size_t tmp2 = 0;
      const PackCount zero{0, 0, 0, 0, 0};
      TT_CUDA(cub::DeviceScan::ExclusiveScan(nullptr, tmp2, ctx->bucket_cnt.as<PackCount>(), ctx->bucket_off.as<PackCount>(),
                                             PackAdd(), zero, buckets_ub + 1, st));
      TT_CUDA(ctx->cub_tmp.ensure(tmp2));
      TT_CUDA(cub::DeviceScan::ExclusiveScan(ctx->cub_tmp.p, tmp2, ctx->bucket_cnt.as<PackCount>(), ctx->bucket_off.as<PackCount>(),
                                             PackAdd(), zero, buckets_ub + 1, st));
      ctx->launches += 2;
    }
    k_chunk_pack<true><<<grid_for(buckets_ub, 128), 128, 0, st>>>(ctx->touched.as<int>(), ctx->tfirst.as<int>(), d_num, ctx->tsplit.as<int>(), nullptr,
                                                                 ctx->bucket_off.as<PackCount>(), ctx->rdesc.as<int4>(),
                                                                 ctx->long_list.as<int>(), ctx->sfirst.as<int>(),
                                                                 ctx->sinfo.as<int4>(), ctx->split_list.as<int4>());
    TT_LAUNCH_CHECK();
    // ---- per-slot segment sort, column ranks, exclusive rows, general-row workspace sizes
    //      (persistent grids: the round / long-triangle counts are read on the device) ----
    const int64_t rounds_ub = (slots_ub + RSYM_WARPS - 1) / RSYM_WARPS;
    const int64_t sym_pers = (int64_t)ctx->sms * 16;
    k_round_symbolic<<<(unsigned)(rounds_ub < sym_pers ? rounds_ub : sym_pers), 32 * RSYM_WARPS, 0, st>>>(
        q->tris, ctx->touched.as<int>(), ctx->rdesc.as<int4>(), &d_tot->rounds, ctx->tfirst.as<int>(), ctx->sfirst.as<int>(),
        ctx->sinfo.as<int4>(), ctx->tsplit.as<int>(), ctx->ent_in.as<uint2>(), vcnt, force_general, ctx->partner.as<int>(),
        ctx->dvals.as<uint16_t>(), ctx->erank.as<int>(), ctx->drank.as<int>(), rowlen, ctx->tlen.as<int64_t>(),
        ctx->slot_excl.as<uint8_t>(), ctx->everts.as<int>(), ctx->vslot1.as<int>());
    TT_LAUNCH_CHECK();
    const int64_t long_ub = n_ub / (RND_MAX_ENT + 1);
    if (long_ub > 0) {  // long triangles that could not be split: one warp per triangle
      const int64_t lg = (long_ub + SYM_WARPS - 1) / SYM_WARPS;
      const int64_t lpers = (int64_t)ctx->sms * 8;
      k_tri_symbolic<<<(unsigned)(lg < lpers ? lg : lpers), 32 * SYM_WARPS, 0, st>>>(
          q->tris, ctx->touched.as<int>(), &d_tot->longs, ctx->tfirst.as<int>(), ctx->sinfo.as<int4>(), ctx->partner.as<int>(),
          ctx->dvals.as<uint16_t>(), vcnt, force_general, ctx->erank.as<int>(), ctx->drank.as<int>(), rowlen,
          ctx->tlen.as<int64_t>(), ctx->slot_excl.as<uint8_t>(), ctx->long_list.as<int>(), ctx->rdesc.as<int4>(),
          ctx->vslot1.as<int>(), ctx->everts.as<int>());
      TT_LAUNCH_CHECK();
    }
  }
  {  // general-row workspace offsets: scan over the bound, lengths beyond 3 n_slots read as 0
    cub::CountingInputIterator<int64_t> idx(0);
    cub::TransformInputIterator<int64_t, MaskedLen, cub::CountingInputIterator<int64_t>> it(idx, MaskedLen{ctx->tlen.as<int64_t>(), &d_tot->slots});
    size_t tmp = 0;
    TT_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tmp, it, ctx->toff.as<int64_t>(), 3 * slots_ub + 1, st));
    TT_CUDA(ctx->cub_tmp.ensure(tmp));
    TT_CUDA(cub::DeviceScan::ExclusiveSum(ctx->cub_tmp.p, tmp, it, ctx->toff.as<int64_t>(), 3 * slots_ub + 1, st));
    ctx->launches += 2;
  }
  // The row-pointer scan is issued speculatively: if there are no general rows (R == 0: always, in a
  // soup) the exclusive row lengths are already final and nnzb arrives in the same host round trip.
  s = scan_i32_to_i64(ctx, rowlen, ctx->rowptr64.as<int64_t>(), nV + 1, st);
  if (s != TT_OK) return s;
  // ---- the ONE host round trip of the phase (soup; general rows add the merge pass below) ----
  int64_t A = 0, R = 0, nnzb = 0;
  int ntch = 0;
  PackCount tot{0, 0, 0, 0, 0};
  TT_CUDA(cudaMemcpyAsync(&A, d_counts, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaMemcpyAsync(&ntch, d_num, sizeof(int), cudaMemcpyDeviceToHost, st));
  if (touched_ub > 0) TT_CUDA(cudaMemcpyAsync(&tot, d_tot, sizeof(PackCount), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaMemcpyAsync(&R, ctx->toff.as<int64_t>() + 3 * slots_ub, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaMemcpyAsync(&nnzb, ctx->rowptr64.as<int64_t>() + nV, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaStreamSynchronize(st));
  const int64_t n = 2 * A;
  const int64_t n_touched = touched_ub > 0 ? ntch : 0, n_chunks = tot.rounds, n_long = tot.longs, n_slots = tot.slots;
  ctx->n_slots = n_slots;
  ctx->n_split = tot.splits;
  ctx->n_parts = tot.parts;
  ctx->A = A;
  ctx->n_dir = n;
  ctx->n_touched = n_touched;
  ctx->n_chunks = n_chunks;
  ctx->n_long = n_long;
  ctx->tri_limit = round_tri_limit(n, n_touched);  // what k_chunk_pack packed with (same rule, same integers)
  if (R >= (int64_t(1) << 31)) return fail(ctx, TT_ERR_INVALID_ARG, "general-row workspace exceeds 2^31 blocks");
  ctx->R = R;
  const unsigned tri_grid = grid_for(n_slots, SYM_WARPS);
  const unsigned rnd_grid = grid_for(n_chunks, RSYM_WARPS);

  // ---- general rows: merge records sorted by (row, col) ----
  int64_t U = 0;
  ctx->rkeys_sorted = nullptr;
  ctx->rvals_sorted = nullptr;
  if (R > 0) {
    for (int i = 0; i < 2; ++i) {
      TT_CUDA(ctx->rkeys[i].ensure(sizeof(uint64_t) * (size_t)R));
      TT_CUDA(ctx->rvals[i].ensure(sizeof(uint32_t) * (size_t)R));
    }
    TT_CUDA(ctx->head.ensure(sizeof(int) * (size_t)R));
    TT_CUDA(ctx->ord.ensure(sizeof(int) * (size_t)R));
    TT_CUDA(ctx->rowfirst.ensure(sizeof(int) * (size_t)(nV + 1)));
    TT_CUDA(ctx->run_start.ensure(sizeof(int) * (size_t)(R + 1)));
    TT_CUDA(ctx->run_dest.ensure(sizeof(int) * (size_t)(R + 1)));
    k_emit_records<<<tri_grid, 32 * SYM_WARPS, 0, st>>>(
        q->tris, ctx->touched.as<int>(), n_slots, ctx->sfirst.as<int>(), ctx->sinfo.as<int4>(), ctx->partner.as<int>(), bitsV,
        ctx->erank.as<int>(), ctx->drank.as<int>(), ctx->toff.as<int64_t>(), ctx->slot_excl.as<uint8_t>(),
        ctx->rkeys[0].as<uint64_t>(), ctx->rvals[0].as<uint32_t>());
    TT_LAUNCH_CHECK();
    s = sort_pairs(ctx, ctx->rkeys, ctx->rvals, R, 0, 2 * bitsV, &ctx->rkeys_sorted, &ctx->rvals_sorted, st);
    if (s != TT_OK) return s;
    k_record_heads<<<grid_for(R, 256), 256, 0, st>>>(ctx->rkeys_sorted, R, ctx->head.as<int>());
    TT_LAUNCH_CHECK();
    s = incl_scan_i32(ctx, ctx->head.as<int>(), ctx->ord.as<int>(), R, st);
    if (s != TT_OK) return s;
    k_record_rows<<<grid_for(R, 256), 256, 0, st>>>(ctx->rkeys_sorted, R, bitsV, ctx->head.as<int>(),
                                                    ctx->ord.as<int>(), rowlen,
                                                    ctx->rowfirst.as<int>(), ctx->run_start.as<int>());
    TT_LAUNCH_CHECK();
    // row pointers again: the general rows have added their (deduplicated) lengths
    s = scan_i32_to_i64(ctx, rowlen, ctx->rowptr64.as<int64_t>(), nV + 1, st);
    if (s != TT_OK) return s;
    int u32 = 0;
    TT_CUDA(cudaMemcpyAsync(&u32, ctx->ord.as<int>() + (R - 1), sizeof(int), cudaMemcpyDeviceToHost, st));
    TT_CUDA(cudaMemcpyAsync(&nnzb, ctx->rowptr64.as<int64_t>() + nV, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    TT_CUDA(cudaStreamSynchronize(st));
    U = u32;
  }
  ctx->U = U;
  if (nnzb >= (int64_t(1) << 31)) return fail(ctx, TT_ERR_INVALID_ARG, "nnzb %lld exceeds int32 BSR indexing", (long long)nnzb);
  ctx->nnzb = nnzb;
  k_i64_to_i32<<<grid_for(nV + 1, 256), 256, 0, st>>>(ctx->rowptr64.as<int64_t>(), nV + 1, ctx->rowptr.as<int>());
  TT_LAUNCH_CHECK();
  TT_CUDA(ctx->colind.ensure(sizeof(int) * (size_t)(nnzb + 1)));
  if (U > 0) {
    k_record_dest<<<grid_for(U + 1, 256), 256, 0, st>>>(ctx->rkeys_sorted, U, R, bitsV, ctx->run_start.as<int>(),
                                                        ctx->rowptr.as<int>(), ctx->rowfirst.as<int>(),
                                                        ctx->run_dest.as<int>(), ctx->colind.as<int>());
    TT_LAUNCH_CHECK();
  }
  if (n_chunks > 0) {
    k_round_fill<<<rnd_grid, 32 * RSYM_WARPS, 0, st>>>(
        q->tris, ctx->touched.as<int>(), ctx->rdesc.as<int4>(), n_chunks, ctx->sfirst.as<int>(), ctx->sinfo.as<int4>(),
        ctx->tsplit.as<int>(), ctx->partner.as<int>(),
        ctx->erank.as<int>(), ctx->drank.as<int>(), ctx->toff.as<int64_t>(), ctx->slot_excl.as<uint8_t>(),
        ctx->rowptr.as<int>(), ctx->rowbase.as<int64_t>(), ctx->colind.as<int>());
    TT_LAUNCH_CHECK();
  }
  if (n_long > 0) {
    k_fill_rows<<<grid_for(n_long, SYM_WARPS), 32 * SYM_WARPS, 0, st>>>(
        q->tris, ctx->touched.as<int>(), n_long, ctx->sfirst.as<int>(), ctx->sinfo.as<int4>(), ctx->partner.as<int>(),
        ctx->erank.as<int>(), ctx->drank.as<int>(), ctx->toff.as<int64_t>(), ctx->slot_excl.as<uint8_t>(),
        ctx->rowptr.as<int>(), ctx->rowbase.as<int64_t>(), ctx->colind.as<int>(), ctx->long_list.as<int>(),
        ctx->rdesc.as<int4>());
    TT_LAUNCH_CHECK();
  }

  // ---- per-slot buffers, vertex -> slot incidence ----
  TT_CUDA(ctx->asm_energy.ensure(sizeof(double) * (size_t)(n_chunks + 1)));
  TT_CUDA(ctx->tvals.ensure(sizeof(T) * 9 * (size_t)(R + 1)));
  TT_CUDA(ctx->tslot.ensure(sizeof(T) * 9 * (size_t)(n_slots + 1)));
  TT_CUDA(ctx->dpart.ensure(sizeof(double) * NDIAG * (size_t)(ctx->n_parts + 1)));
  // vertex -> slot incidence: only when some vertex has more than one slot.  R == 0 means every slot
  // is exclusive, hence every touched vertex has exactly one (k_gather3 then reads vslot1 only).
  ctx->vvals_sorted = nullptr;
  if (R > 0) {
    const int64_t nvs = 3 * n_slots;
    for (int i = 0; i < 2; ++i) {
      TT_CUDA(ctx->vkeys[i].ensure(sizeof(uint64_t) * (size_t)(nvs + 1)));
      TT_CUDA(ctx->vvals[i].ensure(sizeof(uint32_t) * (size_t)(nvs + 1)));
    }
    TT_CUDA(ctx->vptr.ensure(sizeof(int) * (size_t)(nV + 2)));
    uint64_t* vkeys_sorted = ctx->vkeys[0].as<uint64_t>();
    ctx->vvals_sorted = ctx->vvals[0].as<uint32_t>();
    k_emit_vslots<<<grid_for(nvs, 256), 256, 0, st>>>(q->tris, ctx->touched.as<int>(), n_slots, ctx->sinfo.as<int4>(),
                                                      ctx->tsplit.as<int>(), nV, ctx->vkeys[0].as<uint64_t>(),
                                                      ctx->vvals[0].as<uint32_t>());
    TT_LAUNCH_CHECK();
    s = sort_pairs(ctx, ctx->vkeys, ctx->vvals, nvs, 0, ceil_log2(nV + 1), &vkeys_sorted, &ctx->vvals_sorted, st);
    if (s != TT_OK) return s;
    k_segment_ptr<<<grid_for(nV + 1, 256), 256, 0, st>>>(vkeys_sorted, nvs, 0, nV, ctx->vptr.as<int>());
    TT_LAUNCH_CHECK();
  }

  ctx->sig.pos = q->pos;
  ctx->sig.tris = q->tris;
  ctx->sig.pairs = q->pairs;
  ctx->sig.nV = nV;
  ctx->sig.nT = nT;
  ctx->sig.P = P;
  ctx->sig.valid = true;
  ctx->rows_gen = U > 0 ? -1 : 0;  // filled lazily by tt_stats if needed
  if (nnzb_host) *nnzb_host = nnzb;
  if (n_active_host) *n_active_host = A;
  return TT_OK;
}

template <typename T>
ttk::AsmParams<T> make_params(tt_ctx* ctx, const tt_problem* q) {
  ttk::AsmParams<T> p;
  p.pos = (const T*)q->pos;
  p.dvals = ctx->dvals.as<uint16_t>();
  p.everts = ctx->everts.as<int>();
  p.rdesc = ctx->rdesc.as<int4>();
  p.tfirst = ctx->sfirst.as<int>();
  p.dpart = ctx->dpart.as<double>();
  p.long_list = ctx->long_list.as<int>();
  p.erank = ctx->erank.as<int>();
  p.drank = ctx->drank.as<int>();
  p.rowbase = ctx->rowbase.as<int64_t>();
  p.vals = nullptr;
  p.tvals = ctx->tvals.as<T>();
  p.tslot = ctx->tslot.as<T>();
  p.chunk_energy = ctx->asm_energy.as<double>();
  p.n_chunks = ctx->n_chunks;
  p.n_long = ctx->n_long;
  p.pvec = nullptr;
  p.hess_mode = ctx->opt.hess_mode;
  p.sigma = ctx->opt.tc_scale;
  return p;
}

// split triangles: parts' partial sums -> the triangle's first slot (+ the diagonal blocks after K4)
template <typename T, bool HESS>
tt_status launch_split_finish(tt_ctx* ctx, const tt_problem* q, T* vals, cudaStream_t st) {
  if (ctx->n_split <= 0) return TT_OK;
  ttk::k_split_finish<T, HESS><<<grid_for(ctx->n_split, 4), 128, 0, st>>>(
      ctx->split_list.as<int4>(), ctx->n_split, q->tris, ctx->touched.as<int>(), ctx->tsplit.as<int>(), ctx->rowptr.as<int>(),
      ctx->dpart.as<double>(), ctx->tslot.as<T>(), vals);
  TT_LAUNCH_CHECK();
  return TT_OK;
}

// K6 launch: pipelined kernel over all rounds (skips long ones) + the plain kernel over the long rounds
template <typename T, int MODE>
tt_status launch_entry_reduce(tt_ctx* ctx, const ttk::AsmParams<T>& p, cudaStream_t st) {
  using namespace ttk;
  const size_t smem = sizeof(PipeWarpSmem<T, MODE>) * PIPE_WARPS;
  const int64_t full = (ctx->n_chunks + PIPE_WARPS - 1) / PIPE_WARPS;
  const int64_t pers = ctx->pipe_grid[sizeof(T) == 8 ? 0 : 1][MODE - 1];
  k_entry_pipe<T, MODE><<<(unsigned)(full < pers ? full : pers), 32 * PIPE_WARPS, smem, st>>>(p);
  TT_LAUNCH_CHECK();
  if (ctx->n_long > 0) {
    k_entry_reduce<T, MODE><<<grid_for(ctx->n_long, RED_THREADS / 32), RED_THREADS, 0, st>>>(p, ctx->long_list.as<int>(), ctx->n_long);
    TT_LAUNCH_CHECK();
  }
  return TT_OK;
}

template <typename T>
tt_status numeric_impl(tt_ctx* ctx, const tt_problem* q, void* energy_sum, void* grad, int32_t* rowptr,
                       int32_t* colind, void* vals, int64_t cap, cudaStream_t st) {
  using namespace ttk;
  const bool want_h = (vals != nullptr);
  if (want_h && (!rowptr || !colind)) return fail(ctx, TT_ERR_INVALID_ARG, "bsr_rowptr/bsr_colind/bsr_vals must be all set or all NULL");
  if (!energy_sum) return fail(ctx, TT_ERR_INVALID_ARG, "energy_sum is NULL");
  if (want_h && cap < ctx->nnzb) return fail(ctx, TT_ERR_CAPACITY, "nnzb_capacity %lld < nnzb %lld", (long long)cap, (long long)ctx->nnzb);
  const int64_t nV = q->n_verts;
  if (want_h) {
    if (rowptr != ctx->rowptr.as<int>())
      TT_CUDA(cudaMemcpyAsync(rowptr, ctx->rowptr.p, sizeof(int) * (size_t)(nV + 1), cudaMemcpyDeviceToDevice, st));
    if (colind != ctx->colind.as<int>() && ctx->nnzb > 0)
      TT_CUDA(cudaMemcpyAsync(colind, ctx->colind.p, sizeof(int) * (size_t)ctx->nnzb, cudaMemcpyDeviceToDevice, st));
  }
  AsmParams<T> p = make_params<T>(ctx, q);
  p.vals = (T*)vals;
  if (ctx->n_chunks > 0) {
    cudaEvent_t* ev_k4 = ctx->evr[1][ctx->ev_n[1] % tt_ctx::EV_RING];
    TT_CUDA(cudaEventRecord(ev_k4[0], st));
    if (want_h && ctx->opt.hess_mode == TT_HESS_EXACT) {
      // the exact Hessian (tt_exact.cuh): one kernel over every round, same partition, ranks and row bases
      k_assemble_exact<T><<<grid_for(ctx->n_chunks, EX_WARPS), 32 * EX_WARPS, 0, st>>>(p);
      TT_LAUNCH_CHECK();
      tt_status s2 = launch_split_finish<T, true>(ctx, q, (T*)vals, st);
      if (s2 != TT_OK) return s2;
    } else if (want_h) {
      const bool wide = ctx->tri_limit > RND_TRI_LOW;  // which instantiation: per-slot loops unrolled 16 or 8 deep
      const size_t smem = (wide ? sizeof(TileWarpSmem<T, RND_MAX_TRI>) : sizeof(TileWarpSmem<T, RND_TRI_LOW>)) * TILE_WARPS;
      const int64_t full = (ctx->n_chunks + TILE_WARPS - 1) / TILE_WARPS;
      const int64_t pers = ctx->tile_grid[sizeof(T) == 8 ? 0 : 1][wide ? 1 : 0];
      const unsigned grid = (unsigned)(full < pers ? full : pers);
      const bool proj = ctx->opt.hess_mode == TT_HESS_PSDPROJ, parts = ctx->n_parts > 0;
      const int which = (proj ? 4 : 0) | (parts ? 2 : 0) | (wide ? 1 : 0);
      switch (which) {
        case 0: k_assemble_tile<T, false, false, RND_TRI_LOW><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        case 1: k_assemble_tile<T, false, false, RND_MAX_TRI><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        case 2: k_assemble_tile<T, false, true, RND_TRI_LOW><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        case 3: k_assemble_tile<T, false, true, RND_MAX_TRI><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        case 4: k_assemble_tile<T, true, false, RND_TRI_LOW><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        case 5: k_assemble_tile<T, true, false, RND_MAX_TRI><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        case 6: k_assemble_tile<T, true, true, RND_TRI_LOW><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
        default: k_assemble_tile<T, true, true, RND_MAX_TRI><<<grid, 32 * TILE_WARPS, smem, st>>>(p); break;
      }
      if (ctx->n_long > 0) {
        TT_LAUNCH_CHECK();
        k_assemble_long_tile<T, true><<<(unsigned)ctx->n_long, 32, sizeof(LongTileSmem<T, true>), st>>>(p);
        TT_LAUNCH_CHECK();
        k_assemble_long_tile<T, false><<<(unsigned)ctx->n_long, 32, sizeof(LongTileSmem<T, false>), st>>>(p);
        TT_LAUNCH_CHECK();
        k_assemble_long_direct<T><<<grid_for(ctx->n_long, TILE_WARPS), 32 * TILE_WARPS, sizeof(LongWarpSmem) * TILE_WARPS, st>>>(p);
      }
      TT_LAUNCH_CHECK();
      tt_status s2 = launch_split_finish<T, true>(ctx, q, (T*)vals, st);
      if (s2 != TT_OK) return s2;
    } else {
      tt_status s1 = launch_entry_reduce<T, 1>(ctx, p, st);
      if (s1 != TT_OK) return s1;
      s1 = launch_split_finish<T, false>(ctx, q, (T*)nullptr, st);
      if (s1 != TT_OK) return s1;
    }
    TT_CUDA(cudaEventRecord(ev_k4[1], st));
    ctx->ev_n[1]++;
    if (want_h && ctx->U > 0) {
      k_merge<T><<<grid_for(9 * ctx->U, 256), 256, 0, st>>>(ctx->run_start.as<int>(), ctx->run_dest.as<int>(),
                                                            ctx->rvals_sorted, ctx->U, ctx->tvals.as<T>(), (T*)vals);
      TT_LAUNCH_CHECK();
    }
  }
  if (grad && nV > 0) {
    k_gather3<T><<<grid_for(nV, 256), 256, 0, st>>>(ctx->vcnt_p, ctx->vslot1.as<int>(), ctx->vptr.as<int>(), ctx->vvals_sorted, nV, ctx->tslot.as<T>(), (T*)grad);
    TT_LAUNCH_CHECK();
  }
  return sum_partials<T>(ctx, ctx->asm_energy.as<double>(), ctx->n_chunks, (T*)energy_sum, st);
}

template <typename T>
tt_status hessvec_impl(tt_ctx* ctx, const tt_problem* q, const void* pvec, void* y, cudaStream_t st) {
  using namespace ttk;
  AsmParams<T> p = make_params<T>(ctx, q);
  p.pvec = (const T*)pvec;
  p.chunk_energy = nullptr;
  if (ctx->n_chunks > 0) {
    cudaEvent_t* ev_k6 = ctx->evr[2][ctx->ev_n[2] % tt_ctx::EV_RING];
    TT_CUDA(cudaEventRecord(ev_k6[0], st));
    tt_status s1 = TT_OK;
    if (ctx->opt.hess_mode == TT_HESS_EXACT) {
      k_hess_vec_exact<T><<<grid_for(ctx->n_chunks, RED_THREADS / 32), RED_THREADS, 0, st>>>(p);
      TT_LAUNCH_CHECK();
    } else {
      s1 = launch_entry_reduce<T, 2>(ctx, p, st);
    }
    if (s1 != TT_OK) return s1;
    s1 = launch_split_finish<T, false>(ctx, q, (T*)nullptr, st);
    if (s1 != TT_OK) return s1;
    TT_CUDA(cudaEventRecord(ev_k6[1], st));
    ctx->ev_n[2]++;
  }
  if (q->n_verts > 0) {
    k_gather3<T><<<grid_for(q->n_verts, 256), 256, 0, st>>>(ctx->vcnt_p, ctx->vslot1.as<int>(), ctx->vptr.as<int>(), ctx->vvals_sorted, q->n_verts,
                                                                ctx->tslot.as<T>(), (T*)y);
    TT_LAUNCH_CHECK();
  }
  return TT_OK;
}

// ---- the consumer: BSR product, block-Jacobi, PCG (tt_solve.cuh) ----------------------
template <typename T>
tt_status spmv_impl(tt_ctx* ctx, int64_t nV, const int32_t* rowptr, const int32_t* colind, const void* vals, double shift,
                    const void* x, void* y, cudaStream_t st) {
  if (nV == 0) return TT_OK;
  tts::k_bsr_spmv<T><<<grid_for(32 * nV, tts::VEC_THREADS), tts::VEC_THREADS, 0, st>>>(rowptr, colind, (const T*)vals, (const T*)x,
                                                                                       (T*)y, nV, shift);
  TT_LAUNCH_CHECK();
  return TT_OK;
}

// ---- the membrane term (tt_membrane.cuh, reading A18) ----------------------------------
template <typename T>
tt_status membrane_build_impl(tt_ctx* ctx, const void* rest_pos, int64_t nV, const int32_t* tris, int64_t nT, double k, cudaStream_t st) {
  using namespace ttm;
  ctx->mb_nV = -1;
  const int64_t n6 = 6 * nT;
  TT_CUDA(ctx->mb_ptr.ensure(sizeof(int) * (size_t)(nV + 2)));
  TT_CUDA(ctx->mb_num.ensure(sizeof(int64_t) * 2));
  int64_t n_uniq = 0;
  if (n6 > 0) {
    for (int i = 0; i < 2; ++i) TT_CUDA(ctx->mb_keys[i].ensure(sizeof(unsigned long long) * (size_t)n6));
    k_half_edges<<<grid_for(nT, MB_THREADS), MB_THREADS, 0, st>>>(tris, nT, nV, ctx->mb_keys[0].as<unsigned long long>());
    TT_LAUNCH_CHECK();
    cub::DoubleBuffer<unsigned long long> dk(ctx->mb_keys[0].as<unsigned long long>(), ctx->mb_keys[1].as<unsigned long long>());
    const int end_bit = 32 + ceil_log2(nV + 2);
    size_t tmp = 0;
    TT_CUDA(cub::DeviceRadixSort::SortKeys(nullptr, tmp, dk, n6, 0, end_bit, st));
    TT_CUDA(ctx->cub_tmp.ensure(tmp));
    TT_CUDA(cub::DeviceRadixSort::SortKeys(ctx->cub_tmp.p, tmp, dk, n6, 0, end_bit, st));
    ctx->launches += 2 + (end_bit + 7) / 8;
    unsigned long long* sorted = dk.Current();
    unsigned long long* uniq = dk.Alternate();
    tmp = 0;
    TT_CUDA(cub::DeviceSelect::Unique(nullptr, tmp, sorted, uniq, ctx->mb_num.as<int64_t>(), n6, st));
    TT_CUDA(ctx->cub_tmp.ensure(tmp));
    TT_CUDA(cub::DeviceSelect::Unique(ctx->cub_tmp.p, tmp, sorted, uniq, ctx->mb_num.as<int64_t>(), n6, st));
    ctx->launches += 2;
    TT_CUDA(cudaMemcpyAsync(&n_uniq, ctx->mb_num.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    TT_CUDA(cudaStreamSynchronize(st));
    TT_CUDA(ctx->mb_adj.ensure(sizeof(int) * (size_t)(n_uniq + 1)));
    TT_CUDA(ctx->mb_rest.ensure(sizeof(double) * (size_t)(n_uniq + 1)));
    k_adjacency<T><<<grid_for(n_uniq, MB_THREADS), MB_THREADS, 0, st>>>(uniq, n_uniq, nV, (const T*)rest_pos, ctx->mb_adj.as<int>(),
                                                                          ctx->mb_rest.as<double>());
    TT_LAUNCH_CHECK();
    ttk::k_segment_ptr<<<grid_for(nV + 1, 256), 256, 0, st>>>((const uint64_t*)uniq, n_uniq, 32, nV, ctx->mb_ptr.as<int>());
    TT_LAUNCH_CHECK();
  } else {
    TT_CUDA(cudaMemsetAsync(ctx->mb_ptr.p, 0, sizeof(int) * (size_t)(nV + 2), st));
  }
  TT_CUDA(ctx->mb_part.ensure(sizeof(double) * (size_t)(grid_for(nV > 0 ? nV : 1, MB_THREADS) + 2)));
  ctx->mb_half = n_uniq;
  ctx->mb_k = k;
  ctx->mb_nV = nV;
  return TT_OK;
}
// energy -> e_out[0] (double, device), gradient written or added to grad (may be NULL)
template <typename T>
tt_status membrane_energy_grad_impl(tt_ctx* ctx, const void* pos, double* e_out, void* grad, bool accumulate, cudaStream_t st) {
  using namespace ttm;
  const int64_t nV = ctx->mb_nV;
  const unsigned g = grid_for(nV > 0 ? nV : 1, MB_THREADS);
  k_membrane<T, 0><<<g, MB_THREADS, 0, st>>>((const T*)pos, ctx->mb_ptr.as<int>(), ctx->mb_adj.as<int>(), ctx->mb_rest.as<double>(), nV,
                                             ctx->mb_k, nullptr, 0.0, accumulate ? 1 : 0, (T*)grad, ctx->mb_part.as<double>());
  TT_LAUNCH_CHECK();
  ttk::k_sum_partials<double><<<1, 1024, 0, st>>>(ctx->mb_part.as<double>(), (int64_t)g, 1.0, e_out);
  TT_LAUNCH_CHECK();
  return TT_OK;
}
template <typename T, int MODE>  // 1: y (+)= H_m p;  2: minv = (D + mu I)^-1
tt_status membrane_apply_impl(tt_ctx* ctx, const void* pos, const void* p, double mu, bool accumulate, void* out, cudaStream_t st) {
  using namespace ttm;
  const int64_t nV = ctx->mb_nV;
  if (nV <= 0) return TT_OK;
  k_membrane<T, MODE><<<grid_for(nV, MB_THREADS), MB_THREADS, 0, st>>>((const T*)pos, ctx->mb_ptr.as<int>(), ctx->mb_adj.as<int>(),
                                                                          ctx->mb_rest.as<double>(), nV, ctx->mb_k, (const T*)p, mu,
                                                                          accumulate ? 1 : 0, (T*)out, nullptr);
  TT_LAUNCH_CHECK();
  return TT_OK;
}

template <typename T>
tt_status pcg_impl(tt_ctx* ctx, const tt_problem* q, const int32_t* rowptr, const int32_t* colind, const void* vals,
                   const void* minv, const void* b, void* x, const tt_pcg_options* opt, int32_t* iters_host,
                   double* relres_host, cudaStream_t st, bool membrane = false) {
  using namespace tts;
  const int64_t nV = q->n_verts, n = 3 * nV;
  const bool matrix_free = (vals == nullptr);
  if (iters_host) *iters_host = 0;
  if (relres_host) *relres_host = 0.0;
  if (nV == 0) return TT_OK;
  const unsigned gv = grid_for(nV, VEC_THREADS), gn = grid_for(n, VEC_THREADS);
  TT_CUDA(ctx->pcg_r.ensure(sizeof(T) * (size_t)n));
  TT_CUDA(ctx->pcg_p.ensure(sizeof(T) * (size_t)n));
  TT_CUDA(ctx->pcg_q.ensure(sizeof(T) * (size_t)n));
  for (int i = 0; i < 2; ++i) TT_CUDA(ctx->pcg_part[i].ensure(sizeof(double) * (size_t)(gn + 1)));
  TT_CUDA(ctx->pcg_sc.ensure(sizeof(PcgScalars)));
  TT_CUDA(ctx->pcg_hist.ensure(sizeof(double) * (size_t)(opt->max_iter + 2)));
  T* r = ctx->pcg_r.as<T>();
  T* p = ctx->pcg_p.as<T>();
  T* Ap = ctx->pcg_q.as<T>();
  double* part0 = ctx->pcg_part[0].as<double>();
  double* part1 = ctx->pcg_part[1].as<double>();
  PcgScalars* sc = ctx->pcg_sc.as<PcgScalars>();
  double* hist = ctx->pcg_hist.as<double>();
  k_pcg_init<T><<<gv, VEC_THREADS, 0, st>>>((const T*)b, (const T*)minv, nV, (T*)x, r, p, part0, part1);
  TT_LAUNCH_CHECK();
  k_pcg_init_final<<<1, 1024, 0, st>>>(part0, part1, (int64_t)gv, opt->rtol, sc, hist);
  TT_LAUNCH_CHECK();
  const int check_every = opt->rtol > 0.0 ? (opt->check_every > 0 ? opt->check_every : 8) : 0;
  PcgScalars h;
  for (int it = 0; it < opt->max_iter; ++it) {
    tt_status s = matrix_free ? hessvec_impl<T>(ctx, q, p, Ap, st) : spmv_impl<T>(ctx, nV, rowptr, colind, vals, opt->shift, p, Ap, st);
    if (s != TT_OK) return s;
    if (membrane) {  // + H_m p (tt_membrane.cuh)
      s = membrane_apply_impl<T, 1>(ctx, q->pos, p, 0.0, true, Ap, st);
      if (s != TT_OK) return s;
    }
    k_pcg_pq<T><<<gn, VEC_THREADS, 0, st>>>(p, Ap, n, opt->shift, matrix_free ? 1 : 0, part0);
    TT_LAUNCH_CHECK();
    k_pcg_alpha<<<1, 1024, 0, st>>>(part0, (int64_t)gn, sc);
    TT_LAUNCH_CHECK();
    k_pcg_update<T><<<gv, VEC_THREADS, 0, st>>>(p, Ap, (const T*)minv, nV, (T*)x, r, sc, part0, part1);
    TT_LAUNCH_CHECK();
    k_pcg_beta<<<1, 1024, 0, st>>>(part0, part1, (int64_t)gv, sc, hist);
    TT_LAUNCH_CHECK();
    k_pcg_dir<T><<<gn, VEC_THREADS, 0, st>>>(Ap, p, n, sc);
    TT_LAUNCH_CHECK();
    if (check_every && (it + 1) % check_every == 0 && it + 1 < opt->max_iter) {  // the device has already frozen x if converged
      TT_CUDA(cudaMemcpyAsync(&h, sc, sizeof(h), cudaMemcpyDeviceToHost, st));
      TT_CUDA(cudaStreamSynchronize(st));
      if (h.done) break;
    }
  }
  if (iters_host || relres_host) {
    TT_CUDA(cudaMemcpyAsync(&h, sc, sizeof(h), cudaMemcpyDeviceToHost, st));
    TT_CUDA(cudaStreamSynchronize(st));
    if (iters_host) *iters_host = h.iters;
    if (relres_host) *relres_host = h.bb > 0.0 ? sqrt(h.rr / h.bb) : 0.0;
  }
  return TT_OK;
}

// ---- broad phase (tt_broad.cuh) ------------------------------------------------------------------
template <typename T>
tt_status broad_impl(tt_ctx* ctx, const void* pos, int64_t nV, const int32_t* tris, int64_t nT, double inflate,
                     int64_t* n_pairs_host, cudaStream_t st) {
  using namespace ttb;
  ctx->bp_n_pairs = -1;
  *n_pairs_host = 0;
  if (nT < 2) {
    ctx->bp_n_pairs = 0;
    return TT_OK;
  }
  {
    tt_status sv = validate_indices(ctx, tris, nT, nV, nullptr, 0, st);
    if (sv != TT_OK) return sv;
  }
  const unsigned gridT = grid_for(nT, BP_THREADS);
  TT_CUDA(ctx->bp_box.ensure(sizeof(double) * 6 * (size_t)nT));
  TT_CUDA(ctx->bp_part.ensure(sizeof(double) * 8 * (size_t)gridT));
  TT_CUDA(ctx->bp_grid.ensure(sizeof(Grid)));
  TT_CUDA(ctx->bp_cnt.ensure(sizeof(int) * (size_t)(nT + 1)));
  TT_CUDA(ctx->bp_off.ensure(sizeof(int) * (size_t)(nT + 1)));
  k_bp_aabb<T><<<gridT, BP_THREADS, 0, st>>>((const T*)pos, tris, nT, inflate, ctx->bp_box.as<double>(), ctx->bp_part.as<double>());
  TT_LAUNCH_CHECK();
  k_bp_grid<<<1, BP_THREADS, 0, st>>>(ctx->bp_part.as<double>(), (int64_t)gridT, nT, ctx->bp_grid.as<Grid>());
  TT_LAUNCH_CHECK();
  k_bp_cells<false><<<gridT, BP_THREADS, 0, st>>>(ctx->bp_box.as<double>(), nT, ctx->bp_grid.as<Grid>(), ctx->bp_cnt.as<int>(),
                                                  nullptr, nullptr, nullptr);
  TT_LAUNCH_CHECK();
  TT_CUDA(cudaMemsetAsync(ctx->bp_cnt.as<int>() + nT, 0, sizeof(int), st));
  tt_status s = scan_i32(ctx, ctx->bp_cnt.as<int>(), ctx->bp_off.as<int>(), nT + 1, st);
  if (s != TT_OK) return s;
  int n_rec32 = 0;
  Grid g;
  TT_CUDA(cudaMemcpyAsync(&n_rec32, ctx->bp_off.as<int>() + nT, sizeof(int), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaMemcpyAsync(&g, ctx->bp_grid.p, sizeof(Grid), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaStreamSynchronize(st));
  const int64_t n_rec = n_rec32;
  for (int c = 0; c < 3; ++c)
    if (g.dims[c] <= 0 || g.dims[c] > ttb::BP_MAX_DIM)
      return fail(ctx, TT_ERR_INVALID_ARG, "broad phase: invalid grid dimension %d (non-finite positions?)", g.dims[c]);
  const double n_cells = (double)g.dims[0] * (double)g.dims[1] * (double)g.dims[2];
  if (n_cells >= 1.0e14) return fail(ctx, TT_ERR_INVALID_ARG, "broad phase: grid of %d x %d x %d cells exceeds 47-bit cell keys", g.dims[0], g.dims[1], g.dims[2]);
  int cell_bits = 1;
  while (cell_bits < 63 - ttb::BP_QBITS && (double)(1ull << cell_bits) < n_cells) ++cell_bits;
  for (int i = 0; i < 2; ++i) {
    TT_CUDA(ctx->bp_keys[i].ensure(sizeof(uint64_t) * (size_t)(n_rec + 1)));
    TT_CUDA(ctx->bp_vals[i].ensure(sizeof(uint32_t) * (size_t)(n_rec + 1)));
  }
  k_bp_cells<true><<<gridT, BP_THREADS, 0, st>>>(ctx->bp_box.as<double>(), nT, ctx->bp_grid.as<Grid>(), nullptr,
                                                 ctx->bp_off.as<int>(), ctx->bp_keys[0].as<uint64_t>(), ctx->bp_vals[0].as<uint32_t>());
  TT_LAUNCH_CHECK();
  uint64_t* keys = nullptr;
  uint32_t* vals = nullptr;
  s = sort_pairs(ctx, ctx->bp_keys, ctx->bp_vals, n_rec, 0, cell_bits + ttb::BP_QBITS, &keys, &vals, st);
  if (s != TT_OK) return s;
  TT_CUDA(ctx->bp_pcnt.ensure(sizeof(int) * (size_t)(n_rec + 1)));
  TT_CUDA(ctx->bp_poff.ensure(sizeof(int64_t) * (size_t)(n_rec + 1)));
  const unsigned gridR = grid_for(n_rec, BP_THREADS);
  k_bp_pairs<false><<<gridR, BP_THREADS, 0, st>>>(keys, vals, n_rec, ctx->bp_box.as<double>(), tris, nT, ctx->bp_grid.as<Grid>(),
                                                  ctx->bp_pcnt.as<int>(), nullptr, nullptr);
  TT_LAUNCH_CHECK();
  TT_CUDA(cudaMemsetAsync(ctx->bp_pcnt.as<int>() + n_rec, 0, sizeof(int), st));
  s = scan_i32_to_i64(ctx, ctx->bp_pcnt.as<int>(), ctx->bp_poff.as<int64_t>(), n_rec + 1, st);
  if (s != TT_OK) return s;
  int64_t P = 0;
  TT_CUDA(cudaMemcpyAsync(&P, ctx->bp_poff.as<int64_t>() + n_rec, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaStreamSynchronize(st));
  if (P >= (int64_t(1) << 30)) return fail(ctx, TT_ERR_INVALID_ARG, "broad phase: %lld candidate pairs exceed the 2^30 limit of tt_problem", (long long)P);
  for (int i = 0; i < 2; ++i) TT_CUDA(ctx->bp_pkeys[i].ensure(sizeof(uint64_t) * (size_t)(P + 1)));
  TT_CUDA(ctx->bp_pairs.ensure(sizeof(int2) * (size_t)(P + 1)));
  if (P > 0) {
    k_bp_pairs<true><<<gridR, BP_THREADS, 0, st>>>(keys, vals, n_rec, ctx->bp_box.as<double>(), tris, nT, ctx->bp_grid.as<Grid>(),
                                                   nullptr, ctx->bp_poff.as<int64_t>(), ctx->bp_pkeys[0].as<uint64_t>());
    TT_LAUNCH_CHECK();
    cub::DoubleBuffer<uint64_t> dk(ctx->bp_pkeys[0].as<uint64_t>(), ctx->bp_pkeys[1].as<uint64_t>());
    const int bits = 2 * ceil_log2(nT > 1 ? nT : 2);
    size_t tmp = 0;
    TT_CUDA(cub::DeviceRadixSort::SortKeys(nullptr, tmp, dk, P, 0, bits, st));
    TT_CUDA(ctx->cub_tmp.ensure(tmp));
    TT_CUDA(cub::DeviceRadixSort::SortKeys(ctx->cub_tmp.p, tmp, dk, P, 0, bits, st));
    ctx->launches += 2 + (bits + 7) / 8;
    k_bp_unpack<<<grid_for(P, 256), 256, 0, st>>>(dk.Current(), P, nT, ctx->bp_pairs.as<int2>());
    TT_LAUNCH_CHECK();
  }
  ctx->bp_n_pairs = P;
  *n_pairs_host = P;
  return TT_OK;
}


// ---- one Levenberg-Marquardt inexact-Newton step with Armijo backtracking (reading A16) -------------
template <typename T>
tt_status newton_impl(tt_ctx* ctx, void* pos, int64_t nV, const int32_t* tris, int64_t nT, const int32_t* pairs, int64_t P,
                      const tt_newton_options* o, tt_newton_report* rep, cudaStream_t st) {
  using namespace tts;
  std::memset(rep, 0, sizeof(*rep));
  rep->n_pairs = P;
  tt_problem q{pos, nV, tris, nT, pairs, P};
  int64_t nnzb = 0, A = 0;
  tt_status s = symbolic_impl<T>(ctx, &q, &nnzb, &A, st);
  if (s != TT_OK) return s;
  rep->n_active = A;
  rep->nnzb = nnzb;
  if (A == 0 || nV == 0) {  // nothing intersects: the loop's goal is reached (the membrane alone is not relaxed further)
    rep->accepted = 1;
    return TT_OK;
  }
  const int64_t n = 3 * nV;
  const bool mf = o->matrix_free != 0;
  const bool mb = o->membrane != 0;  // E = E_T + E_m (tt_membrane.cuh, reading A18)
  TT_CUDA(ctx->nw_g.ensure(sizeof(T) * (size_t)n));
  TT_CUDA(ctx->nw_d.ensure(sizeof(T) * (size_t)n));
  TT_CUDA(ctx->nw_x.ensure(sizeof(T) * (size_t)n));
  TT_CUDA(ctx->nw_sc.ensure(sizeof(double) * 8));
  if (!mf) TT_CUDA(ctx->nw_vals.ensure(sizeof(T) * 9 * (size_t)(nnzb + 1)));
  if (!mf || mb) TT_CUDA(ctx->nw_minv.ensure(sizeof(T) * 9 * (size_t)nV));
  T* g = ctx->nw_g.as<T>();
  T* d = ctx->nw_d.as<T>();
  T* x_try = ctx->nw_x.as<T>();
  double* sc = ctx->nw_sc.as<double>();        // [0] g.d  [1] g.g
  T* e_dev = reinterpret_cast<T*>(sc + 2);      // [0] E0   [1] E(x_try)
  double* em_dev = sc + 4;                      // [0] E_m(x)  [1] E_m(x_try)   (membrane only)
  int* rowptr = ctx->rowptr.as<int>();
  int* colind = ctx->colind.as<int>();
  T* vals = mf ? nullptr : ctx->nw_vals.as<T>();
  s = numeric_impl<T>(ctx, &q, e_dev, g, mf ? nullptr : rowptr, mf ? nullptr : colind, vals, nnzb, st);
  if (s != TT_OK) return s;
  T* minv = nullptr;
  if (mb) {  // g += g_m;  the preconditioner is the membrane's own diagonal blocks + mu I (in both back ends)
    s = membrane_energy_grad_impl<T>(ctx, pos, em_dev, g, true, st);
    if (s != TT_OK) return s;
    minv = ctx->nw_minv.as<T>();
    s = membrane_apply_impl<T, 2>(ctx, pos, nullptr, o->mu, false, minv, st);
    if (s != TT_OK) return s;
  } else if (!mf) {
    minv = ctx->nw_minv.as<T>();
    k_block_jacobi<T><<<grid_for(nV, VEC_THREADS), VEC_THREADS, 0, st>>>(rowptr, colind, vals, nV, o->mu, minv);
    TT_LAUNCH_CHECK();
  }
  tt_pcg_options po = o->pcg;
  po.shift = o->mu;
  int32_t iters = 0;
  double relres = 0.0;
  s = pcg_impl<T>(ctx, &q, rowptr, colind, vals, minv, g, d, &po, &iters, &relres, st, mb);
  if (s != TT_OK) return s;
  rep->pcg_iters = iters;
  rep->pcg_relres = relres;
  const unsigned gn = grid_for(n, VEC_THREADS);
  double* part0 = ctx->pcg_part[0].as<double>();
  double* part1 = ctx->pcg_part[1].as<double>();
  k_dot2<T><<<gn, VEC_THREADS, 0, st>>>(g, d, n, part0, part1);
  TT_LAUNCH_CHECK();
  k_dot2_final<<<1, 1024, 0, st>>>(part0, part1, (int64_t)gn, sc);
  TT_LAUNCH_CHECK();
  double h_sc[2] = {0.0, 0.0}, h_em[2] = {0.0, 0.0};
  T h_e[2] = {(T)0, (T)0};
  TT_CUDA(cudaMemcpyAsync(h_sc, sc, sizeof(h_sc), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaMemcpyAsync(h_e, e_dev, sizeof(T), cudaMemcpyDeviceToHost, st));
  if (mb) TT_CUDA(cudaMemcpyAsync(h_em, em_dev, sizeof(double), cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaStreamSynchronize(st));
  const double E0 = (double)h_e[0] + h_em[0], gd = h_sc[0];
  rep->energy_membrane = h_em[0];
  rep->energy0 = rep->energy1 = E0;
  rep->gd = gd;
  rep->grad_norm = sqrt(h_sc[1]);
  // ---- Armijo backtracking on the energy of the SAME candidate list ----
  tt_problem qt{x_try, nV, tris, nT, pairs, P};
  double alpha = 1.0;
  for (int j = 0; j <= o->max_backtrack; ++j) {
    k_step<T><<<gn, VEC_THREADS, 0, st>>>((const T*)pos, d, alpha, n, x_try);
    TT_LAUNCH_CHECK();
    s = energy_impl<T>(ctx, &qt, e_dev + 1, nullptr, nullptr, nullptr, nullptr, st);
    if (s != TT_OK) return s;
    if (mb) {
      s = membrane_energy_grad_impl<T>(ctx, x_try, em_dev + 1, nullptr, false, st);
      if (s != TT_OK) return s;
      TT_CUDA(cudaMemcpyAsync(h_em + 1, em_dev + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    TT_CUDA(cudaMemcpyAsync(h_e + 1, e_dev + 1, sizeof(T), cudaMemcpyDeviceToHost, st));
    TT_CUDA(cudaStreamSynchronize(st));
    const double Et = (double)h_e[1] + h_em[1];
    if (Et <= E0 - o->armijo_c1 * alpha * gd) {
      TT_CUDA(cudaMemcpyAsync(pos, x_try, sizeof(T) * (size_t)n, cudaMemcpyDeviceToDevice, st));
      rep->energy1 = Et;
      rep->energy_membrane = h_em[1];
      rep->alpha = alpha;
      rep->backtracks = j;
      rep->accepted = 1;
      ctx->sig.valid = false;  // the positions have moved: the cached active set and branch decisions are stale
      return TT_OK;
    }
    alpha *= 0.5;
  }
  rep->backtracks = o->max_backtrack + 1;
  return TT_OK;
}

tt_status check_newton_args(tt_ctx* ctx, const void* pos, int64_t nV, const int32_t* tris, int64_t nT, const tt_newton_options* o) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (!o || !(o->mu > 0.0) || !(o->armijo_c1 > 0.0 && o->armijo_c1 < 1.0) || o->max_backtrack < 0 || o->pcg.max_iter < 0 ||
      !(o->pcg.rtol >= 0.0))
    return fail(ctx, TT_ERR_INVALID_ARG, "newton options: need mu > 0, 0 < armijo_c1 < 1, max_backtrack >= 0, pcg.max_iter >= 0, pcg.rtol >= 0");
  if (nV < 0 || nT < 0 || (nV > 0 && !pos) || (nT > 0 && !tris)) return fail(ctx, TT_ERR_INVALID_ARG, "NULL array or negative size");
  if (o->membrane != 0 && ctx->mb_nV != nV)
    return fail(ctx, TT_ERR_STATE, "newton options ask for the membrane term, but tt_membrane_build has not been called for a mesh of %lld vertices",
                (long long)nV);
  return TT_OK;
}

}  // namespace

// =================================================================================== C ABI
extern "C" {

tt_status tt_create(const tt_options* opt, tt_ctx** out) {
  if (!opt || !out) return TT_ERR_INVALID_ARG;
  *out = nullptr;
  if (opt->dtype != TT_F64 && opt->dtype != TT_F32) return TT_ERR_INVALID_ARG;
  if (opt->hess_mode < TT_HESS_EQ4 || opt->hess_mode > TT_HESS_EXACT) return TT_ERR_INVALID_ARG;
  if (!(opt->tc_scale > 0.0)) return TT_ERR_INVALID_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || opt->device < 0 || opt->device >= ndev) {
    (void)cudaGetLastError();
    return TT_ERR_CUDA;
  }
  if (cudaSetDevice(opt->device) != cudaSuccess) return TT_ERR_CUDA;
  tt_ctx* c = new (std::nothrow) tt_ctx();
  if (!c) return TT_ERR_NOMEM;
  c->opt = *opt;
  for (int i = 0; i < 3; ++i)
    for (int r = 0; r < tt_ctx::EV_RING; ++r)
      for (int j = 0; j < 2; ++j)
        if (cudaEventCreate(&c->evr[i][r][j]) != cudaSuccess) { (void)cudaGetLastError(); tt_destroy(c); return TT_ERR_CUDA; }
  if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_in, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_p, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_num, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_side, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_sig, cudaEventDisableTiming) != cudaSuccess ||
      cudaMallocHost((void**)&c->h_sig, 2 * sizeof(unsigned long long)) != cudaSuccess) {
    (void)cudaGetLastError();
    tt_destroy(c);
    return TT_ERR_CUDA;
  }
  {
    cudaError_t e = cudaSuccess;
    auto opt_in = [&](const void* f, size_t smem) { if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); };
    int sms = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, opt->device);
    auto tile_setup = [&](const void* f, size_t smem, int* grid) {  // opt in; persistent grid = one wave of resident CTAs
      int nb = 0;
      opt_in(f, smem);
      if (grid && e == cudaSuccess) {
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, f, 32 * ttk::TILE_WARPS, smem);
        *grid = sms * (nb > 0 ? nb : 1);
      }
    };
#define TT_TILE_SETUP(T, DI, MT, MI)                                                                                        \
    tile_setup((const void*)ttk::k_assemble_tile<T, false, false, MT>, sizeof(ttk::TileWarpSmem<T, MT>) * ttk::TILE_WARPS, nullptr); \
    tile_setup((const void*)ttk::k_assemble_tile<T, false, true, MT>, sizeof(ttk::TileWarpSmem<T, MT>) * ttk::TILE_WARPS, nullptr);  \
    tile_setup((const void*)ttk::k_assemble_tile<T, true, false, MT>, sizeof(ttk::TileWarpSmem<T, MT>) * ttk::TILE_WARPS, nullptr);  \
    tile_setup((const void*)ttk::k_assemble_tile<T, true, true, MT>, sizeof(ttk::TileWarpSmem<T, MT>) * ttk::TILE_WARPS, &c->tile_grid[DI][MI]);
    TT_TILE_SETUP(double, 0, ttk::RND_TRI_LOW, 0)
    TT_TILE_SETUP(double, 0, ttk::RND_MAX_TRI, 1)
    TT_TILE_SETUP(float, 1, ttk::RND_TRI_LOW, 0)
    TT_TILE_SETUP(float, 1, ttk::RND_MAX_TRI, 1)
#undef TT_TILE_SETUP
    opt_in((const void*)ttk::k_assemble_long_tile<double, true>, sizeof(ttk::LongTileSmem<double, true>));
    opt_in((const void*)ttk::k_assemble_long_tile<double, false>, sizeof(ttk::LongTileSmem<double, false>));
    opt_in((const void*)ttk::k_assemble_long_tile<float, true>, sizeof(ttk::LongTileSmem<float, true>));
    opt_in((const void*)ttk::k_assemble_long_tile<float, false>, sizeof(ttk::LongTileSmem<float, false>));
    // tt_energy_static's scratch: the device address of the file-scope array on THIS device (the name itself is a host
    // stand-in); asked for here, at set-up, so that the entry point itself does nothing but launch
    if (e == cudaSuccess) e = cudaGetSymbolAddress((void**)&c->static_scratch, tt_static_scratch);
    if (e != cudaSuccess) { (void)cudaGetLastError(); delete c; return TT_ERR_CUDA; }
    auto pipe_setup = [&](const void* f, size_t smem, int& grid) {
      int nb = 0;
      opt_in(f, smem);
      if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessorWithFlags(&nb, f, 32 * ttk::PIPE_WARPS, smem, cudaOccupancyDefault);
      grid = sms * (nb > 0 ? nb : 1);
    };
    pipe_setup((const void*)ttk::k_entry_pipe<double, 1>, sizeof(ttk::PipeWarpSmem<double, 1>) * ttk::PIPE_WARPS, c->pipe_grid[0][0]);
    pipe_setup((const void*)ttk::k_entry_pipe<double, 2>, sizeof(ttk::PipeWarpSmem<double, 2>) * ttk::PIPE_WARPS, c->pipe_grid[0][1]);
    pipe_setup((const void*)ttk::k_entry_pipe<float, 1>, sizeof(ttk::PipeWarpSmem<float, 1>) * ttk::PIPE_WARPS, c->pipe_grid[1][0]);
    pipe_setup((const void*)ttk::k_entry_pipe<float, 2>, sizeof(ttk::PipeWarpSmem<float, 2>) * ttk::PIPE_WARPS, c->pipe_grid[1][1]);
    if (e != cudaSuccess) { (void)cudaGetLastError(); delete c; return TT_ERR_CUDA; }
    c->sms = sms;
  }
  *out = c;
  return TT_OK;
}

void tt_destroy(tt_ctx* ctx) {
  if (!ctx) return;
  cudaSetDevice(ctx->opt.device);
  for (int i = 0; i < 3; ++i)
    for (int r = 0; r < tt_ctx::EV_RING; ++r)
      for (int j = 0; j < 2; ++j)
        if (ctx->evr[i][r][j]) cudaEventDestroy(ctx->evr[i][r][j]);
  for (cudaEvent_t e : {ctx->ev_in, ctx->ev_p, ctx->ev_num, ctx->ev_side, ctx->ev_sig})
    if (e) cudaEventDestroy(e);
  if (ctx->h_sig) cudaFreeHost(ctx->h_sig);
  if (ctx->side) cudaStreamDestroy(ctx->side);
  delete ctx;
}

tt_status tt_energy(tt_ctx* ctx, const tt_problem* prob, void* energy_sum, void* energy_per_pair,
                    uint32_t* active_mask, void* tc, int64_t* n_active, void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if (!energy_sum) return fail(ctx, TT_ERR_INVALID_ARG, "energy_sum is NULL");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64
             ? energy_impl<double>(ctx, prob, energy_sum, energy_per_pair, active_mask, tc, n_active, st)
             : energy_impl<float>(ctx, prob, energy_sum, energy_per_pair, active_mask, tc, n_active, st);
}

#ifdef TT_K4_PROFILE
int tt_debug_k4_prof(unsigned long long* out16, int reset) {
  cudaDeviceSynchronize();
  if (out16) cudaMemcpyFromSymbol(out16, ttk::tt_k4_prof, 16 * sizeof(unsigned long long));
  if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(ttk::tt_k4_prof, z, sizeof(z)); }
  return 0;
}
#endif
tt_status tt_energy_static(tt_ctx* ctx, const tt_problem* prob, void* energy_sum, int64_t* n_active, void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if (!energy_sum) return fail(ctx, TT_ERR_INVALID_ARG, "energy_sum is NULL");
  if (prob->n_pairs > TT_STATIC_MAX_PAIRS)
    return fail(ctx, TT_ERR_CAPACITY, "tt_energy_static: n_pairs %lld exceeds TT_STATIC_MAX_PAIRS = %lld (the size of the library's static scratch); use tt_energy",
                (long long)prob->n_pairs, (long long)TT_STATIC_MAX_PAIRS);
  if (!ctx->static_scratch) return fail(ctx, TT_ERR_STATE, "tt_energy_static: the static scratch has no device address");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? energy_static_impl<double>(ctx, prob, energy_sum, n_active, st)
                                  : energy_static_impl<float>(ctx, prob, energy_sum, n_active, st);
}

tt_status tt_hess_symbolic(tt_ctx* ctx, const tt_problem* prob, int64_t* nnzb_host, int64_t* n_active_host,
                           void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if (!nnzb_host) return fail(ctx, TT_ERR_INVALID_ARG, "nnzb_host is NULL");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? symbolic_impl<double>(ctx, prob, nnzb_host, n_active_host, st)
                                  : symbolic_impl<float>(ctx, prob, nnzb_host, n_active_host, st);
}

tt_status tt_energy_grad_hess(tt_ctx* ctx, const tt_problem* prob, void* energy_sum, void* grad,
                              int32_t* bsr_rowptr, int32_t* bsr_colind, void* bsr_vals, int64_t nnzb_capacity,
                              void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if (!ctx->sig.matches(prob)) return fail(ctx, TT_ERR_STATE, "tt_energy_grad_hess: no matching tt_hess_symbolic for this problem");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  s = check_positions_begin(ctx, prob, st);
  if (s != TT_OK) return s;
  s = ctx->opt.dtype == TT_F64
          ? numeric_impl<double>(ctx, prob, energy_sum, grad, bsr_rowptr, bsr_colind, bsr_vals, nnzb_capacity, st)
          : numeric_impl<float>(ctx, prob, energy_sum, grad, bsr_rowptr, bsr_colind, bsr_vals, nnzb_capacity, st);
  const tt_status s_pos = check_positions_end(ctx, "tt_energy_grad_hess");
  return s_pos != TT_OK ? s_pos : s;
}

tt_status tt_hess_vec(tt_ctx* ctx, const tt_problem* prob, const void* p, void* y, void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if (!p || !y || p == y) return fail(ctx, TT_ERR_INVALID_ARG, "p / y NULL or aliased");
  if (!ctx->sig.matches(prob)) return fail(ctx, TT_ERR_STATE, "tt_hess_vec: no matching tt_hess_symbolic for this problem");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  s = check_positions_begin(ctx, prob, st);
  if (s != TT_OK) return s;
  s = ctx->opt.dtype == TT_F64 ? hessvec_impl<double>(ctx, prob, p, y, st) : hessvec_impl<float>(ctx, prob, p, y, st);
  const tt_status s_pos = check_positions_end(ctx, "tt_hess_vec");
  return s_pos != TT_OK ? s_pos : s;
}

namespace {
// body of tt_energy_grad_hess_host; the wrapper below drains both streams on ANY failure, so that no
// copy from / into the caller's host buffers is still in flight when an error is returned
tt_status host_impl(tt_ctx* ctx, const tt_problem* prob, void* energy_host, void* grad_host, int64_t* nnzb_host,
                    int64_t* n_active_host, int32_t* rowptr_host, int32_t* colind_host, void* vals_host,
                    int64_t nnzb_capacity, const void* p_host, void* y_host, cudaStream_t st) {
  tt_status s = TT_OK;
  const size_t w = ctx->opt.dtype == TT_F64 ? 8 : 4;
  const int64_t nV = prob->n_verts, nT = prob->n_tris, P = prob->n_pairs;
  TT_CUDA(ctx->h_pos.ensure(w * 3 * (size_t)nV + 16));
  TT_CUDA(ctx->h_tris.ensure(sizeof(int) * 3 * (size_t)nT + 16));
  TT_CUDA(ctx->h_pairs.ensure(sizeof(int) * 2 * (size_t)P + 16));
  TT_CUDA(ctx->o_grad.ensure(w * 3 * (size_t)nV + 16));
  TT_CUDA(ctx->o_energy.ensure(16));
  // Copy schedule (PCIe is full duplex; the step is shorter than its copies):
  //   stream : H2D pos, tris, pairs -> symbolic -> [wait p] H.p -> numeric -> D2H energy, grad, pattern, values
  //   side   : [after the inputs] H2D p (under the symbolic phase)
  //            [after H.p] D2H y (under the numeric phase)
  const bool want_hv = p_host && nV;
  if (want_hv) {
    TT_CUDA(ctx->h_p.ensure(w * 3 * (size_t)nV + 16));
    TT_CUDA(ctx->o_y.ensure(w * 3 * (size_t)nV + 16));
  }
  if (nV) TT_CUDA(cudaMemcpyAsync(ctx->h_pos.p, prob->pos, w * 3 * (size_t)nV, cudaMemcpyHostToDevice, st));
  if (nT) TT_CUDA(cudaMemcpyAsync(ctx->h_tris.p, prob->tris, sizeof(int) * 3 * (size_t)nT, cudaMemcpyHostToDevice, st));
  if (P) TT_CUDA(cudaMemcpyAsync(ctx->h_pairs.p, prob->pairs, sizeof(int) * 2 * (size_t)P, cudaMemcpyHostToDevice, st));
  TT_CUDA(cudaEventRecord(ctx->ev_in, st));
  if (want_hv) {
    TT_CUDA(cudaStreamWaitEvent(ctx->side, ctx->ev_in, 0));
    TT_CUDA(cudaMemcpyAsync(ctx->h_p.p, p_host, w * 3 * (size_t)nV, cudaMemcpyHostToDevice, ctx->side));
    TT_CUDA(cudaEventRecord(ctx->ev_p, ctx->side));
  }
  tt_problem d = *prob;
  d.pos = ctx->h_pos.p;
  d.tris = ctx->h_tris.as<int32_t>();
  d.pairs = ctx->h_pairs.as<int32_t>();
  int64_t nnzb = 0, A = 0;
  s = ctx->opt.dtype == TT_F64 ? symbolic_impl<double>(ctx, &d, &nnzb, &A, st) : symbolic_impl<float>(ctx, &d, &nnzb, &A, st);
  if (s != TT_OK) return s;
  *nnzb_host = nnzb;
  if (n_active_host) *n_active_host = A;
  if ((colind_host || vals_host) && nnzb_capacity < nnzb)
    return fail(ctx, TT_ERR_CAPACITY, "nnzb_capacity %lld < nnzb %lld", (long long)nnzb_capacity, (long long)nnzb);
  TT_CUDA(ctx->o_vals.ensure(w * 9 * (size_t)nnzb + 16));
  // H.p first: it needs only the symbolic phase and p, and its result then leaves (side stream)
  // under the numeric phase; the numeric results leave last.  (The positions are the ctx-owned copy
  // made above: no state check needed.)
  if (want_hv) {
    TT_CUDA(cudaStreamWaitEvent(st, ctx->ev_p, 0));
    s = ctx->opt.dtype == TT_F64 ? hessvec_impl<double>(ctx, &d, ctx->h_p.p, ctx->o_y.p, st)
                                 : hessvec_impl<float>(ctx, &d, ctx->h_p.p, ctx->o_y.p, st);
    if (s != TT_OK) return s;
    TT_CUDA(cudaEventRecord(ctx->ev_num, st));
    TT_CUDA(cudaStreamWaitEvent(ctx->side, ctx->ev_num, 0));
    TT_CUDA(cudaMemcpyAsync(y_host, ctx->o_y.p, w * 3 * (size_t)nV, cudaMemcpyDeviceToHost, ctx->side));
  }
  s = ctx->opt.dtype == TT_F64
          ? numeric_impl<double>(ctx, &d, ctx->o_energy.p, ctx->o_grad.p, ctx->rowptr.as<int>(), ctx->colind.as<int>(), ctx->o_vals.p, nnzb, st)
          : numeric_impl<float>(ctx, &d, ctx->o_energy.p, ctx->o_grad.p, ctx->rowptr.as<int>(), ctx->colind.as<int>(), ctx->o_vals.p, nnzb, st);
  if (s != TT_OK) return s;
  ctx->host_nnzb = nnzb;
  TT_CUDA(cudaMemcpyAsync(energy_host, ctx->o_energy.p, w, cudaMemcpyDeviceToHost, st));
  if (grad_host && nV) TT_CUDA(cudaMemcpyAsync(grad_host, ctx->o_grad.p, w * 3 * (size_t)nV, cudaMemcpyDeviceToHost, st));
  if (rowptr_host) TT_CUDA(cudaMemcpyAsync(rowptr_host, ctx->rowptr.p, sizeof(int) * (size_t)(nV + 1), cudaMemcpyDeviceToHost, st));
  if (colind_host && nnzb) TT_CUDA(cudaMemcpyAsync(colind_host, ctx->colind.p, sizeof(int) * (size_t)nnzb, cudaMemcpyDeviceToHost, st));
  if (vals_host && nnzb) TT_CUDA(cudaMemcpyAsync(vals_host, ctx->o_vals.p, w * 9 * (size_t)nnzb, cudaMemcpyDeviceToHost, st));
  TT_CUDA(cudaEventRecord(ctx->ev_side, ctx->side));
  TT_CUDA(cudaStreamWaitEvent(st, ctx->ev_side, 0));  // `stream` completes only after the side copies
  TT_CUDA(cudaStreamSynchronize(st));
  return TT_OK;
}
}  // namespace

tt_status tt_energy_grad_hess_host(tt_ctx* ctx, const tt_problem* prob, void* energy_host, void* grad_host,
                                   int64_t* nnzb_host, int64_t* n_active_host, int32_t* rowptr_host,
                                   int32_t* colind_host, void* vals_host, int64_t nnzb_capacity,
                                   const void* p_host, void* y_host, void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if ((p_host == nullptr) != (y_host == nullptr)) return fail(ctx, TT_ERR_INVALID_ARG, "p_host and y_host must both be set or both NULL");
  if (!energy_host || !nnzb_host) return fail(ctx, TT_ERR_INVALID_ARG, "energy_host / nnzb_host is NULL");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  s = host_impl(ctx, prob, energy_host, grad_host, nnzb_host, n_active_host, rowptr_host, colind_host, vals_host,
                nnzb_capacity, p_host, y_host, st);
  if (s != TT_OK) {  // no DMA from / into the caller's buffers may outlive a failed call
    (void)cudaStreamSynchronize(ctx->side);
    (void)cudaStreamSynchronize(st);
    (void)cudaGetLastError();
  }
  return s;
}

tt_status tt_broad_phase(tt_ctx* ctx, const void* pos, int64_t n_verts, const int32_t* tris, int64_t n_tris,
                         double inflate, int64_t* n_pairs_host, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (!n_pairs_host) return fail(ctx, TT_ERR_INVALID_ARG, "n_pairs_host is NULL");
  if (n_verts < 0 || n_tris < 0 || !(inflate >= 0.0)) return fail(ctx, TT_ERR_INVALID_ARG, "negative size or inflate");
  if (n_verts >= (int64_t(1) << 31) / 3 || n_tris >= (int64_t(1) << 31) / 128)
    return fail(ctx, TT_ERR_INVALID_ARG, "sizes exceed int32 indexing (nV < 2^31/3, nT < 2^31/128)");
  if ((n_verts > 0 && !pos) || (n_tris > 0 && !tris)) return fail(ctx, TT_ERR_INVALID_ARG, "NULL array with non-zero size");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? broad_impl<double>(ctx, pos, n_verts, tris, n_tris, inflate, n_pairs_host, st)
                                  : broad_impl<float>(ctx, pos, n_verts, tris, n_tris, inflate, n_pairs_host, st);
}

tt_status tt_broad_phase_pairs(tt_ctx* ctx, const int32_t** pairs, int64_t* n_pairs) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (ctx->bp_n_pairs < 0) return fail(ctx, TT_ERR_STATE, "tt_broad_phase_pairs: no tt_broad_phase result");
  if (pairs) *pairs = ctx->bp_pairs.as<int32_t>();
  if (n_pairs) *n_pairs = ctx->bp_n_pairs;
  return TT_OK;
}

tt_status tt_broad_phase_copy(tt_ctx* ctx, int32_t* pairs_out, int64_t capacity, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (ctx->bp_n_pairs < 0) return fail(ctx, TT_ERR_STATE, "tt_broad_phase_copy: no tt_broad_phase result");
  if (capacity < ctx->bp_n_pairs) return fail(ctx, TT_ERR_CAPACITY, "capacity %lld < %lld pairs", (long long)capacity, (long long)ctx->bp_n_pairs);
  if (ctx->bp_n_pairs > 0) {
    if (!pairs_out) return fail(ctx, TT_ERR_INVALID_ARG, "pairs_out is NULL");
    TT_CUDA(cudaSetDevice(ctx->opt.device));
    TT_CUDA(cudaMemcpyAsync(pairs_out, ctx->bp_pairs.p, sizeof(int32_t) * 2 * (size_t)ctx->bp_n_pairs, cudaMemcpyDeviceToDevice,
                            (cudaStream_t)stream));
  }
  return TT_OK;
}

tt_status tt_bsr_spmv(tt_ctx* ctx, int64_t n_rows, const int32_t* rowptr, const int32_t* colind, const void* vals,
                      double shift, const void* x, void* y, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (n_rows < 0 || n_rows >= (int64_t(1) << 31) / 3) return fail(ctx, TT_ERR_INVALID_ARG, "tt_bsr_spmv: n_rows out of range");
  if (n_rows > 0 && (!rowptr || !x || !y || x == y)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_bsr_spmv: NULL or aliased argument");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? spmv_impl<double>(ctx, n_rows, rowptr, colind, vals, shift, x, y, st)
                                  : spmv_impl<float>(ctx, n_rows, rowptr, colind, vals, shift, x, y, st);
}

tt_status tt_block_jacobi(tt_ctx* ctx, int64_t n_rows, const int32_t* rowptr, const int32_t* colind, const void* vals,
                          double shift, void* minv, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (n_rows < 0 || n_rows >= (int64_t(1) << 31) / 3) return fail(ctx, TT_ERR_INVALID_ARG, "tt_block_jacobi: n_rows out of range");
  if (n_rows > 0 && (!rowptr || !minv)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_block_jacobi: NULL argument");
  if (n_rows == 0) return TT_OK;
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  if (ctx->opt.dtype == TT_F64)
    tts::k_block_jacobi<double><<<grid_for(n_rows, tts::VEC_THREADS), tts::VEC_THREADS, 0, st>>>(rowptr, colind, (const double*)vals, n_rows, shift, (double*)minv);
  else
    tts::k_block_jacobi<float><<<grid_for(n_rows, tts::VEC_THREADS), tts::VEC_THREADS, 0, st>>>(rowptr, colind, (const float*)vals, n_rows, shift, (float*)minv);
  TT_LAUNCH_CHECK();
  return TT_OK;
}

tt_status tt_pcg_solve(tt_ctx* ctx, const tt_problem* prob, const int32_t* rowptr, const int32_t* colind, const void* vals,
                       const void* minv, const void* b, void* x, const tt_pcg_options* opt, int32_t* iters_host,
                       double* relres_host, void* stream) {
  tt_status s = check_problem(ctx, prob);
  if (s != TT_OK) return s;
  if (!opt || opt->max_iter < 0 || !(opt->rtol >= 0.0) || !(opt->shift >= 0.0))
    return fail(ctx, TT_ERR_INVALID_ARG, "tt_pcg_solve: options NULL or max_iter / rtol / shift negative");
  if (prob->n_verts > 0 && (!b || !x || b == x)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_pcg_solve: b / x NULL or aliased");
  const bool matrix_free = (vals == nullptr);
  if (!matrix_free && (!rowptr || !colind)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_pcg_solve: rowptr / colind / vals must be all set (BSR) or all NULL (matrix-free)");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  if (matrix_free) {
    if (!ctx->sig.matches(prob)) return fail(ctx, TT_ERR_STATE, "tt_pcg_solve (matrix-free): no matching tt_hess_symbolic for this problem");
    s = check_positions(ctx, prob, "tt_pcg_solve", st);  // once per solve, not per product
    if (s != TT_OK) return s;
  }
  return ctx->opt.dtype == TT_F64 ? pcg_impl<double>(ctx, prob, rowptr, colind, vals, minv, b, x, opt, iters_host, relres_host, st)
                                  : pcg_impl<float>(ctx, prob, rowptr, colind, vals, minv, b, x, opt, iters_host, relres_host, st);
}

tt_status tt_membrane_build(tt_ctx* ctx, const void* rest_pos, int64_t n_verts, const int32_t* tris, int64_t n_tris,
                            double stiffness, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (n_verts < 0 || n_tris < 0 || n_verts >= (int64_t(1) << 31) / 3 || n_tris >= (int64_t(1) << 31) / 6)
    return fail(ctx, TT_ERR_INVALID_ARG, "tt_membrane_build: size out of range");
  if ((n_verts > 0 && !rest_pos) || (n_tris > 0 && !tris)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_membrane_build: NULL array");
  if (!(stiffness >= 0.0)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_membrane_build: stiffness must be >= 0");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  if (n_tris > 0) {
    tt_status s = validate_indices(ctx, tris, n_tris, n_verts, nullptr, 0, st);
    if (s != TT_OK) return s;
  }
  return ctx->opt.dtype == TT_F64 ? membrane_build_impl<double>(ctx, rest_pos, n_verts, tris, n_tris, stiffness, st)
                                  : membrane_build_impl<float>(ctx, rest_pos, n_verts, tris, n_tris, stiffness, st);
}

tt_status tt_membrane_energy_grad(tt_ctx* ctx, const void* pos, double* energy, void* grad, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (ctx->mb_nV < 0) return fail(ctx, TT_ERR_STATE, "tt_membrane_energy_grad without tt_membrane_build");
  if (!energy || (ctx->mb_nV > 0 && !pos)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_membrane_energy_grad: NULL argument");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? membrane_energy_grad_impl<double>(ctx, pos, energy, grad, false, st)
                                  : membrane_energy_grad_impl<float>(ctx, pos, energy, grad, false, st);
}

tt_status tt_membrane_hess_vec(tt_ctx* ctx, const void* pos, const void* p, void* y, void* stream) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (ctx->mb_nV < 0) return fail(ctx, TT_ERR_STATE, "tt_membrane_hess_vec without tt_membrane_build");
  if (ctx->mb_nV > 0 && (!pos || !p || !y || p == y)) return fail(ctx, TT_ERR_INVALID_ARG, "tt_membrane_hess_vec: NULL or aliased argument");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? membrane_apply_impl<double, 1>(ctx, pos, p, 0.0, false, y, st)
                                  : membrane_apply_impl<float, 1>(ctx, pos, p, 0.0, false, y, st);
}

tt_status tt_newton_step(tt_ctx* ctx, void* pos, int64_t n_verts, const int32_t* tris, int64_t n_tris, const int32_t* pairs,
                         int64_t n_pairs, const tt_newton_options* opt, tt_newton_report* report_host, void* stream) {
  tt_status s = check_newton_args(ctx, pos, n_verts, tris, n_tris, opt);
  if (s != TT_OK) return s;
  if (!report_host) return fail(ctx, TT_ERR_INVALID_ARG, "tt_newton_step: report_host is NULL");
  tt_problem q{pos, n_verts, tris, n_tris, pairs, n_pairs};
  s = check_problem(ctx, &q);
  if (s != TT_OK) return s;
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->opt.dtype == TT_F64 ? newton_impl<double>(ctx, pos, n_verts, tris, n_tris, pairs, n_pairs, opt, report_host, st)
                                  : newton_impl<float>(ctx, pos, n_verts, tris, n_tris, pairs, n_pairs, opt, report_host, st);
}

tt_status tt_untangle(tt_ctx* ctx, void* pos, int64_t n_verts, const int32_t* tris, int64_t n_tris, double inflate,
                      int32_t max_steps, const tt_newton_options* opt, tt_newton_report* history_host, int32_t* steps_host,
                      void* stream) {
  tt_status s = check_newton_args(ctx, pos, n_verts, tris, n_tris, opt);
  if (s != TT_OK) return s;
  if (max_steps < 0 || (max_steps > 0 && !history_host) || !steps_host || !(inflate >= 0.0))
    return fail(ctx, TT_ERR_INVALID_ARG, "tt_untangle: max_steps / inflate negative, or history_host / steps_host NULL");
  TT_CUDA(cudaSetDevice(ctx->opt.device));
  cudaStream_t st = (cudaStream_t)stream;
  *steps_host = 0;
  for (int it = 0; it < max_steps; ++it) {
    int64_t n_pairs = 0;
    s = ctx->opt.dtype == TT_F64 ? broad_impl<double>(ctx, pos, n_verts, tris, n_tris, inflate, &n_pairs, st)
                                 : broad_impl<float>(ctx, pos, n_verts, tris, n_tris, inflate, &n_pairs, st);
    if (s != TT_OK) return s;
    const int32_t* pairs = n_pairs > 0 ? ctx->bp_pairs.as<int32_t>() : nullptr;
    tt_newton_report* rep = history_host + it;
    s = ctx->opt.dtype == TT_F64 ? newton_impl<double>(ctx, pos, n_verts, tris, n_tris, pairs, n_pairs, opt, rep, st)
                                 : newton_impl<float>(ctx, pos, n_verts, tris, n_tris, pairs, n_pairs, opt, rep, st);
    if (s != TT_OK) return s;
    *steps_host = it + 1;
    if (rep->n_active == 0 || !rep->accepted) break;
  }
  return TT_OK;
}

tt_status tt_hess_pattern(tt_ctx* ctx, const int32_t** rowptr, const int32_t** colind, int64_t* nnzb) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (!ctx->sig.valid) return fail(ctx, TT_ERR_STATE, "tt_hess_pattern: no tt_hess_symbolic result");
  if (rowptr) *rowptr = ctx->rowptr.as<int32_t>();
  if (colind) *colind = ctx->colind.as<int32_t>();
  if (nnzb) *nnzb = ctx->nnzb;
  return TT_OK;
}

tt_status tt_bsr_device(tt_ctx* ctx, const int32_t** rowptr, const int32_t** colind, const void** vals, int64_t* nnzb) {
  if (!ctx) return TT_ERR_INVALID_ARG;
  if (!ctx->o_vals.p) return fail(ctx, TT_ERR_STATE, "tt_bsr_device: no tt_energy_grad_hess_host result");
  if (rowptr) *rowptr = ctx->rowptr.as<int32_t>();
  if (colind) *colind = ctx->colind.as<int32_t>();
  if (vals) *vals = ctx->o_vals.p;
  if (nnzb) *nnzb = ctx->host_nnzb;
  return TT_OK;
}

tt_status tt_stats(const tt_ctx* ctx, int64_t* what, int32_t n) {
  if (!ctx || !what || n < 0) return TT_ERR_INVALID_ARG;
  const int64_t v[13] = {ctx->A, ctx->n_dir, ctx->n_touched, ctx->nnzb - ctx->U, ctx->U, ctx->R, ctx->nnzb, ctx->launches,
                         ctx->n_slots, ctx->n_split, ctx->n_parts, ctx->n_long, ctx->n_chunks};
  for (int i = 0; i < n && i < 13; ++i) what[i] = v[i];
  return TT_OK;
}

tt_status tt_kernel_ms(tt_ctx* ctx, float* ms, int32_t n) {
  if (!ctx || !ms || n < 0) return TT_ERR_INVALID_ARG;
  for (int i = 0; i < n && i < 3; ++i) {
    ms[i] = -1.0f;
    if (ctx->ev_n[i] == 0) continue;
    cudaEvent_t* e = ctx->evr[i][(ctx->ev_n[i] - 1) % tt_ctx::EV_RING];
    TT_CUDA(cudaEventSynchronize(e[1]));
    TT_CUDA(cudaEventElapsedTime(&ms[i], e[0], e[1]));
  }
  return TT_OK;
}

tt_status tt_kernel_ms_mean(tt_ctx* ctx, float* ms, int32_t* launches, int32_t n, int32_t reset) {
  if (!ctx || !ms || n < 0) return TT_ERR_INVALID_ARG;
  for (int i = 0; i < n && i < 3; ++i) {
    ms[i] = -1.0f;
    const int64_t cnt = ctx->ev_n[i] < tt_ctx::EV_RING ? ctx->ev_n[i] : tt_ctx::EV_RING;
    if (launches) launches[i] = (int32_t)cnt;
    if (cnt == 0) continue;
    double tot = 0.0;
    for (int64_t k = 0; k < cnt; ++k) {
      cudaEvent_t* e = ctx->evr[i][(ctx->ev_n[i] - 1 - k) % tt_ctx::EV_RING];
      float t = 0.0f;
      TT_CUDA(cudaEventSynchronize(e[1]));
      TT_CUDA(cudaEventElapsedTime(&t, e[0], e[1]));
      tot += t;
    }
    ms[i] = (float)(tot / (double)cnt);
  }
  if (reset) ctx->ev_n[0] = ctx->ev_n[1] = ctx->ev_n[2] = 0;
  return TT_OK;
}

tt_status tt_probe_peaks(int32_t device, double* tflops) {
  if (!tflops) return TT_ERR_INVALID_ARG;
  if (cudaSetDevice(device) != cudaSuccess) { (void)cudaGetLastError(); return TT_ERR_CUDA; }
  tflops[0] = ttp::fma_tflops<double>(nullptr);
  tflops[1] = ttp::fma_tflops<float>(nullptr);
  return (tflops[0] > 0.0 && tflops[1] > 0.0) ? TT_OK : TT_ERR_CUDA;
}

tt_status tt_probe_gather(int32_t device, double* gbs) {
  if (!gbs) return TT_ERR_INVALID_ARG;
  if (cudaSetDevice(device) != cudaSuccess) { (void)cudaGetLastError(); return TT_ERR_CUDA; }
  const size_t bytes = (size_t)144 << 20;       // the size of config 4's position array (6 M vertices, fp64)
  const long long items = 60ll * 1000 * 1000;   // K1 gathers 60 M vertices per 10 M candidates
  gbs[0] = ttp::gather_gbs<3>(bytes, items, nullptr);
  gbs[1] = ttp::gather_gbs<9>(bytes, items / 3, nullptr);
  return (gbs[0] > 0.0 && gbs[1] > 0.0) ? TT_OK : TT_ERR_CUDA;
}

const char* tt_status_string(tt_status s) {
  switch (s) {
    case TT_OK: return "TT_OK";
    case TT_ERR_INVALID_ARG: return "TT_ERR_INVALID_ARG";
    case TT_ERR_CUDA: return "TT_ERR_CUDA";
    case TT_ERR_NOMEM: return "TT_ERR_NOMEM";
    case TT_ERR_CAPACITY: return "TT_ERR_CAPACITY";
    case TT_ERR_STATE: return "TT_ERR_STATE";
  }
  return "TT_ERR_UNKNOWN";
}

const char* tt_last_error(const tt_ctx* ctx) { return ctx ? ctx->err.c_str() : "ctx is NULL"; }

}  // extern "C"
