/* include/tt.h -- C ABI of libtt.so: the B200 (sm_100a) hot path of arXiv 2606.06511,
 * "Differentiable 3D Triangle-Triangle Intersection Energy".
 *
 * The problem is stated as the paper states it: vertex positions,
 * triangles, and a list of candidate triangle pairs.  The candidate list is an INPUT of the hot
 * path; the broad phase that produces it (L51) is a separate call of this library, tt_broad_phase
 * below, whose output can be passed straight in.  For every candidate pair (T_a, T_b)
 * that is not topologically adjacent (shares no vertex index, L11):
 *   1. Moeller's intervals I_a, I_b on the planes' intersection line and
 *      I_c = [t_c^0, t_c^1] = [t_a^0 - t_b^1, t_a^1 - t_b^0]            (L9-15, Eq. 1);
 *      the pair is ACTIVE iff t_c^0 < 0 < t_c^1 (strict; coplanar/touching/degenerate: inactive)
 *   2. energy  T = (t_c^0 t_c^1)^2 for active pairs, 0 otherwise           (L17, Eq. 2)
 *   3. g0 = d t_c^0/dx, g1 = d t_c^1/dx over the pair's 18 DOF; gradient
 *      2 t_c^0 (t_c^1)^2 g0 + 2 t_c^1 (t_c^0)^2 g1                          (L21-24, Eq. 3)
 *      and the outer-product Hessian  c00 g0 g0^T + c11 g1 g1^T + c01 (g1 g0^T + g0 g1^T),
 *      c00 = 2 (t_c^1)^2, c11 = 2 (t_c^0)^2, c01 = 4 t_c^0 t_c^1 * keep     (L26-33, Eq. 4),
 *      `keep` chosen by tt_hess_mode from the eigen-analysis of L47
 *   4. assembly into a per-vertex gradient [nV,3] and a 3x3-block BSR matrix (L51), or the
 *      matrix-free product y = H p.
 *
 * Conventions
 *   - Unless a parameter says HOST, every array pointer is a DEVICE pointer owned by the caller
 *     (e.g. a PyTorch tensor's data_ptr()).  The library never frees or reallocates caller memory.
 *     Workspace is owned by the opaque tt_ctx (cudaMalloc, grow-only, freed by tt_destroy).
 *   - dtype (tt_options.dtype) selects the element type of pos, energy, grad, vals, p, y, tc:
 *     TT_F64 = double, TT_F32 = float.  With TT_F32 the discrete decisions (plane sides, min/max,
 *     t_c^0 < 0 < t_c^1, the FILTER sign) are still taken in fp64 on the fp32-rounded positions, so the
 *     active set equals the fp64 oracle's on those positions (reading A12).
 *   - Layouts: pos [nV,3] row-major; tris [nT,3] int32 vertex ids; pairs [P,2] int32 triangle ids
 *     (pairs[k,0] is T_a, pairs[k,1] is T_b); grad, p, y [nV,3]; BSR: rowptr [nV+1] int32,
 *     colind [nnzb] int32 (ascending within a row), vals [nnzb,3,3] row-major blocks.  The
 *     pattern is the union over active pairs of their 6x6 vertex pairs (both triangles, full --
 *     not only the upper triangle).
 *   - All work is enqueued on `stream` (a cudaStream_t passed as void*, NULL = default stream).
 *     tt_energy, tt_energy_grad_hess and tt_hess_vec are asynchronous; tt_hess_symbolic blocks
 *     until the sizes it hands to the host are known (one host round trip on `stream`, a second one when
 *     some vertex is shared by several touched triangles; its last
 *     kernels may still be running on return, later calls on the same stream are ordered after
 *     them); the *_host call synchronises the stream before returning.
 *   - Outputs are OVERWRITTEN, never accumulated into: grad / y / vals are fully defined on
 *     return (zeros where nothing contributes).
 *   - Errors: every call returns a tt_status (negative = failure) and leaves a message readable
 *     with tt_last_error(ctx).  Index range (tris < nV, pairs < nT) is the caller's
 *     responsibility (undefined behaviour otherwise); sizes, NULLs and state are checked.
 *   - One tt_ctx per stream; a ctx is not thread-safe.  There is no CPU fallback anywhere.
 */
#ifndef TT_H_
#define TT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tt_ctx tt_ctx;

typedef enum {
  TT_OK = 0,
  TT_ERR_INVALID_ARG = -1, /* NULL / negative size / unknown enum / too many rows for int32        */
  TT_ERR_CUDA = -2,        /* a CUDA runtime call failed (message holds cudaGetErrorString)        */
  TT_ERR_NOMEM = -3,       /* workspace allocation failed                                           */
  TT_ERR_CAPACITY = -4,    /* nnzb_capacity smaller than the pattern computed by tt_hess_symbolic   */
  TT_ERR_STATE = -5        /* numeric / H.p call without a matching tt_hess_symbolic, or `pos` changed since */
} tt_status;

typedef enum { TT_F64 = 0, TT_F32 = 1 } tt_dtype;

/* Treatment of Eq. 4's third part ("might be negative"; reading A7):
 *   TT_HESS_EQ4    all three parts as printed
 *   TT_HESS_FILTER third part kept iff L47's quantity 8 t_c^0 t_c^1 (g0.g1) >= 0   (default)
 *   TT_HESS_PSD2   first two parts only (always positive semi-definite)
 *   TT_HESS_PSDPROJ the projection of Eq. 4's per-pair matrix onto the positive semi-definite cone
 *                  (its negative eigenvalue removed): the closest PSD matrix to the pair's Eq. 4
 *   TT_HESS_EXACT  the exact Hessian of T (Eq. 4 "ignores" part of it): Eq. 4, all three parts, plus
 *                  2 t_c^0 (t_c^1)^2 d2 t_c^0 + 2 t_c^1 (t_c^0)^2 d2 t_c^1 -- the second derivatives of the end-points.
 *                  Same BSR pattern; symmetric, in general indefinite.  A variant for Newton's method proper and for
 *                  checking Eq. 4 against it: its kernels are plain (about 9 gradient evaluations per directed
 *                  entry for the assembly, one for H p), not tuned like the Eq. 4 path.                       */
typedef enum { TT_HESS_EQ4 = 0, TT_HESS_FILTER = 1, TT_HESS_PSD2 = 2, TT_HESS_PSDPROJ = 3, TT_HESS_EXACT = 4 } tt_hess_mode;

typedef struct {
  int32_t dtype;      /* tt_dtype                                                                   */
  int32_t hess_mode;  /* tt_hess_mode                                                               */
  double tc_scale;    /* sigma multiplying t_c^0, t_c^1: 1.0 = Eq. 1 (L13); 0.5 = App. A   */
  int32_t device;     /* CUDA device ordinal                                                        */
  int32_t flags;      /* TT_FLAG_* bits, 0 for defaults                                             */
} tt_options;

/* Force every BSR row through the general (shared-vertex) merge path; used by tests to cover it
 * on inputs whose rows would otherwise all take the exclusive-row fast path.                      */
#define TT_FLAG_FORCE_GENERAL_ROWS 1
/* Check every index on the device before it is used: tris < n_verts (tt_energy, tt_hess_symbolic,
 * the *_host call, tt_broad_phase) and pairs < n_tris; an out-of-range index returns
 * TT_ERR_INVALID_ARG with the count in tt_last_error.  Costs one small kernel and one host round
 * trip per call; without the flag out-of-range indices are undefined behaviour (not checked).      */
#define TT_FLAG_VALIDATE_INDICES 2
/* tt_energy_grad_hess and tt_hess_vec replay the branch decisions (lone vertex, min/max order,
 * on-plane flag, active mask) that tt_hess_symbolic recorded at the positions it saw.  By default
 * both calls re-take a 64-bit checksum of `pos` (one read of the array, ~0.03 ms per 6 M vertices;
 * the call enqueues its kernels and then waits for the checksum only, so the GPU does not idle) and
 * return TT_ERR_STATE if the positions have changed since tt_hess_symbolic -- the outputs of such a
 * call are not valid.  This flag skips the check: the caller then guarantees unchanged positions
 * (tt_pcg_solve checks once per solve, not per product).                                          */
#define TT_FLAG_NO_STATE_CHECK 4

typedef struct {
  const void* pos;      int64_t n_verts;   /* [nV,3] dtype                                          */
  const int32_t* tris;  int64_t n_tris;    /* [nT,3]                                                */
  const int32_t* pairs; int64_t n_pairs;   /* [P,2], any order, duplicates allowed                  */
} tt_problem;

/* Create / destroy a context.  tt_create validates options and selects the device. */
tt_status tt_create(const tt_options* opt, tt_ctx** out);
void tt_destroy(tt_ctx* ctx);

/* Steps 1-2 (Eq. 1-2) for every candidate pair.
 *   energy_sum      [1] dtype: sum of T over all pairs (deterministic reduction order)
 *   energy_per_pair [P] dtype or NULL
 *   active_mask     [ceil(P/32)] uint32 or NULL: bit (k & 31) of word k >> 5 set iff pair k active
 *   tc              [P,2] dtype or NULL: (t_c^0, t_c^1), (0,0) for inactive pairs
 *   n_active        [1] int64 on the device or NULL                                               */
tt_status tt_energy(tt_ctx* ctx, const tt_problem* prob, void* energy_sum, void* energy_per_pair,
                    uint32_t* active_mask, void* tc, int64_t* n_active, void* stream);

/* tt_energy without any allocation (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  The same steps 1-2 as tt_energy, total only:
 *   energy_sum [1] dtype DEVICE: sum of T over all pairs -- bit-identical to tt_energy's (same per-CTA partials, same
 *                                fixed-order two-level sum);   n_active [1] int64 DEVICE or NULL.
 * The per-CTA partial sums and counts live in a file-scope device array of the library (1.5 MB, held by every GPU that
 * loads the library until the process exits) instead of the context's growable workspace, so
 *   - n_pairs <= TT_STATIC_MAX_PAIRS, else TT_ERR_CAPACITY (message in tt_last_error) and nothing is launched;
 *   - the call makes no cudaMalloc / cudaFree / allocating library call, no host round trip and no synchronisation: it
 *     enqueues 2-4 kernels on `stream` and returns (TT_FLAG_VALIDATE_INDICES, which needs a round trip, is NOT honoured);
 *   - every call on a device shares the array, whatever the context, and leaves its contents behind: nothing in it has
 *     to start at zero (a call reads only the slots it has written), but two calls that OVERLAP on the GPU (different
 *     streams, or different contexts / threads on the same device) race on it -- serialise them.
 * tt_create obtains the array's device address once, at set-up (the only preparation the call needs).               */
#define TT_STATIC_MAX_PAIRS 16777216 /* 2^24 candidate pairs */
tt_status tt_energy_static(tt_ctx* ctx, const tt_problem* prob, void* energy_sum, int64_t* n_active, void* stream);

/* Symbolic phase of step 4 (L51): classifies the candidates at the current positions, compacts
 * the active pairs (order preserving) and builds the BSR pattern.  Caches all of it in ctx.
 *   nnzb_host     HOST [1]: number of 3x3 blocks the numeric phase will write
 *   n_active_host HOST [1] or NULL
 * Blocks until nnzb is known; the tail of the phase completes asynchronously on `stream`.         */
tt_status tt_hess_symbolic(tt_ctx* ctx, const tt_problem* prob, int64_t* nnzb_host,
                           int64_t* n_active_host, void* stream);

/* Device views of the pattern built by the last tt_hess_symbolic (owned by ctx, valid until the next
 * tt_hess_symbolic / *_host call or tt_destroy): rowptr [nV+1], colind [nnzb].  Passing exactly these pointers as
 * bsr_rowptr / bsr_colind to tt_energy_grad_hess makes that call skip its copy of the pattern into caller memory
 * (the pattern is then shared, not duplicated: 4 (nV + 1 + nnzb) bytes less to move per numeric call).        */
tt_status tt_hess_pattern(tt_ctx* ctx, const int32_t** rowptr, const int32_t** colind, int64_t* nnzb);

/* Steps 2-4 (Eq. 2-4), numeric phase, on the active set cached by tt_hess_symbolic for
 * the same problem (same pointers and sizes, and unchanged positions: TT_ERR_STATE otherwise --
 * the positions are verified by checksum unless TT_FLAG_NO_STATE_CHECK: the call returns once the
 * checksum, enqueued ahead of its kernels, has been read back).
 *   energy_sum [1] dtype; grad [nV,3] dtype or NULL;
 *   bsr_rowptr [nV+1], bsr_colind [nnzb_capacity], bsr_vals [nnzb_capacity,3,3] dtype -- all
 *   three NULL to skip the Hessian.  TT_ERR_CAPACITY if nnzb_capacity < nnzb.                     */
tt_status tt_energy_grad_hess(tt_ctx* ctx, const tt_problem* prob, void* energy_sum, void* grad,
                              int32_t* bsr_rowptr, int32_t* bsr_colind, void* bsr_vals,
                              int64_t nnzb_capacity, void* stream);

/* Matrix-free y = H p with the same Hessian (Eq. 4, same tt_hess_mode) on the cached active set;
 * never forms a block.  p, y: [nV,3] dtype, p != y.  Needs tt_hess_symbolic first, at the same
 * positions (checked like tt_energy_grad_hess).                                                   */
tt_status tt_hess_vec(tt_ctx* ctx, const tt_problem* prob, const void* p, void* y, void* stream);

/* End-to-end convenience with HOST buffers: copies pos/tris/pairs host->device (pinned host
 * memory recommended), runs tt_hess_symbolic + tt_energy_grad_hess into ctx-owned device buffers,
 * and copies the results back.  `prob` holds HOST pointers.
 *   energy_host HOST [1] dtype; grad_host HOST [nV,3] dtype or NULL;
 *   nnzb_host HOST [1]; n_active_host HOST [1] or NULL;
 *   rowptr_host [nV+1] / colind_host [nnzb_capacity] / vals_host [nnzb_capacity,3,3]: HOST, each
 *   may be NULL (the BSR then stays on the device, see tt_bsr_device);
 *   p_host / y_host HOST [nV,3] dtype, both set or both NULL: additionally y = H p (tt_hess_vec).
 * Synchronises `stream`.                                                                          */
tt_status tt_energy_grad_hess_host(tt_ctx* ctx, const tt_problem* prob, void* energy_host,
                                   void* grad_host, int64_t* nnzb_host, int64_t* n_active_host,
                                   int32_t* rowptr_host, int32_t* colind_host, void* vals_host,
                                   int64_t nnzb_capacity, const void* p_host, void* y_host,
                                   void* stream);

/* Broad phase ("we use spatial hashing structure [Pabst et al. 2010] to eliminate
 * redundant computations").  The paper gives no detail, so the operation is
 * defined by its result: ALL pairs i < j of triangles that share no vertex index and whose
 * axis-aligned bounding boxes, each grown by `inflate` (>= 0) on every side, overlap (closed
 * intervals; bounds in fp64 from the stored positions), in lexicographic order -- i.e. a `pairs`
 * array for tt_problem.  Built on a uniform grid, sort based, no atomics.  Cell size =
 * min(largest box extent, max(2 x mean extent, largest / 4)), raised if needed so that no axis has
 * more than 32768 cells; a box is registered in every cell it touches (at most 5 per axis) and a pair
 * is reported only by the cell that owns max(lo_i, lo_j).  The result is deterministic and
 * independent of the grid.
 *   pos [nV,3] dtype, tris [nT,3] int32: DEVICE, read only.   n_pairs_host HOST [1].
 * The pairs stay in ctx (device memory owned by ctx, valid until the next tt_broad_phase or
 * tt_destroy): tt_broad_phase_pairs returns the view, tt_broad_phase_copy copies them to a caller
 * array [capacity,2] (TT_ERR_CAPACITY if too small).  tt_broad_phase blocks until the count is known
 * (two host round trips on `stream`); TT_ERR_INVALID_ARG if the count reaches 2^30.               */
tt_status tt_broad_phase(tt_ctx* ctx, const void* pos, int64_t n_verts, const int32_t* tris,
                         int64_t n_tris, double inflate, int64_t* n_pairs_host, void* stream);
tt_status tt_broad_phase_pairs(tt_ctx* ctx, const int32_t** pairs, int64_t* n_pairs);
tt_status tt_broad_phase_copy(tt_ctx* ctx, int32_t* pairs_out, int64_t capacity, void* stream);

/* Device views of the BSR produced by the last tt_energy_grad_hess_host (owned by ctx, valid
 * until the next *_host call or tt_destroy).                                                      */
tt_status tt_bsr_device(tt_ctx* ctx, const int32_t** rowptr, const int32_t** colind,
                        const void** vals, int64_t* nnzb);

/* ---- The consumer of the assembly ("a GPU-based inexact Newton optimization route";
 * SURVEY.md 8(f) NEXT-2).  The paper gives no detail, so each operation is its textbook definition.
 * All arrays DEVICE; vectors [n_rows,3] dtype; the BSR layout is this library's (3x3 row-major blocks,
 * int32 rowptr / colind, columns ascending within a row).
 *
 * tt_bsr_spmv:     y = (H + shift I) x.   x != y.
 * tt_block_jacobi: minv [n_rows,3,3] dtype = inverse of every 3x3 diagonal block of (H + shift I); a row
 *                  without a stored diagonal block gets I / shift.  The blocks must be non-singular (with a
 *                  PSD hess_mode -- TT_HESS_PSD2 or TT_HESS_PSDPROJ -- any shift > 0 guarantees it).
 * tt_pcg_solve:    preconditioned conjugate gradients (Hestenes-Stiefel recurrences) for (H + shift I) x = b
 *                  from x_0 = 0, stopped before step k when |r_k|_2 <= rtol |b|_2 or after max_iter steps.
 *                    vals != NULL : H is the BSR matrix (rowptr, colind, vals)            [assembled back end]
 *                    vals == NULL : H p is tt_hess_vec on `prob` (needs tt_hess_symbolic at the current
 *                                   positions; checked once per solve, TT_ERR_STATE)       [matrix-free back end]
 *                    minv         : tt_block_jacobi's output, or NULL for plain CG
 *                  prob->n_verts is the number of rows.  All scalars of the recurrence live on the device and
 *                  every dot product is a fixed-order tree (deterministic; no floating-point atomics); with
 *                  rtol > 0 the host looks at the residual every `check_every` steps (0 = 8), the iterate is
 *                  frozen ON THE DEVICE at the first step that meets the bound, so x does not depend on
 *                  check_every.  iters_host / relres_host (HOST [1], may be NULL): steps taken and
 *                  |r|_2 / |b|_2 of the recurred residual; if either is given the call synchronises `stream`. */
typedef struct {
  int32_t max_iter;     /* >= 0                                                                       */
  int32_t check_every;  /* host convergence checks (only if rtol > 0); 0 = every 8 steps              */
  double rtol;          /* >= 0; 0 = run exactly max_iter steps, fully asynchronous                   */
  double shift;         /* mu >= 0 added to the diagonal (Levenberg-Marquardt / "stay close" term)    */
} tt_pcg_options;
tt_status tt_bsr_spmv(tt_ctx* ctx, int64_t n_rows, const int32_t* rowptr, const int32_t* colind,
                      const void* vals, double shift, const void* x, void* y, void* stream);
tt_status tt_block_jacobi(tt_ctx* ctx, int64_t n_rows, const int32_t* rowptr, const int32_t* colind,
                          const void* vals, double shift, void* minv, void* stream);
tt_status tt_pcg_solve(tt_ctx* ctx, const tt_problem* prob, const int32_t* rowptr, const int32_t* colind,
                       const void* vals, const void* minv, const void* b, void* x,
                       const tt_pcg_options* opt, int32_t* iters_host, double* relres_host, void* stream);

/* ---- One damped inexact-Newton step on E(x) = sum of T over a fixed candidate list, and the untangling loop around
 * it ("inexact Newton optimization route", L41-43 / Fig. 2; SURVEY.md 8(f) NEXT-2 "line search on
 * tt_energy", NEXT-4).  The paper gives no formula, tolerance or step rule; reading A16 fixes the textbook
 * choice (line-search Newton-CG with a Levenberg-Marquardt shift):
 *     E0, g, H  at x (this ctx's hess_mode: use a PSD one, TT_HESS_PSD2 or TT_HESS_PSDPROJ, so that H + mu I is SPD)
 *     d         = pcg.max_iter / pcg.rtol steps of block-Jacobi PCG on (H + mu I) d = g from 0   (tt_pcg_solve)
 *     alpha     = first of 1, 1/2, 1/4, ... (at most max_backtrack halvings) with
 *                 E(x - alpha d) <= E0 - armijo_c1 alpha g.d                                      (tt_energy)
 *     x        <- x - alpha d, IN PLACE; x is left unchanged when no alpha is accepted (accepted = 0).
 * Everything runs on the device; the host sees the scalars of `report` (one round trip per trial step length).
 *   pos DEVICE [nV,3] dtype, read AND written; tris, pairs DEVICE as in tt_problem; report HOST [1].
 * The call invalidates the state cached by tt_hess_symbolic (the positions have moved).
 * tt_untangle: repeat { candidates = tt_broad_phase(pos, inflate); tt_newton_step } until no pair is active, a step
 * is rejected, or max_steps steps were taken.  history HOST [max_steps] (one report per step taken), steps_host HOST [1]. */
typedef struct {
  double mu;              /* > 0: Levenberg-Marquardt shift added to the diagonal                                  */
  double armijo_c1;       /* in (0, 1), e.g. 1e-4                                                                   */
  int32_t max_backtrack;  /* >= 0: halvings of alpha after the full step                                            */
  int32_t matrix_free;    /* 0: assemble the BSR, block-Jacobi PCG; 1: CG on tt_hess_vec, no BSR, no preconditioner */
  tt_pcg_options pcg;     /* max_iter, rtol, check_every of the inner solve (its shift is ignored: mu is used)      */
  int32_t membrane;       /* 0: E = E_T;  1: E = E_T + E_m, the mesh of the last tt_membrane_build (see below)      */
  int32_t reserved;       /* 0                                                                                       */
} tt_newton_options;
typedef struct {
  double energy0, energy1;  /* E at x before / after the step (equal if rejected)                                   */
  double grad_norm;         /* |g|_2 at x                                                                           */
  double gd;                /* g . d  (> 0 for a descent step x - alpha d)                                          */
  double alpha;             /* accepted step length, 0 if rejected or nothing is active                             */
  double pcg_relres;        /* |r|_2 / |g|_2 of the inner solve                                                     */
  int64_t n_pairs, n_active, nnzb;
  int32_t pcg_iters, backtracks, accepted, reserved;
  double energy_membrane;   /* E_m's share of energy1 (0 without the membrane term)                                 */
} tt_newton_report;
tt_status tt_newton_step(tt_ctx* ctx, void* pos, int64_t n_verts, const int32_t* tris, int64_t n_tris,
                         const int32_t* pairs, int64_t n_pairs, const tt_newton_options* opt,
                         tt_newton_report* report_host, void* stream);
tt_status tt_untangle(tt_ctx* ctx, void* pos, int64_t n_verts, const int32_t* tris, int64_t n_tris, double inflate,
                      int32_t max_steps, const tt_newton_options* opt, tt_newton_report* history_host,
                      int32_t* steps_host, void* stream);

/* ---- The membrane term of the untangling demo (Fig. 2: the paper optimises
 * meshes "from an invalid to a valid state" inside a simulation whose elastic model it does not give; DESIGN.md
 * reading A18 takes the simplest textbook one, springs on the mesh's own edges):
 *     E_m(x) = k/2 sum over the mesh's unique edges (i, j) of (|x_i - x_j| - L_ij)^2,   L_ij = |r_i - r_j| at rest,
 *     grad_i = k sum_j (|d| - L) n,       d = x_i - x_j,  n = d / |d|,
 *     H_m p  at i = sum_j K (p_i - p_j),  K = k [ n n^T + max(0, 1 - L / |d|) (I - n n^T) ]
 * (K = the edge's exact Hessian block with the negative part of a compressed spring clamped to zero, so H_m is PSD).
 * An edge whose two ends coincide (|d| = 0) has no direction and contributes nothing.
 *
 * tt_membrane_build:       builds the vertex -> neighbour adjacency of `tris` (sort + unique of the half-edges; an
 *                          edge shared by several triangles counts once, a degenerate edge i == i is dropped) and the
 *                          rest lengths from rest_pos.  rest_pos DEVICE [n_verts,3] dtype, tris DEVICE [n_tris,3]
 *                          int32; both are only read during the call.  The result is owned by ctx and replaces the
 *                          previous one; one host round trip on `stream` (the number of unique half-edges).
 * tt_membrane_energy_grad: energy DEVICE [1] DOUBLE (whatever the dtype), grad DEVICE [n_verts,3] dtype or NULL.
 * tt_membrane_hess_vec:    y = H_m(pos) p;  pos, p, y DEVICE [n_verts,3] dtype, p != y.
 * Both need a preceding tt_membrane_build (TT_ERR_STATE otherwise) and use ITS n_verts.  One thread per vertex walks
 * the neighbours in ascending order: no atomics, results bit-reproducible; arithmetic in fp64 for both dtypes.
 * With tt_newton_options.membrane = 1, tt_newton_step / tt_untangle minimise E_T + E_m: g = g_T + g_m, the inner
 * solve applies H_T p (assembled or matrix-free) + H_m p + mu p, and the preconditioner is the inverse of the
 * MEMBRANE's diagonal blocks + mu I in both back ends (TT_ERR_STATE if the built mesh has another n_verts).         */
tt_status tt_membrane_build(tt_ctx* ctx, const void* rest_pos, int64_t n_verts, const int32_t* tris, int64_t n_tris,
                            double stiffness, void* stream);
tt_status tt_membrane_energy_grad(tt_ctx* ctx, const void* pos, double* energy, void* grad, void* stream);
tt_status tt_membrane_hess_vec(tt_ctx* ctx, const void* pos, const void* p, void* y, void* stream);

/* Counters of the last tt_hess_symbolic: what[0]=n_active, [1]=directed entries (2*n_active),
 * [2]=touched triangles, [3]=blocks written directly (exclusive rows), [4]=blocks produced by the
 * general-row merge, [5]=merge records, [6]=nnzb, [7]=kernels launched by this ctx so far (CUB calls
 * counted by the kernels they launch), [8]=slots of the work partition, [9]=triangles with more than 32
 * partners that were split into parts, [10]=parts, [11]=such triangles that could not be split (rounds of
 * their own, long-triangle kernels), [12]=rounds of the work partition (one warp each in K4 / K6: a round holds at
 * most 32 directed entries, so [1] / (32 [12]) is the lane fill).                                     */
tt_status tt_stats(const tt_ctx* ctx, int64_t* what, int32_t n);

/* Device durations (CUDA events on the caller's stream) of the most recent launch of the three
 * large kernels: ms[0] = classification (K1), ms[1] = assembly (K4), ms[2] = H.p (K6); -1 if the
 * kernel has not run.  Blocks until those launches have finished.                                 */
tt_status tt_kernel_ms(tt_ctx* ctx, float* ms, int32_t n);
/* The same, averaged over the launches recorded since the last reset (the library keeps the events of
 * the last 64 launches of each kernel, so a timed loop needs no synchronisation inside it):
 *   ms HOST [n]: mean duration, -1 if none; launches HOST [n] or NULL: how many were averaged;
 *   reset != 0 forgets the recorded launches afterwards.  Blocks until those launches have finished. */
tt_status tt_kernel_ms_mean(tt_ctx* ctx, float* ms, int32_t* launches, int32_t n, int32_t reset);

/* Diagnostic (not on the hot path): measured vector-FMA issue rate of `device`, FMA = 2 flop.
 *   tflops HOST [2]: [0] = fp64 (DFMA), [1] = fp32 (FFMA).  Runs ~10 ms of register-only FMA
 *   chains on the default stream and blocks until done.  bench.py reports it beside the derived
 *   ALU peak.                                                              */
tt_status tt_probe_peaks(int32_t device, double* tflops);

/* Diagnostic (not on the hot path): useful bytes per second of RANDOM gathers from a 144 MB array (the size of the
 * 6 M-vertex fp64 position array of BASELINE configs[4]; larger than the L2), one item per thread:
 *   gbs HOST [2]: [0] = 24-byte items (one vertex), [1] = 72-byte items (the three vertices of a soup triangle), GB/s.
 * This is the ceiling that the access pattern of the classification (K1) and H.p (K6) kernels can reach on this
 * memory system -- sector granularity and DRAM row locality included; bench.py reports it beside the copy bandwidth. */
tt_status tt_probe_gather(int32_t device, double* gbs);

const char* tt_status_string(tt_status s);
const char* tt_last_error(const tt_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TT_H_ */
