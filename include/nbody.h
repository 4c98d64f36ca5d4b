/*
 * include/nbody.h -- C ABI of libnbody.so: the B200 (sm_100a) hot path of the block-time-step Hermite direct
 * N-body method benchmarked in arXiv:1312.1789.
 *
 * Method statement.  The paper names the scheme only -- "individual hierarchically block time-steps with the
 * high (4th, 6th and 8th) order Hermite integration schemes" (abstract), forces on the GPU
 * (section 2), "mixed (fp32 + fp64) precision" (Fig. 1 caption) -- and prints no
 * formula.  The operations below are therefore defined by DESIGN.md section 3 (readings R1..R12, restating
 * SURVEY.md 8(c) items c-1..c-14), each cited per call.
 *
 * Conventions (all calls)
 *   - G = 1, potential negative, one Plummer softening eps2 for all pairs (R3, R11).
 *   - `order` p is 4, 6 or 8; K = p/2 force derivatives (acc, jerk | +snap | +crackle).
 *   - Unless a parameter is marked HOST, every array pointer is a DEVICE pointer into caller-owned memory,
 *     fp64, contiguous, 8-byte aligned (int32 arrays 4-byte aligned; anything else is NBODY_EINVAL); 3-vectors are
 *     row-major [n][3].  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     nbody_predict / nbody_force / nbody_force_static / nbody_nearest / nbody_correct / nbody_initial_dt /
 *     nbody_get_predicted / nbody_pack_rows / nbody_unpack_rows only enqueue work and return: they never synchronise
 *     and never allocate (all scratch is sized in nbody_create).  Calls that return a value to the host say so (nbody_next_block, nbody_run_blocks, *_host);
 *     with the "validate" option on, nbody_force and nbody_correct also synchronise (debug mode).
 *   - The ctx owns scratch only (packed j-store, split partials, control block, staging for the *_host calls).  It
 *     never frees or keeps caller memory.  A ctx is bound to the device given at creation: every call switches to that
 *     device and restores the caller's current device on return.  A ctx is not thread-safe.
 *   - Every call returns an int status: NBODY_OK (0) or a negative NBODY_E* code; nothing aborts, throws or
 *     prints.  nbody_strerror() maps a code to a static string.
 *   - There is no CPU fallback anywhere: without a CUDA device nbody_create() returns NBODY_ECUDA.
 */
#ifndef NBODY_H_
#define NBODY_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NBODY_OK       0
#define NBODY_EINVAL  (-1) /* bad argument: order, sizes, NULL where required, eps2 < 0, misaligned pointer,
                              dt range, a failed "validate" check                                              */
#define NBODY_ESTATE  (-2) /* call order: force before predict, force order > order of the last predict       */
#define NBODY_ECUDA   (-3) /* a CUDA runtime call or launch failed; see nbody_last_cuda_error()               */
#define NBODY_ENOMEM  (-4) /* device or host allocation failed                                                */
#define NBODY_ESCRATCH (-5) /* nbody_force_static: the launch needs more than NBODY_FORCE_STATIC_SCRATCH_BYTES     */

typedef struct nbody_ctx nbody_ctx;

/* ABI version of this header (bumped on any signature change). */
int nbody_abi_version(void);

/* Static description of `code`; never NULL. */
const char *nbody_strerror(int code);

/* Create a context for up to n_capacity particles on CUDA device `device`.  Allocates, with cudaMalloc, the packed
 * j-store (6 planes x 16 B x n_capacity rounded up to the 256-particle j-tile; 4 of them in use unless diff_mode is
 * 1), the j-split scratch (rows of 13 doubles: max(4 SMs x 1024, 4 n_capacity) rows, at most 512 MB; the split
 * heuristic never asks for more, so nbody_force never allocates), the selection's candidate list (4 B x n_capacity)
 * and small control blocks.  *out is set only on
 * success.  Synchronises the device; the caller's current device is left unchanged. */
int nbody_create(nbody_ctx **out, int64_t n_capacity, int device);

/* Device bytes nbody_create(n_capacity) allocates on a 148-SM part (j-store + split scratch + selection candidates + control blocks);
 * -1 for an invalid capacity.  HOST arithmetic only. */
int64_t nbody_workspace_bytes(int64_t n_capacity);

/* Free everything the ctx owns (synchronises the device first).  NULL is a no-op. */
int nbody_destroy(nbody_ctx *ctx);

/* The cudaError_t (as int) of the last failing CUDA call made through this ctx, 0 if none. */
int nbody_last_cuda_error(const nbody_ctx *ctx);

/* Tuning / evidence knobs (host-side integers; unknown key -> NBODY_EINVAL).
 *   "diff_mode"   0 = literal: d = fl32(x_j - x_i), subtraction in fp64 (DADD + F2F)          [default]
 *                 1 = double-single: x = hi + lo (two fp32), d = (hi_j - hi_i) + (lo_j - lo_i)  (R10 note)
 *   "dt_criterion_order" pc: dt = eta (A^(1)/A^(pc-2))^(1/(pc-3)) evaluated on the lowest pc derivatives at t_now.
 *                 0 = automatic [default]: pc = p for order 4, pc = 4 (Aarseth's formula) for orders 6 and 8 (R8b:
 *                 only derivatives the force call computes directly decide the step; for p = 6 the fourth entry is
 *                 the mean crackle (s1 - s0)/h).  4 | 6 | 8 = pc = min(p, value); value = p is the order-p
 *                 criterion of R8, which fp32 force noise collapses for p >= 6 (R8b): fp64 forces only.
 *   "force_split" 0 = automatic j-split, S >= 1 = force exactly S j-splits (tests: split independence); a forced S
 *                 with S * n_act beyond the split scratch makes nbody_force return NBODY_EINVAL
 *   "force_lanes" 0 = automatic, else force the j-lanes-per-CTA variant (1, 2, 4, ..., 256)
 *   "geometry_n_act" 0 = the call's n_act decides the j-lane variant and the j-split [default]; G > 0 = decide as if the
 *                 call had G active particles (G >= n_act).  An i-sharded rank passes its slice of the active list and
 *                 G = the size of the whole block: every particle is then summed in exactly the order of the unsharded
 *                 call, so the shards reproduce it bit for bit.
 *   "validate"    0 = off [default]; 1 = debug mode: nbody_force checks on the device that active_idx is strictly
 *                 ascending (hence unique) and in [0, n), nbody_correct additionally that t[i] + dt[i] == t_now for
 *                 every active i; a violation returns NBODY_EINVAL before any arithmetic.  Synchronises `stream`.
 *   "use_graph"   1 = nbody_run_blocks replays its launches as CUDA graphs [default]; 0 = plain launches
 *   "use_fused"   N1, fused small-block step.  0 [default] = every block of a run goes through the general step (four
 *                 launches: selection, predictor, force, reduce + corrector).  1 = blocks that fit one i-tile (n_act <=
 *                 1024) go through TWO launches: selection + a persistent kernel whose CTAs predict their j-tiles on the
 *                 fly from the raw fp64 state (TMA-staged; the bit-exact predictor arithmetic) before the pair loop, and
 *                 whose last CTA sums the j-split partials and runs the corrector; a larger block ends such a batch and is
 *                 taken by the general step.  Bit-identical results either way.  Off by default because it is not yet
 *                 faster (profiles/r02_latency.md: one 53 KB raw stage in flight per SM is latency-bound).
 *   "corrector_order_limit" R15, corrector order limiter (a reading added by this build; the paper is silent): 0 = off
 *                 [default]; 1 = the corrector's velocity line is a sum of K = p/2 quadrature terms T_1 = h/2 (a0+a1),
 *                 T_2 = w2 (j0-j1), T_3 = w3 (s0+s1), T_4 = w4 (c0-c1); M = the number of leading terms whose norms do not
 *                 increase; a particle with M < K gets its x1, v1 from the corrector of order 2M (M = 1: trapezoid); if
 *                 already the first end-point correction h/2 (a1 - a0) exceeds h a0 (an acceleration spike on the end
 *                 point), M = 0: x1, v1 are the particle's own fp64 Taylor prediction and the end point is not used.  On
 *                 smooth steps the terms fall off geometrically and nothing changes (bit-identical results); when an
 *                 encounter sits on an end point they grow, and the higher ones are dropped instead of summed.  Stored
 *                 derivatives, criterion and new dt are unchanged.  Bit-exact against the oracle's limit_order.
 *   "step_reject_ratio" R14, a-posteriori step rejection (a reading added by this build; the paper is silent):
 *                 0 = off [default], the textbook scheme.  R = 2^r in [2, 2^20]: if the criterion evaluated at the END of
 *                 a particle's step asks for dt_new <= h/R and h/R >= dt_min, nbody_correct does not take the step: x, v,
 *                 a_derivs, pot_state and t of that particle keep their values and only dt := h/R is written.  The
 *                 particle is then due at t + h/R, BEFORE the current block time: nbody_next_block / nbody_run_blocks pick
 *                 it next and nbody_predict extrapolates everybody else back to that time (tau < 0 is legal).  Guards the
 *                 end-point quadrature against encounters the start-of-step criterion could not see (a perturber at its
 *                 closest approach on the end point of a long step: end-point derivatives m v^k / r^(k+2) times h^(k+1)).
 *                 Bit-exact against the oracle's reject_ratio.  Count: nbody_rejected_steps / nbody_run_result.rejected.
 */
int nbody_set_option(nbody_ctx *ctx, const char *key, int64_t value);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_predict -- a-2, Taylor predictor of ALL n particles to the block time t_now (R5 = SURVEY c-5;
 * PAPER.md:43 "Hermite integration scheme" implies predict-evaluate-correct).
 *   tau = t_now - t[i];  D_k = a_derivs[k] = a^(k)(t_i), k = 0 .. order-3 (entries above that are ignored and
 *   may be NULL):
 *     x_p = x + v tau + Sum_k D_k tau^(k+2)/(k+2)!      v_p = v + Sum_k D_k tau^(k+1)/(k+1)!
 *     a_p = Sum_k D_k tau^k/k!  (order >= 6)            j_p = Sum_{k>=1} D_k tau^(k-1)/(k-1)!  (order == 8)
 *   evaluated in fp64 by Horner, innermost term first, with c_k = tau / k, no FMA contraction (bit-exact
 *   against the oracle, R12).  Results go to the ctx-owned packed j-store: x_p as fp64, v_p a_p j_p m rounded
 *   to fp32 (round-to-nearest-even).  The j-store stays valid until the next nbody_predict on this ctx.
 *   a_derivs is a HOST array of 6 device pointers; it is read during the call only.
 * Errors: EINVAL (order, n < 0, n > capacity, NULL t/m/x/v or NULL a_derivs[k] for k <= order-3).
 * n == 0 is a successful no-op that marks the j-store as holding 0 particles.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_predict(nbody_ctx *ctx, int64_t n, double t_now, int order,
                  const double *t, const double *m, const double *x, const double *v,
                  const double *const a_derivs[6] /* HOST array of device pointers */, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_force -- a-3 (+ a-3b), the O(n_act * n) hot loop (R1..R4, R10 = SURVEY c-1..c-4, c-12; PAPER.md:43,
 * PAPER.md:65 eq. (1) alpha-term; mixed precision PAPER.md:31).
 *   For each active i (index into the j-store of the last nbody_predict), over all j != i (excluded BY INDEX):
 *     r = x_j - x_i (fp64 subtraction, rounded to fp32), v = v_j - v_i, a = a_j - a_i, jk = j_j - j_i (fp32)
 *     s2 = r.r + eps2;  q = m_j / s2^(3/2);  alpha = (r.v)/s2;  beta = (v.v + r.a)/s2 + alpha^2
 *     gamma = (3 v.a + r.jk)/s2 + alpha (3 beta - 4 alpha^2)
 *     A = q r;  J = q v - 3 alpha A;  S = q a - 6 alpha J - 3 beta A;  C = q jk - 9 alpha S - 9 beta J - 3 gamma A
 *     acc = Sum A, jerk = Sum J, snap = Sum S (order >= 6), crackle = Sum C (order == 8), pot = -Sum m_j/sqrt(s2)
 *   fp32 pair arithmetic (MUFU rsqrt), per-thread fp32 partial sums over <= 64 consecutive j, then fp64.
 *   Outputs are in ACTIVE-LIST order: acc, jerk, snap, crackle [n_act][3], pot [n_act], fully overwritten.
 *   snap may be NULL when order < 6, crackle when order < 8 (they are not written then).
 *   active_idx: device int32 [n_act], each in [0, n), unique (ascending recommended, not required; checked only
 *   with the "validate" option, otherwise an out-of-range index reads out of bounds).
 *   Deterministic: the same inputs and options give bit-identical outputs run to run, and the result for a particle
 *   depends on (j-lane variant, j-split) only, never on the other members of the active list.
 *   Coincident particles: a DIFFERENT particle at the same position is included (R2); with eps2 > 0 it adds exactly 0
 *   to acc/jerk/snap/crackle and -m/eps to pot; with eps2 == 0 the pair term is 0 x inf and the outputs of both
 *   particles are NaN (undefined by the method; not an error code).  The zero-mass pads that fill the last j-tile are
 *   excluded by index, so no real particle can collide with them.
 * Errors: EINVAL (order, n_act < 0, n_act > n, eps2 < 0 or NaN, 0 < eps2 < 1.18e-38 (flushes to 0 in fp32), NULL or
 * misaligned pointer, validation failure), ESTATE (no predict yet, or order > the order of the last predict).
 * n_act == 0 is a successful no-op.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_force(nbody_ctx *ctx, const int32_t *active_idx, int64_t n_act, int order, double eps2,
                double *acc, double *jerk, double *snap, double *crackle, double *pot, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_force_static -- nbody_force (a-3 + a-3b, same arithmetic, arguments, layout and errors) for callers that may
 * not allocate: code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  The call performs no
 * cudaMalloc / cudaFree and calls no allocating library routine, and the fp64 partials [S][NC][n_act] of a j-split
 * launch (NC = 3 * order / 2 + 1) go to a STATIC device array of NBODY_FORCE_STATIC_SCRATCH_BYTES inside libnbody.so
 * instead of the ctx's scratch.  Every GPU that loads the library holds that array until the process exits.
 *   Limit: a launch that needs S * NC * n_act * 8 bytes > NBODY_FORCE_STATIC_SCRATCH_BYTES returns NBODY_ESCRATCH and
 *   launches nothing (outputs untouched).  S is the j-split count of the same geometry rule nbody_force uses, so the
 *   outputs are bit-identical to nbody_force's.  Every block of n_act <= 1024 particles fits on a B200 (one i-tile,
 *   S <= 148 SMs: 148 * 13 * 1024 * 8 = 15 761 408 bytes); larger blocks fit when S * NC * n_act <= 2 097 152
 *   (unsplit launches, S == 1, use no scratch and always fit); "force_split" can push S beyond the limit.
 *   Sharing: all calls on a device use the same array, and it keeps the last call's contents.  Nothing in it has to
 *   start at zero (the call writes every entry before it reads it), so consecutive calls on ONE stream are safe; two
 *   calls that overlap on the GPU (different streams, or different ctxs on one device) RACE -- order them yourself.
 *   Set-up: the first call on a device resolves the array's device address (cudaGetSymbolAddress, no allocation); a
 *   call with n_act == 0 does only that, so issue one after nbody_create to keep it out of a capture.
 * The ctx, its j-store and nbody_predict are as for nbody_force: nbody_create allocates, so it comes before.
 * ---------------------------------------------------------------------------------------------------------- */
#define NBODY_FORCE_STATIC_SCRATCH_BYTES 16777216 /* 16 MiB */
int nbody_force_static(nbody_ctx *ctx, const int32_t *active_idx, int64_t n_act, int order, double eps2,
                       double *acc, double *jerk, double *snap, double *crackle, double *pot, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_correct -- a-4, Hermite corrector + Aarseth-style block time step with power-of-two quantisation for the
 * active particles (R6..R9 = SURVEY c-6..c-9; "hierarchically block time-steps").
 *   For each active i, h = dt[i], 0 = stored state at t[i], 1 = force-call values at t_now:
 *     compact two-point Hermite corrector for v then x (R6), interpolated a^(K..2K-1)(t_now) (R7),
 *     dt_crit = eta (A^(1)/A^(p-2))^(1/(p-3)), A^(k) = sqrt(|a^(k-1)||a^(k+1)| + |a^(k)|^2) (R8),
 *     dt_new = 2^floor(log2 dt_crit) by exact comparisons; <= 2 dt_old; doubling only if t_now is a multiple
 *     of the doubled step; clamped to [dt_min, dt_max] (R9).
 *   In place: x, v, a_derivs[0..order-1], pot_state, t := t_now, dt := dt_new for the active rows.
 *   fp64, no FMA contraction, IEEE div/sqrt, operation order as DESIGN.md section 3 states: bit-exact vs oracle.
 *   acc .. pot are the force-call outputs in active-list order.  a_derivs is a HOST array of 8 device pointers,
 *   entries 0 .. order-1 required.  dt_min, dt_max must be exact powers of two.
 * Errors: EINVAL (order, n_act < 0, NULL or misaligned pointer, eta <= 0, dt_min/dt_max not powers of two or
 * dt_min > dt_max, (max(|log2 dt_min|, |log2 dt_max|) + 1) (pc - 3) > 1022 for the criterion order pc in use (the
 * exact power-of-two comparison of R9 stays inside the fp64 exponent range), validation failure).
 * n_act == 0 is a successful no-op.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_correct(nbody_ctx *ctx, const int32_t *active_idx, int64_t n_act, int order,
                  double t_now, double eta, double dt_min, double dt_max,
                  double *t, double *dt, double *x, double *v,
                  double *const a_derivs[8] /* HOST array of device pointers */, double *pot_state,
                  const double *acc, const double *jerk, const double *snap, const double *crackle,
                  const double *pot, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_initial_dt -- start-up step of the bootstrap (R9b = SURVEY c-10): dt_i = 2^floor(log2(eta_s |a|/|j|))
 * clamped to [dt_min, dt_max]; |j| == 0 -> dt_max.  acc, jerk, dt: device [n][3], [n][3], [n].  Bit-exact.
 * Errors: EINVAL (n < 0, eta_s <= 0, dt_min/dt_max not powers of two, dt_min > dt_max, |log2| > 1021, NULL pointer).
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_initial_dt(nbody_ctx *ctx, int64_t n, const double *acc, const double *jerk,
                     double eta_s, double dt_min, double dt_max, double *dt, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_next_block -- a-1, block selection on the device (R9c = SURVEY c-11): t_next = min_i (t[i] + dt[i])
 * (exact for dyadic values); active = { i : t[i] + dt[i] == t_next } ascending.  Writes active_idx (device
 * int32, capacity n: entries [0, n_act) are the block, entries at and beyond n_act are scratch and may be
 * overwritten) and returns t_next and n_act through HOST pointers; this call synchronises `stream`.
 * One kernel, one pass, no grid barrier: every CTA lists the particles of its chunk due at the chunk's own minimum;
 * the last CTA to finish takes the global minimum and concatenates the lists that belong to it, in order.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_next_block(nbody_ctx *ctx, int64_t n, const double *t, const double *dt,
                     int32_t *active_idx, double *t_next_host, int64_t *n_act_host, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_nearest -- SURVEY 8(f) N4 "nearest-neighbour output" (reading R16, oracle c-17; not in PAPER.md, which only
 * names the neighbour scheme of its second code).  For each active i (index into the j-store of the last
 * nbody_predict) the nearest OTHER particle (excluded by index) at the predicted positions:
 *     d = fl32(x_j - x_i), each component formed in fp64 (the force kernel's differences, R10);
 *     r2 = fma(dz, dz, fma(dy, dy, dx * dx)) in fp32;  the smallest r2 wins, ties go to the lowest j.
 *   nn_idx: device int32 [n_act] (-1 when n == 1); nn_r2: device fp64 [n_act] holding the fp32 value (+inf when
 *   n == 1), both in ACTIVE-LIST order.  Bit-exact against the oracle; independent of the launch geometry.
 *   Uses the ctx's split scratch (as nbody_force does): order it with the other calls on this ctx by the stream.
 * Errors: EINVAL (n_act < 0, n_act > n, NULL or misaligned pointer, validation failure), ESTATE (no predict yet),
 * ENOMEM (n_act * 8 bytes beyond the split scratch: cannot happen below 67 M particles).  n_act == 0 is a no-op.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_nearest(nbody_ctx *ctx, const int32_t *active_idx, int64_t n_act, int32_t *nn_idx, double *nn_r2, void *stream);

/* count_host[0] = steps refused by the "step_reject_ratio" rule, count_host[1] = steps taken with a lower-order corrector
 * ("corrector_order_limit"), since the counters were last reset (nbody_run_blocks resets them at the start of every run);
 * reset != 0 clears them.  count_host is a HOST array of 2; synchronises `stream`. */
int nbody_rejected_steps(nbody_ctx *ctx, int reset, int64_t *count_host, void *stream);

/* Test hook: export the packed j-store of the last predict (n particles) into plain arrays.  xp fp64 [n][3];
 * vp, ap, jp fp32 [n][3] (ap/jp may be NULL; ap requires order >= 6, jp order == 8 else EINVAL); m32 fp32 [n]. */
int nbody_get_predicted(nbody_ctx *ctx, double *xp, float *vp, float *ap, float *jp, float *m32, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_force_host -- the same path (predict at t_now, then force) with HOST buffers: every pointer below is a
 * HOST pointer (pageable or pinned).  Copies t, m, x, v, D_0..D_{order-3} and active_idx to ctx-owned device
 * staging, runs nbody_predict + nbody_force, copies acc/jerk/snap/crackle/pot back, and returns after the
 * results are in host memory (synchronises).  Used for the end-to-end measurement; results are identical to
 * the device-pointer calls.  h2d_bytes / d2h_bytes (may be NULL) receive the bytes copied each way.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_force_host(nbody_ctx *ctx, int64_t n, double t_now, int order,
                     const double *t, const double *m, const double *x, const double *v,
                     const double *const a_derivs[6] /* HOST array of HOST pointers */,
                     const int32_t *active_idx, int64_t n_act, double eps2,
                     double *acc, double *jerk, double *snap, double *crackle, double *pot,
                     int64_t *h2d_bytes, int64_t *d2h_bytes);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_step_host -- ONE WHOLE BLOCK STEP (a-1 .. a-4: selection, predict, force, correct) with HOST state: every
 * pointer is a HOST pointer.  Copies t, dt, m, x, v, a_derivs[0..order-1], pot_state to ctx-owned staging, runs
 * nbody_next_block + nbody_predict + nbody_force + nbody_correct (the same kernels), copies the updated t, dt, x, v,
 * a_derivs[0..order-1], pot_state back IN PLACE and returns when they are in host memory.  *t_next_host and
 * *n_act_host receive the block time and size.  a_derivs is a HOST array of 8 HOST pointers.  This is the call
 * the end-to-end measurement times (host<->device copies inside the timed region).
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_step_host(nbody_ctx *ctx, int64_t n, int order, double eps2, double eta, double dt_min, double dt_max,
                    double *t, double *dt, const double *m, double *x, double *v,
                    double *const a_derivs[8] /* HOST array of HOST pointers */, double *pot_state,
                    double *t_next_host, int64_t *n_act_host, int64_t *h2d_bytes, int64_t *d2h_bytes);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_run_blocks -- N2, the device-driven block step ("individual hierarchically block time-steps";
 * PAPER.md:65 eq. (1): the latency term).  Runs whole block steps a-1 .. a-4 (selection, predict, force, correct)
 * back to back WITHOUT the host learning n_act: the selection kernel leaves t_next, n_act and the force geometry in a
 * device control block, the other kernels read them there (persistent grids of fixed size), and the five launches of
 * one block step (select, predict, force, split reduce, correct) are replayed as ONE CUDA graph.  The host looks at the control block only every 4 .. 64 block
 * steps.  A block is executed iff t_next <= t_end, n_act <= max_n_act and fewer than max_blocks blocks have run; the
 * first block that is not executed ends the run (the state is then exactly the state before that block).
 * Results are bit-identical to the same blocks run through nbody_next_block + nbody_predict + nbody_force +
 * nbody_correct (same kernels, same geometry rule).
 *   state t, dt, m, x, v, a_derivs[0..order-1], pot_state: as nbody_correct (in/out, device).
 *   active_idx (int32 [n]), acc, jerk, snap, crackle ([n][3]), pot ([n]): caller-owned device scratch of the step.
 *   res (HOST): blocks executed, pairs = Sum n_act * n, the block that stopped the run (t_next, n_act_next),
 *   stop_reason (1 = t_next > t_end, 2 = n_act > max_n_act, 3 = max_blocks reached) and the executed blocks counted
 *   by floor(log2 n_act).
 * The run executes on a ctx-owned stream ordered after everything queued on `stream`; `stream` is made to wait for the
 * run.  Synchronises.  Requires diff_mode 0.
 * Errors: as nbody_correct / nbody_force, plus EINVAL for max_blocks < 0 or max_n_act < 1; ESTATE for diff_mode 1.
 * ---------------------------------------------------------------------------------------------------------- */
typedef struct nbody_run_result {
    int64_t blocks;
    int64_t pairs;
    double  t_next;
    int64_t n_act_next;
    int32_t stop_reason;
    int32_t reserved;
    int64_t rejected;       /* steps refused by the "step_reject_ratio" rule during this run */
    int64_t limited;        /* steps taken with a lower-order corrector ("corrector_order_limit") during this run */
    int64_t hist_log2[40];
} nbody_run_result;

int nbody_run_blocks(nbody_ctx *ctx, int64_t n, int order, double eps2, double eta, double dt_min, double dt_max,
                     double t_end, int64_t max_blocks, int64_t max_n_act,
                     double *t, double *dt, const double *m, double *x, double *v,
                     double *const a_derivs[8] /* HOST array of device pointers */, double *pot_state,
                     int32_t *active_idx, double *acc, double *jerk, double *snap, double *crackle, double *pot,
                     nbody_run_result *res /* HOST */, void *stream);

/* ------------------------------------------------------------------------------------------------------------
 * nbody_pack_rows / nbody_unpack_rows -- the exchange record of the i-sharded multi-GPU step (
 * PAPER.md:43 "Both use MPI", eq. (1) beta-term: one exchange per block).  rec[k] = { t, dt, pot_state,
 * x[3], v[3], a^(0)[3] .. a^(order-1)[3] } of particle idx[k]: 9 + 3 order doubles per row, device memory.
 * pack gathers the rows of idx[0..n_rows) into rec; unpack scatters rec back into the state arrays.  One kernel
 * each; between them sits the caller's all-gather (torch.distributed / NCCL).  Only enqueues.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_pack_rows(nbody_ctx *ctx, const int32_t *idx, int64_t n_rows, int order,
                    const double *t, const double *dt, const double *pot_state, const double *x, const double *v,
                    const double *const a_derivs[8] /* HOST array of device pointers */, double *rec, void *stream);
int nbody_unpack_rows(nbody_ctx *ctx, const int32_t *idx, int64_t n_rows, int order,
                      double *t, double *dt, double *pot_state, double *x, double *v,
                      double *const a_derivs[8] /* HOST array of device pointers */, const double *rec, void *stream);

/* Kernel launches issued through this ctx since creation (all kernels of this library). */
int64_t nbody_launch_count(const nbody_ctx *ctx);

/* Geometry of the last nbody_force call (for tests / bench): lanes, j-splits, CTAs of the force kernel. */
int nbody_last_force_geometry(const nbody_ctx *ctx, int *i_per_thread, int *j_lanes, int *j_splits, int64_t *ctas);

#ifdef __cplusplus
}
#endif
#endif /* NBODY_H_ */
