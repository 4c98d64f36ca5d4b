// Internal declarations shared by the translation units of libnbody.so (CUDA path only; nothing here is used
// by oracle/).  Public contract: include/nbody.h, include/nbody_bench.h.  Design: DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "nbody.h"

namespace nbody {

// ---- packed j-store ---------------------------------------------------------------
// Planes of 16-byte quads, plane p at jstore + p * cap_pad (in quads):
//   Q0 = { x (f64), y (f64) }            Q1 = { z (f64), m (f32), vx (f32) }
//   Q2 = { vy, vz, ax, ay } (f32)        Q3 = { az, jx, jy, jz } (f32)
//   Q4 = { xhi, xlo, yhi, ylo } (f32)    Q5 = { zhi, zlo, m, vx } (f32)     (double-single twin of Q0/Q1)
// order 4 reads Q0..Q2, order 6 and 8 read Q0..Q3; diff_mode 1 reads Q4, Q5 instead of Q0, Q1.  The force kernel
// feeds a j-value to both lanes of a packed f32x2 instruction as a broadcast 32-bit register operand.
// Entries [n, n_pad) are zero-mass pads; the force kernel masks them by index (they never contribute).
constexpr int kPlanes = 6;
constexpr int kTileJ = 256;    // j-particles per TMA stage (and the padding granule of the j-store)
constexpr int kThreads = 512;  // threads per force CTA (one CTA per SM)
constexpr double kPadPos = 1.0e6;
constexpr int kNumLanes = 9;   // j-lane variants of the force kernel: a CTA is (kThreads / JL) i-lanes x JL j-lanes

__host__ __device__ inline int lane_variant(int k) {
    return 1 << k;  // 1, 2, 4, ..., 256 (256 = kTileJ: one j per thread and tile)
}

// ---- launch geometry of K_force (a-3), shared by the host launcher and the device-driven block step --------
// Integer arithmetic only, so host and device take the same decision bit for bit (the summation order of the
// force depends on JL and S, never on which CTA computes what).
struct ForceGeo {
    int jl;            // j-lanes per CTA
    int i_per_cta;     // 2 * kThreads / jl i-particles per CTA
    long long i_tiles; // ceil(n_act / i_per_cta)
    int splits;        // S: the j-range is cut into S contiguous runs of tiles
};

__host__ __device__ inline ForceGeo force_geometry(long long n_act, int n_tiles, int sm_count, int force_lanes,
                                                   int force_split, long long partial_rows_budget) {
    ForceGeo g;
    if (force_lanes) g.jl = force_lanes;
    else {  // the most j-lanes whose CTA still holds all active particles (2 * kThreads / JL i-slots)
        g.jl = 1;
        for (int k = kNumLanes - 1; k >= 1; --k)
            if ((long long)2 * kThreads / lane_variant(k) >= n_act) { g.jl = lane_variant(k); break; }
    }
    g.i_per_cta = 2 * (kThreads / g.jl);
    g.i_tiles = (n_act + g.i_per_cta - 1) / g.i_per_cta;
    // j-splits: the chip holds `slots` CTAs at once (one per SM); a launch of i_tiles * S work items takes
    // ceil(i_tiles * S / slots) waves of (ceil(n_tiles / S) + fixed per-item cost) tile-times.  Pick the S that
    // minimises it: small blocks get S ~ slots / i_tiles (fill the chip), mid-size blocks a work-item count close to a
    // multiple of `slots` (no half-empty last wave), big blocks (>= 8 waves) run unsplit.
    const long long slots = sm_count;
    long long S = 1;
    if (force_split) S = force_split;
    else if (g.i_tiles < 8 * slots) {
        const long long fixed = 3;  // prologue + epilogue + reduce, in tile-times
        long long best = -1, cost1 = 0;
        long long s_max = n_tiles < 4 * slots ? n_tiles : 4 * slots;
        if (n_act > 0 && s_max > partial_rows_budget / n_act) s_max = partial_rows_budget / n_act;
        for (long long s = 1; s <= s_max; ++s) {
            const long long waves = (g.i_tiles * s + slots - 1) / slots;
            const long long cost = waves * ((n_tiles + s - 1) / s + fixed);
            if (s == 1) cost1 = cost;
            if (best < 0 || cost < best) { best = cost; S = s; }
        }
        if (best < 0 || 100 * best > 97 * cost1) S = 1;  // a split costs S x NC x n_act doubles of scratch: only for a real gain
    }
    if (S > n_tiles) S = n_tiles;
    if (S > 65535) S = 65535;
    if (S < 1) S = 1;
    g.splits = (int)S;
    return g;
}

// ---- device control block of the device-driven block step (a-1 .. a-4 without host round trips) ---------------
struct Ctl {
    double t_next;                // block time of the current block
    double t_end;                 // blocks with t_next > t_end are not executed (stop is set instead)
    long long n_act;              // size of the current block
    long long max_blocks;         // run budget (blocks executed since the run started)
    unsigned long long blocks;    // blocks executed in this run
    unsigned long long pairs;     // Sum n_act * n over the executed blocks
    int stop;                     // 1 = t_next > t_end or budget reached: every kernel of the step is a no-op
    int error;                    // validation failure code (device-side checks)
    int jl, splits;               // force geometry of the current block (force_geometry(), evaluated on the device)
    long long i_tiles;
    unsigned long long rejected;  // steps refused by the a-posteriori rule (R14) since the counter was last reset
    unsigned long long limited;   // steps taken with a lower-order corrector (R15) since the counter was last reset
    unsigned int tickets[4];      // last-CTA tickets ([0] fused step, [1] selection)
    unsigned long long hist[40];  // executed blocks by floor(log2 n_act)
};

struct Ctx {
    int device = 0;
    int sm_count = 0;
    int64_t cap = 0;      // particles
    int64_t cap_pad = 0;  // rounded up to kTileJ
    uint4 *jstore = nullptr;
    // state of the last predict
    int64_t n = -1;
    int64_t n_pad = 0;
    int pred_order = 0;
    bool ds_valid = false;
    // split partials: [S][NC][n_act] doubles, sized once in nbody_create (nbody_force never allocates)
    double *partials = nullptr;
    size_t partials_bytes = 0;
    int64_t partial_rows = 0;  // S * n_act budget (rows of 13 doubles)
    // selection scratch
    int *d_counts = nullptr;  // per selection CTA: particles due at the CTA's own minimum
    unsigned long long *d_keys = nullptr;  // per selection CTA: that minimum (order-preserving key)
    int32_t *d_cand = nullptr;  // [cap] their indices (CTA b's slice starts at b * chunk)
    Ctl *d_ctl = nullptr;     // device control block
    Ctl *h_ctl = nullptr;     // pinned host copy (read back after a synchronisation)
    int *d_flag = nullptr;    // validation result
    // host-buffer path staging (allocated on first use)
    void *stage = nullptr;
    size_t stage_bytes = 0;
    // block-step graph cache (nbody_run_blocks)
    cudaGraphExec_t graph_exec = nullptr;        // general step: select, predict, force, reduce, correct
    cudaGraphExec_t graph_small = nullptr;       // fused small-block step (N1): select, fused step
    unsigned long long graph_key[24] = {0};
    // options
    int diff_mode = 0;
    int force_split = 0;
    int force_lanes = 0;
    int64_t geometry_n_act = 0;  // 0 = the call's n_act decides JL and S; else this value does (i-sharded ranks)
    int crit_order = 0;  // 0 = automatic (4 for p >= 6, else p); 4 | 6 | 8 = criterion order min(p, value) (R8 / R8b)
    int validate = 0;
    int use_graph = 1;
    int use_fused = 0;     // N1: 1 = runs of blocks that fit one i-tile go through the fused step (measured no faster yet)
    int limit_order = 0;   // R15: 1 = corrector order limiter
    int reject_ratio = 0;  // R14: 0 = off; R = 2^r >= 2: a step whose end-point criterion asks for dt <= h/R is refused
    // bookkeeping
    int last_cuda_error = 0;
    int64_t launches = 0;
    int last_r = 0, last_jl = 0, last_s = 0;
    int64_t last_ctas = 0;
};

inline int cuda_fail(Ctx *c, cudaError_t e) {
    if (c) c->last_cuda_error = (int)e;
    return e == cudaErrorMemoryAllocation ? NBODY_ENOMEM : NBODY_ECUDA;
}

#define NB_CUDA(ctx, expr)                                        \
    do {                                                          \
        cudaError_t e__ = (expr);                                 \
        if (e__ != cudaSuccess) return ::nbody::cuda_fail(ctx, e__); \
    } while (0)

// Binds the calling thread to the ctx's device for the duration of a call and restores the caller's device.
struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    explicit DeviceGuard(int device) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) changed = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (changed) cudaSetDevice(prev);
    }
};

}  // namespace nbody

// the opaque handle of include/nbody.h
struct nbody_ctx {
    nbody::Ctx c;
    cudaStream_t run_stream = nullptr;  // private stream of nbody_run_blocks (graph capture)
    cudaEvent_t ev_in = nullptr, ev_out = nullptr;
};

namespace nbody {

// implemented in nbody_force.cu
int launch_force(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2,
                 double *acc, double *jerk, double *snap, double *crackle, double *pot, cudaStream_t st);
// device-driven variant: n_act and the geometry are read from the control block on the device
int launch_force_dyn(Ctx *c, const int32_t *active_idx, int order, float eps2, double *acc, double *jerk, double *snap,
                     double *crackle, double *pot, cudaStream_t st);
// allocation-free variant: split partials in the library's static device array (nbody_force_static)
int launch_force_static(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2, double *acc, double *jerk,
                        double *snap, double *crackle, double *pot, cudaStream_t st);
int force_static_init(Ctx *c);
// device-driven step: K_reduce with S and n_act from the control block
int launch_reduce_dyn(Ctx *c, int order, double *acc, double *jerk, double *snap, double *crackle, double *pot,
                      cudaStream_t st);
struct CorrArgs;
// N1: predict + force + reduce + correct of a block that fits one i-tile, in one launch (reads the control block)
int launch_step_fused(Ctx *c, int order, float eps2, const int32_t *active_idx, const double *t, const double *m,
                      const double *x, const double *v, const double *const a_derivs[8], const CorrArgs &corr,
                      double *acc, double *jerk, double *snap, double *crackle, double *pot, cudaStream_t st);
// implemented in nbody_probe.cu
int probe_peak(Ctx *c, int kind, int millis, double *tera_ops);

}  // namespace nbody
