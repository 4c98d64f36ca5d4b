// Internal declarations shared by the translation units of libnbody.so (CUDA path only; nothing here is used
// by oracle/).  Public contract: include/nbody.h.  Design: DESIGN.md.
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
// feeds a j-value to both lanes of a packed f32x2 instruction as a broadcast 32-bit register operand.  Entries [n, n_pad) are zero-mass pads parked far away.
constexpr int kPlanes = 6;
#ifndef NB_TILEJ
#define NB_TILEJ 256
#endif
constexpr int kTileJ = NB_TILEJ;  // j-particles per TMA stage (and the padding granule of the j-store)
#ifndef NB_THREADS
#define NB_THREADS 512
#endif
constexpr int kThreads = NB_THREADS;  // threads per force CTA
constexpr double kPadPos = 1.0e6;

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
    // split partials: [S][NC][n_act] doubles
    double *partials = nullptr;
    size_t partials_bytes = 0;
    // next_block scratch
    unsigned long long *d_min_key = nullptr;  // 1
    int *d_counts = nullptr;                  // per selection block counts / offsets
    int64_t counts_cap = 0;
    long long *d_nact = nullptr;              // 1
    double *h_pinned = nullptr;               // small pinned return block (4 doubles)
    // host-buffer path staging (allocated on first use)
    void *stage = nullptr;
    size_t stage_bytes = 0;
    // options
    int diff_mode = 0;
    int force_split = 0;
    int force_lanes = 0;
    int crit_order = 0;  // 0 = automatic (4 for p >= 6, else p); 4 | 6 | 8 = criterion order min(p, value) (R8 / R8b)
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

// implemented in nbody_force.cu
int launch_force(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2,
                 double *acc, double *jerk, double *snap, double *crackle, double *pot, cudaStream_t st);
int probe_peak(Ctx *c, int kind, int millis, double *tera_ops);
int force_static_init(Ctx *c);

}  // namespace nbody
