// libnbody.so, translation unit 1: context management and the fp64 bit-exact kernels
//   K_pred (a-2), K_corr (a-4), initial dt, block selection (a-1), j-store export, row pack/unpack for the multi-GPU
//   exchange, argument validation, the device-driven block step (nbody_run_blocks) and the host-buffer path.
// Compiled with -fmad=false; in addition every fp64 operation whose rounding matters is written with the
// __d*_rn intrinsics, which are never contracted, so the results equal a plain IEEE evaluation in the
// stated order (R12).  The formulas restate DESIGN.md section 3 (R5..R9); the paper
// itself names the scheme only.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "nbody_exact.cuh"
#include "nbody_internal.h"

using namespace nbody;

namespace {

struct PredArgs {
    const double *t, *m, *x, *v;
    const double *D[6];
    uint4 *q[kPlanes];
    double t_now;
    long long n, n_pad;
    int write_ds;
    const Ctl *ctl;  // device-driven step: t_now = ctl->t_next, no-op when the run has stopped (else NULL)
};

// K_pred: one thread per j-store slot (particles, then pads).  R5: Horner, innermost first, c_k = tau / k.
template <int ORDER>
__global__ void __launch_bounds__(256) k_predict(PredArgs A) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.n_pad) return;
    double t_now = A.t_now;
    if (A.ctl) {
        if (A.ctl->stop) return;
        t_now = A.ctl->t_next;
    }
    double xp[3];
    float vp[3], ap[3] = {0.f, 0.f, 0.f}, jp[3] = {0.f, 0.f, 0.f}, m32 = 0.f;
    if (i < A.n) {
        const double *Dp[6];
#pragma unroll
        for (int k = 0; k < ORDER - 2; ++k) Dp[k] = A.D[k] + 3 * i;
        predict_particle<ORDER>(d_sub(t_now, A.t[i]), A.x + 3 * i, A.v + 3 * i, Dp, xp, vp, ap, jp);
        m32 = __double2float_rn(A.m[i]);
    } else {
        xp[0] = xp[1] = xp[2] = kPadPos;
        vp[0] = vp[1] = vp[2] = 0.f;
    }
    A.q[0][i] = pack_dd(xp[0], xp[1]);
    A.q[1][i] = pack_dff(xp[2], m32, vp[0]);
    A.q[2][i] = pack_ffff(vp[1], vp[2], ap[0], ap[1]);
    if (ORDER >= 6) A.q[3][i] = pack_ffff(ap[2], jp[0], jp[1], jp[2]);
    if (A.write_ds) {
        float hi[3], lo[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            hi[d] = __double2float_rn(xp[d]);
            lo[d] = __double2float_rn(d_sub(xp[d], (double)hi[d]));
        }
        A.q[4][i] = pack_ffff(hi[0], lo[0], hi[1], lo[1]);
        A.q[5][i] = pack_ffff(hi[2], lo[2], m32, vp[0]);
    }
}

// export of the j-store (test hook)
__global__ void k_unpack(const uint4 *q0, const uint4 *q1, const uint4 *q2, const uint4 *q3, long long n, int order,
                         double *xp, float *vp, float *ap, float *jp, float *m32) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 a = q0[i], b = q1[i], c = q2[i];
    xp[3 * i + 0] = __longlong_as_double(((long long)a.y << 32) | a.x);
    xp[3 * i + 1] = __longlong_as_double(((long long)a.w << 32) | a.z);
    xp[3 * i + 2] = __longlong_as_double(((long long)b.y << 32) | b.x);
    m32[i] = __uint_as_float(b.z);
    vp[3 * i + 0] = __uint_as_float(b.w);
    vp[3 * i + 1] = __uint_as_float(c.x);
    vp[3 * i + 2] = __uint_as_float(c.y);
    if (order >= 6) {
        const uint4 d = q3[i];
        if (ap) {
            ap[3 * i + 0] = __uint_as_float(c.z);
            ap[3 * i + 1] = __uint_as_float(c.w);
            ap[3 * i + 2] = __uint_as_float(d.x);
        }
        if (jp && order >= 8) {
            jp[3 * i + 0] = __uint_as_float(d.y);
            jp[3 * i + 1] = __uint_as_float(d.z);
            jp[3 * i + 2] = __uint_as_float(d.w);
        }
    }
}

// ---- nearest-neighbour output (reading R16 = oracle c-17) -----------------------------------------
// For each active i the nearest other particle of the j-store: d = fl32(x_j - x_i) formed in fp64 (the force kernel's
// differences), r2 = fma(dz, dz, fma(dy, dy, dx * dx)) in fp32, ties to the lowest index.  One thread per active
// particle, j-tiles of kNnTile staged in shared memory, S j-splits; the splits meet in an atomicMin on the 64-bit key
// (bits of r2) << 32 | j -- r2 >= 0, so the order of the keys is the order of (r2, j) and the result does not depend
// on S or on the order in which the splits arrive.
constexpr int kNnTile = 256;

__global__ void __launch_bounds__(kNnTile) k_nearest(const uint4 *q0, const uint4 *q1, long long n,
                                                      const int32_t *active_idx, int n_act, int n_tiles, int splits,
                                                      unsigned long long *keys) {
    __shared__ uint4 s0[kNnTile], s1[kNnTile];
    const int tid = threadIdx.x;
    const int ia = blockIdx.x * kNnTile + tid;
    const bool live = ia < n_act;
    const int i = live ? active_idx[ia] : 0;
    double xi = 0.0, yi = 0.0, zi = 0.0;
    if (live) {
        const uint4 a = q0[i], b = q1[i];
        xi = __longlong_as_double(((long long)a.y << 32) | a.x);
        yi = __longlong_as_double(((long long)a.w << 32) | a.z);
        zi = __longlong_as_double(((long long)b.y << 32) | b.x);
    }
    const int per = (n_tiles + splits - 1) / splits;
    const int tile_lo = blockIdx.y * per, tile_hi = tile_lo + per < n_tiles ? tile_lo + per : n_tiles;
    unsigned long long best = ~0ull;
    for (int tile = tile_lo; tile < tile_hi; ++tile) {
        const long long j0 = (long long)tile * kNnTile;
        __syncthreads();
        if (j0 + tid < n) {
            s0[tid] = q0[j0 + tid];
            s1[tid] = q1[j0 + tid];
        }
        __syncthreads();
        const int cnt = n - j0 < kNnTile ? (int)(n - j0) : kNnTile;
#pragma unroll 4
        for (int jj = 0; jj < cnt; ++jj) {
            const uint4 a = s0[jj], b = s1[jj];
            const float dx = __double2float_rn(__dsub_rn(__longlong_as_double(((long long)a.y << 32) | a.x), xi));
            const float dy = __double2float_rn(__dsub_rn(__longlong_as_double(((long long)a.w << 32) | a.z), yi));
            const float dz = __double2float_rn(__dsub_rn(__longlong_as_double(((long long)b.y << 32) | b.x), zi));
            const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const unsigned long long key = ((unsigned long long)__float_as_uint(r2) << 32) | (unsigned)(j0 + jj);
            if (j0 + jj != i && r2 == r2 && key < best) best = key;  // ascending j: a tie keeps the earlier one
        }
    }
    if (live && best != ~0ull) atomicMin(keys + ia, best);
}

__global__ void k_nearest_out(const unsigned long long *keys, int n_act, int32_t *nn_idx, double *nn_r2) {
    const int ia = blockIdx.x * blockDim.x + threadIdx.x;
    if (ia >= n_act) return;
    const unsigned long long k = keys[ia];
    if (k == ~0ull) {  // no other particle
        nn_idx[ia] = -1;
        nn_r2[ia] = __longlong_as_double(0x7ff0000000000000ll);
    } else {
        nn_idx[ia] = (int32_t)(k & 0xffffffffull);
        nn_r2[ia] = (double)__uint_as_float((unsigned)(k >> 32));
    }
}

}  // namespace

// K_pred's particle arithmetic and the whole of K_corr (k_correct, correct_one) live in nbody_exact.cuh.
namespace {

// R9b start-up step
__global__ void k_initial_dt(long long n, const double *acc, const double *jerk, double eta_s, int k_min, int k_max,
                             double dt_min, double dt_max, double *dt) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double a[3] = {acc[3 * i], acc[3 * i + 1], acc[3 * i + 2]};
    double j[3] = {jerk[3 * i], jerk[3 * i + 1], jerk[3 * i + 2]};
    const double na = nrm3(a), nj = nrm3(j);
    const int k = floor_log2_ratio(na, nj, eta_s, 1, k_min - 1, k_max + 1);
    double d = pow2i(k);
    if (d > dt_max) d = dt_max;
    if (d < dt_min) d = dt_min;
    dt[i] = d;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
// Block selection (a-1, R9c) in ONE kernel, one pass, no grid barrier.  Every CTA owns a contiguous chunk of the
// particles: it takes the chunk's own minimum of t + dt and writes the indices of the chunk's particles due at THAT
// time, in order, to its slice of a candidate array.  The last CTA to finish (ticket) takes the minimum over the
// CTAs, concatenates the candidate lists of the CTAs whose minimum it is -- in CTA order, so the active list is
// ascending -- and leaves the block time, the block size, the force geometry (force_geometry(), evaluated by 1024
// threads in parallel) and the run bookkeeping in the device control block, so that the rest of the block step can be
// launched without the host knowing n_act (nbody_run_blocks).  The concatenation is a copy of at most n_act indices by
// one CTA (n_act * 8 bytes against n_act * n pair interactions of the force call that follows); every CTA also writes
// its list to the same place of the active list, which is its final place in an all-active block: no copy then.
// Entries of the active list at and beyond n_act are scratch.
// ---------------------------------------------------------------------------------------------------------
namespace {

constexpr int kSelThreads = 1024;
constexpr int kSelMaxGrid = 1024;  // CTAs of the selection kernel (<= the SM count; bounds the tail's shared arrays)

// order-preserving map double -> uint64 (total order of finite values)
__device__ __forceinline__ unsigned long long dkey(double v) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dunkey(unsigned long long k) {
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

struct SelArgs {
    long long n;
    const double *t, *dt;
    Ctl *ctl;
    unsigned long long *keys;  // [grid] minimum of each CTA's chunk
    int *counts;               // [grid] particles of the chunk due at the CTA's own minimum
    int32_t *cand;             // [n]    their indices, CTA b's at cand[chunk start of b ...]
    int32_t *active_idx;       // [n]
    // force geometry inputs (force_geometry)
    int n_tiles, sm_count, force_lanes, force_split;
    long long rows_budget;
    // run control
    int run_mode;         // 0 = plain selection (never stops); 1 = run: honour t_end / max_blocks / max_n_act;
                          // 2 = as 1, and stop (4) in front of a block that does not fit one i-tile (fused run, N1)
    long long max_n_act;  // run: a block larger than this stops the run (stop = 2) for the host to handle
};

// minimum over the CTA of a 64-bit key (every thread gets it); s_red: one slot per warp
__device__ __forceinline__ unsigned long long cta_min_key(unsigned long long k, unsigned long long *s_red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other < k ? other : k;
    }
    if (lane == 0) s_red[warp] = k;
    __syncthreads();
    k = s_red[lane];  // kSelThreads / 32 == 32 slots
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other < k ? other : k;
    }
    __syncthreads();  // s_red may be reused
    return k;
}

constexpr int kSelRows = 16;  // rows of kSelThreads consecutive particles compacted per pass (bounds the shared counts)

__global__ void __launch_bounds__(kSelThreads, 1) k_select(const SelArgs A) {
    extern __shared__ unsigned long long s_keys[];  // [min(rows of the chunk, kSelRows)][kSelThreads]
    __shared__ unsigned long long s_red[kSelThreads / 32];
    __shared__ int s_cntw[kSelRows * 32];  // due particles per (row, warp), then their exclusive offsets
    __shared__ int s_cnt[kSelMaxGrid];
    __shared__ long long s_off[kSelMaxGrid];
    __shared__ long long s_all;
    __shared__ int s_tot;
    __shared__ bool s_last;
    const unsigned grid = gridDim.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    Ctl *ctl = A.ctl;
    // a stopped run stays stopped (nothing after the stopping selection touches the state): replays are no-ops
    if (A.run_mode && *(volatile int *)&ctl->stop) return;
    // run control read early (whichever CTA turns out to be the last one needs it; nobody writes it meanwhile)
    double t_end = 0.0;
    long long max_blocks = 0;
    unsigned long long blocks = 0;
    if (A.run_mode && tid == 0) {
        t_end = ctl->t_end;
        max_blocks = ctl->max_blocks;
        blocks = ctl->blocks;
    }
    const long long chunk = (A.n + grid - 1) / grid;
    const long long c0 = (long long)blockIdx.x * chunk;
    const long long c1 = c0 + chunk < A.n ? c0 + chunk : A.n;
    const long long per = (chunk + kSelThreads - 1) / kSelThreads;  // rows of this CTA's chunk

    // ---- the chunk's minimum of t + dt (exact for dyadic values); row r holds particles c0 + r * 1024 + tid ----
    unsigned long long k = ~0ull;
#pragma unroll 4
    for (long long r = 0; r < per; ++r) {
        const long long i = c0 + r * kSelThreads + tid;
        if (i < c1) {
            const unsigned long long ki = dkey(__dadd_rn(A.t[i], A.dt[i]));
            k = ki < k ? ki : k;
            if (r < kSelRows) s_keys[r * kSelThreads + tid] = ki;  // the first kSelRows rows stay in shared memory
        }
    }
    const unsigned long long key_cta = cta_min_key(k, s_red);

    // ---- the chunk's particles due at it, in index order, to the CTA's slice of the candidate array: per row one
    // ballot per warp, the (row, warp) counts scanned in shared memory, kSelRows rows at a time (the keys of the first
    // kSelRows rows come from shared memory, those of later rows -- N > 2.4 M -- are recomputed from t and dt) ----
    int base = 0;
    for (long long r0 = 0; r0 < per; r0 += kSelRows) {
        const int rows = per - r0 < kSelRows ? (int)(per - r0) : kSelRows;
#pragma unroll 1
        for (int r = 0; r < rows; ++r) {
            const long long i = c0 + (r0 + r) * kSelThreads + tid;
            const bool due = i < c1 && (r0 == 0 ? s_keys[r * kSelThreads + tid] : dkey(__dadd_rn(A.t[i], A.dt[i]))) == key_cta;
            const unsigned m = __ballot_sync(0xffffffffu, due);
            if (lane == 0) s_cntw[r * 32 + warp] = __popc(m);
        }
        __syncthreads();
        if (warp == 0) {  // exclusive scan of the rows * 32 counts: lane l owns entries [l * rows, (l + 1) * rows)
            int sum = 0;
            for (int e = 0; e < rows; ++e) sum += s_cntw[lane * rows + e];
            int incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += up;
            }
            int run = incl - sum;
            for (int e = 0; e < rows; ++e) {
                const int v = s_cntw[lane * rows + e];
                s_cntw[lane * rows + e] = run;
                run += v;
            }
            if (lane == 31) s_tot = incl;
        }
        __syncthreads();
        if (s_tot) {  // uniform
#pragma unroll 1
            for (int r = 0; r < rows; ++r) {
                const long long i = c0 + (r0 + r) * kSelThreads + tid;
                const bool due = i < c1 && (r0 == 0 ? s_keys[r * kSelThreads + tid] : dkey(__dadd_rn(A.t[i], A.dt[i]))) == key_cta;
                const unsigned m = __ballot_sync(0xffffffffu, due);
                if (due) {  // also to the same place of the active list: a CTA whose final offset is its chunk start is done
                    const long long q = c0 + base + s_cntw[r * 32 + warp] + __popc(m & ((1u << lane) - 1u));
                    A.cand[q] = (int32_t)i;
                    A.active_idx[q] = (int32_t)i;
                }
            }
        }
        base += s_tot;
        __syncthreads();
    }
    if (tid == 0) {
        A.counts[blockIdx.x] = base;
        A.keys[blockIdx.x] = key_cta;
    }

    // ---- ticket: the last CTA to get here finishes the selection ----
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned ticket = atomicAdd(&ctl->tickets[1], 1u);
        s_last = ticket == grid - 1;
        if (s_last) ctl->tickets[1] = 0;  // ready for the next selection (stream-ordered after this one)
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();

    // global minimum, and the size of the block = the counts of the CTAs whose minimum it is
    unsigned long long kb = ~0ull;
    int cb = 0;
    if (tid < (int)grid) {
        kb = __ldcg(A.keys + tid);
        cb = __ldcg(A.counts + tid);
    }
    const unsigned long long key = cta_min_key(kb, s_red);
    if (tid < (int)grid) s_cnt[tid] = kb == key ? cb : 0;
    __syncthreads();
    if (warp == 0) {  // exclusive scan of s_cnt over the CTAs, 32 at a time
        long long running = 0;
        for (unsigned b0 = 0; b0 < grid; b0 += 32) {
            const int v = b0 + lane < grid ? s_cnt[b0 + lane] : 0;
            long long in = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const long long up = __shfl_up_sync(0xffffffffu, in, o);
                if (lane >= o) in += up;
            }
            if (b0 + lane < grid) s_off[b0 + lane] = running + in - v;
            running += __shfl_sync(0xffffffffu, in, 31);
        }
        if (lane == 0) s_all = running;
    }
    __syncthreads();
    // ordered concatenation: warp w copies the candidate lists of CTAs w, w + 32, ... (a list that already sits at its
    // final offset -- every list of an all-active block -- is left alone)
    for (unsigned b = warp; b < grid; b += kSelThreads / 32) {
        const int nb = s_off[b] == (long long)b * chunk ? 0 : s_cnt[b];
        const int32_t *src = A.cand + (long long)b * chunk;
        int32_t *dst = A.active_idx + s_off[b];
        for (int e = lane; e < nb; e += 32) dst[e] = __ldcg(src + e);
    }

    // block time, size, run control, force geometry (the parallel form of force_geometry()'s search)
    const long long n_act = s_all;
    const double t_next = dunkey(key);
    ForceGeo g = force_geometry(n_act, A.n_tiles, A.sm_count, A.force_lanes, /*force_split=*/1, A.rows_budget);
    const long long slots = A.sm_count;
    long long S = 1;
    if (A.force_split) S = A.force_split;
    else if (g.i_tiles < 8 * slots) {
        long long s_max = A.n_tiles < 4 * slots ? A.n_tiles : 4 * slots;
        if (n_act > 0 && s_max > A.rows_budget / n_act) s_max = A.rows_budget / n_act;
        unsigned long long mine = ~0ull;  // (cost << 20) | s : the minimum is the cheapest s, smallest s on ties
        // 32-bit arithmetic is exact here: i_tiles < 8 * slots and sc <= 4 * slots, n_tiles < 2^23
        const unsigned it32 = (unsigned)g.i_tiles, sl32 = (unsigned)slots, nt32 = (unsigned)A.n_tiles;
        for (unsigned sc = 1 + tid; sc <= (unsigned)s_max; sc += kSelThreads) {
            const unsigned waves = (it32 * sc + sl32 - 1) / sl32;
            const unsigned long long cost = (unsigned long long)waves * ((nt32 + sc - 1) / sc + 3);
            const unsigned long long kk = (cost << 20) | (unsigned long long)sc;
            mine = kk < mine ? kk : mine;
        }
        mine = cta_min_key(mine, s_red);
        if (mine != ~0ull) {
            const long long best = (long long)(mine >> 20);
            const long long cost1 = ((g.i_tiles + slots - 1) / slots) * ((long long)A.n_tiles + 3);
            S = (long long)(mine & 0xfffffull);
            if (100 * best > 97 * cost1) S = 1;
        }
    }
    if (tid == 0) {
        int stop = 0;
        if (A.run_mode) {
            if (t_next > t_end) stop = 1;
            else if (n_act > A.max_n_act) stop = 2;
            else if ((long long)blocks >= max_blocks) stop = 3;
            else if (A.run_mode == 2 && g.i_tiles != 1) stop = 4;  // fused small-block run: this block needs the general step
        }
        if (S > A.n_tiles) S = A.n_tiles;
        if (S > 65535) S = 65535;
        if (S < 1) S = 1;
        ctl->t_next = t_next;
        ctl->n_act = n_act;
        ctl->jl = g.jl;
        ctl->splits = (int)S;
        ctl->i_tiles = g.i_tiles;
        ctl->stop = stop;
        if (A.run_mode && !stop) {
            ctl->blocks = blocks + 1;
            atomicAdd(&ctl->pairs, (unsigned long long)n_act * (unsigned long long)A.n);
            int b = 0;
            while ((n_act >> (b + 1)) != 0) ++b;
            atomicAdd(&ctl->hist[b < 39 ? b : 39], 1ull);
        }
    }
}

bool is_pow2(double x, int *e) {
    if (!(x > 0.0) || isinf(x)) return false;
    int ex;
    const double f = frexp(x, &ex);
    *e = ex - 1;
    return f == 0.5;
}

// ---- argument validation on the device ("validate" option): index range, strict ascent, due times -------------
__global__ void k_validate(const int32_t *idx, long long n_act, long long n, const double *t, const double *dt,
                           double t_now, int *flag) {
    for (long long ia = (long long)blockIdx.x * blockDim.x + threadIdx.x; ia < n_act;
         ia += (long long)gridDim.x * blockDim.x) {
        const long long i = idx[ia];
        int bad = 0;
        if (i < 0 || i >= n) bad = 1;
        else if (ia > 0 && idx[ia - 1] >= i) bad = 2;
        else if (t && __dadd_rn(t[i], dt[i]) != t_now) bad = 3;
        if (bad) atomicMax(flag, bad);
    }
}

// ---- packed particle records for the multi-GPU exchange: rec[k] = { t, dt, pot, x[3], v[3], D_0[3] .. }
struct RowArgs {
    const int32_t *idx;
    long long n_rows;
    int order;
    double *t, *dt, *pot, *x, *v, *D[8];
    double *rec;
};

template <bool PACK>
__global__ void __launch_bounds__(256) k_rows(const RowArgs A) {
    const int ncol = 9 + 3 * A.order;
    const long long tot = A.n_rows * ncol;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < tot; o += (long long)gridDim.x * blockDim.x) {
        const long long k = o / ncol;
        const int c = (int)(o % ncol);
        const long long i = A.idx[k];
        double *p;
        if (c == 0) p = A.t + i;
        else if (c == 1) p = A.dt + i;
        else if (c == 2) p = A.pot + i;
        else if (c < 6) p = A.x + 3 * i + (c - 3);
        else if (c < 9) p = A.v + 3 * i + (c - 6);
        else p = A.D[(c - 9) / 3] + 3 * i + (c - 9) % 3;
        if (PACK) A.rec[o] = *p;
        else *p = A.rec[o];
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------------------
namespace {

inline bool misaligned(const void *p, size_t a) { return p && ((uintptr_t)p & (a - 1)) != 0; }

// Every fp64 array must be 8-byte aligned, every int32 array 4-byte aligned.
#define NB_ALIGN8(...)                                          \
    do {                                                        \
        const void *ps__[] = {__VA_ARGS__};                     \
        for (const void *p__ : ps__)                            \
            if (misaligned(p__, 8)) return NBODY_EINVAL;        \
    } while (0)

size_t select_smem(const Ctx *c, int64_t n);

int select_grid(const Ctx *c, int64_t n) {
    int64_t g = (n + kSelThreads - 1) / kSelThreads;
    if (g > c->sm_count) g = c->sm_count;
    if (g > kSelMaxGrid) g = kSelMaxGrid;
    return (int)(g < 1 ? 1 : g);
}

size_t select_smem(const Ctx *c, int64_t n) {  // the key cache of k_select: rows of the chunk, at most kSelRows
    const int64_t grid = select_grid(c, n);
    const int64_t chunk = (n + grid - 1) / grid;
    int64_t rows = (chunk + kSelThreads - 1) / kSelThreads;
    if (rows > kSelRows) rows = kSelRows;
    return (size_t)rows * kSelThreads * sizeof(unsigned long long);
}

void fill_select(nbody_ctx *h, SelArgs &A, int64_t n, const double *t, const double *dt, int32_t *active_idx,
                 int run_mode, int64_t max_n_act) {
    Ctx *c = &h->c;
    A.n = n; A.t = t; A.dt = dt; A.ctl = c->d_ctl; A.keys = c->d_keys; A.counts = c->d_counts; A.cand = c->d_cand; A.active_idx = active_idx;
    A.n_tiles = (int)((n + kTileJ - 1) / kTileJ);
    A.sm_count = c->sm_count; A.force_lanes = c->force_lanes; A.force_split = c->force_split;
    A.rows_budget = c->partial_rows;
    A.run_mode = run_mode; A.max_n_act = max_n_act;
}

int launch_predict(Ctx *c, int64_t n, double t_now, int order, const double *t, const double *m, const double *x,
                   const double *v, const double *const a_derivs[6], const Ctl *ctl, cudaStream_t st) {
    PredArgs A;
    A.t = t; A.m = m; A.x = x; A.v = v;
    for (int k = 0; k < 6; ++k) A.D[k] = k <= order - 3 ? a_derivs[k] : nullptr;
    for (int p = 0; p < kPlanes; ++p) A.q[p] = c->jstore + (size_t)p * c->cap_pad;
    A.t_now = t_now;
    A.n = n;
    A.n_pad = c->n_pad;
    A.write_ds = c->ds_valid ? 1 : 0;
    A.ctl = ctl;
    const unsigned grid = (unsigned)((c->n_pad + 255) / 256);
    if (order == 4) k_predict<4><<<grid, 256, 0, st>>>(A);
    else if (order == 6) k_predict<6><<<grid, 256, 0, st>>>(A);
    else k_predict<8><<<grid, 256, 0, st>>>(A);
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

// criterion order in use (R8 / R8b) and the exponent range check of R9 (pow2i is exact for |e| <= 1022)
int criterion_order(const Ctx *c, int order) {
    return c->crit_order ? (c->crit_order < order ? c->crit_order : order) : (order >= 6 ? 4 : order);
}
bool dt_range_ok(int kmin, int kmax, int q) {
    const long long a = kmin < 0 ? -(long long)kmin : kmin, b = kmax < 0 ? -(long long)kmax : kmax;
    return ((a > b ? a : b) + 1) * q <= 1022;
}

int launch_correct(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, double t_now, double eta,
                   double dt_min, double dt_max, int kmin, int kmax, double *t, double *dt, double *x, double *v,
                   double *const a_derivs[8], double *pot_state, const double *acc, const double *jerk,
                   const double *snap, const double *crackle, const double *pot, const Ctl *ctl, cudaStream_t st) {
    CorrArgs A;
    A.idx = active_idx; A.n_act = n_act; A.t_now = t_now; A.eta = eta; A.dt_min = dt_min; A.dt_max = dt_max;
    A.k_min = kmin; A.k_max = kmax;
    A.crit_order = criterion_order(c, order);
    A.t = t; A.dt = dt; A.x = x; A.v = v; A.pot_state = pot_state;
    for (int k = 0; k < 8; ++k) A.D[k] = k < order ? a_derivs[k] : nullptr;
    A.acc = acc; A.jerk = jerk; A.snap = snap; A.crk = crackle; A.pot = pot;
    A.ctl = ctl;
    A.reject_ratio = c->reject_ratio;
    A.n_rejected = &c->d_ctl->rejected;
    A.limit_order = c->limit_order;
    A.n_limited = &c->d_ctl->limited;
    long long blocks = ctl ? 2LL * c->sm_count : (n_act + 127) / 128;
    if (blocks > 16LL * c->sm_count) blocks = 16LL * c->sm_count;
    if (order == 4) k_correct<4><<<(unsigned)blocks, 128, 0, st>>>(A);
    else if (order == 6) k_correct<6><<<(unsigned)blocks, 128, 0, st>>>(A);
    else k_correct<8><<<(unsigned)blocks, 128, 0, st>>>(A);
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

// "validate" option: device-side check of an active list (and of the due times when t != NULL); synchronises.
int validate_active(Ctx *c, const int32_t *idx, int64_t n_act, int64_t n, const double *t, const double *dt,
                    double t_now, cudaStream_t st) {
    NB_CUDA(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int), st));
    long long blocks = (n_act + 255) / 256;
    if (blocks > 8LL * c->sm_count) blocks = 8LL * c->sm_count;
    k_validate<<<(unsigned)blocks, 256, 0, st>>>(idx, n_act, n, t, dt, t_now, c->d_flag);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    int flag = 0;
    NB_CUDA(c, cudaMemcpyAsync(&flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    return flag ? NBODY_EINVAL : NBODY_OK;
}

}  // namespace

extern "C" {

int nbody_abi_version(void) { return 2; }

const char *nbody_strerror(int code) {
    switch (code) {
        case NBODY_OK: return "ok";
        case NBODY_EINVAL: return "invalid argument";
        case NBODY_ESTATE: return "invalid call order (predict first; force order <= predict order)";
        case NBODY_ECUDA: return "CUDA runtime error (see nbody_last_cuda_error)";
        case NBODY_ENOMEM: return "out of memory";
        case NBODY_ESCRATCH: return "nbody_force_static: S * NC * n_act * 8 bytes exceeds NBODY_FORCE_STATIC_SCRATCH_BYTES";
        default: return "unknown nbody error code";
    }
}

int64_t nbody_workspace_bytes(int64_t n_capacity) {
    if (n_capacity < 1 || n_capacity > (int64_t)1 << 30) return -1;
    const int64_t cap_pad = (n_capacity + kTileJ - 1) / kTileJ * kTileJ;
    // the split scratch depends on the SM count (known at create); this is the bound for a 148-SM part
    int64_t rows = 4LL * 148 * 2 * kThreads > 4 * n_capacity ? 4LL * 148 * 2 * kThreads : 4 * n_capacity;
    if (rows * 13 * 8 > (int64_t)512 << 20) rows = ((int64_t)512 << 20) / (13 * 8);
    const int64_t n_tiles = cap_pad / kTileJ;
    if (rows > n_tiles * n_capacity) rows = n_tiles * n_capacity;
    return (int64_t)sizeof(uint4) * kPlanes * cap_pad + rows * 13 * 8 + 4 * n_capacity /* selection candidates */ + 8192;
}

int nbody_create(nbody_ctx **out, int64_t n_capacity, int device) {
    if (!out || n_capacity < 1 || n_capacity > (int64_t)1 << 30) return NBODY_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return NBODY_ECUDA;
    }
    nbody_ctx *h = new (std::nothrow) nbody_ctx();
    if (!h) return NBODY_ENOMEM;
    Ctx *c = &h->c;
    c->device = device;
    DeviceGuard guard(device);
    int rc = NBODY_OK;
    do {
        cudaError_t e;
        cudaDeviceProp prop;
        if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        c->sm_count = prop.multiProcessorCount;
        c->cap = n_capacity;
        c->cap_pad = (n_capacity + kTileJ - 1) / kTileJ * kTileJ;
        if ((e = cudaMalloc(&c->jstore, sizeof(uint4) * kPlanes * c->cap_pad)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        // split scratch, sized ONCE: rows of 13 doubles, S * n_act <= partial_rows for every geometry force_geometry() picks
        int64_t rows = 4LL * c->sm_count * 2 * kThreads > 4 * n_capacity ? 4LL * c->sm_count * 2 * kThreads : 4 * n_capacity;
        if (rows * 13 * 8 > (int64_t)512 << 20) rows = ((int64_t)512 << 20) / (13 * 8);
        const int64_t n_tiles = c->cap_pad / kTileJ;
        if (rows > n_tiles * n_capacity) rows = n_tiles * n_capacity;  // S <= n_tiles, n_act <= capacity
        c->partial_rows = rows;
        c->partials_bytes = (size_t)rows * 13 * sizeof(double);
        if ((e = cudaMalloc(&c->partials, c->partials_bytes)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_counts, sizeof(int) * (c->sm_count + 1))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_ctl, sizeof(Ctl))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_keys, sizeof(unsigned long long) * (c->sm_count + 1))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_cand, sizeof(int32_t) * n_capacity)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_flag, sizeof(int))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMallocHost(&c->h_ctl, sizeof(Ctl))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        memset(c->h_ctl, 0, sizeof(Ctl));
        if ((e = cudaMemcpy(c->d_ctl, c->h_ctl, sizeof(Ctl), cudaMemcpyHostToDevice)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaStreamCreateWithFlags(&h->run_stream, cudaStreamNonBlocking)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaEventCreateWithFlags(&h->ev_in, cudaEventDisableTiming)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaEventCreateWithFlags(&h->ev_out, cudaEventDisableTiming)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        rc = force_static_init(c);
        if (rc != NBODY_OK) break;
        if ((e = cudaFuncSetAttribute((const void *)k_select, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      kSelRows * kSelThreads * (int)sizeof(unsigned long long))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaDeviceSynchronize()) != cudaSuccess) { rc = cuda_fail(c, e); break; }
    } while (0);
    if (rc != NBODY_OK) {
        nbody_destroy(h);
        return rc;
    }
    *out = h;
    return NBODY_OK;
}

int nbody_destroy(nbody_ctx *h) {
    if (!h) return NBODY_OK;
    Ctx *c = &h->c;
    DeviceGuard guard(c->device);
    cudaDeviceSynchronize();
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->graph_small) cudaGraphExecDestroy(c->graph_small);
    if (h->ev_in) cudaEventDestroy(h->ev_in);
    if (h->ev_out) cudaEventDestroy(h->ev_out);
    if (h->run_stream) cudaStreamDestroy(h->run_stream);
    cudaFree(c->jstore);
    cudaFree(c->partials);
    cudaFree(c->d_counts);
    cudaFree(c->d_ctl);
    cudaFree(c->d_keys);
    cudaFree(c->d_cand);
    cudaFree(c->d_flag);
    cudaFree(c->stage);
    if (c->h_ctl) cudaFreeHost(c->h_ctl);
    cudaGetLastError();
    delete h;
    return NBODY_OK;
}

int nbody_last_cuda_error(const nbody_ctx *h) { return h ? h->c.last_cuda_error : 0; }
int64_t nbody_launch_count(const nbody_ctx *h) { return h ? h->c.launches : 0; }

int nbody_last_force_geometry(const nbody_ctx *h, int *r, int *jl, int *s, int64_t *ctas) {
    if (!h) return NBODY_EINVAL;
    if (r) *r = h->c.last_r;
    if (jl) *jl = h->c.last_jl;
    if (s) *s = h->c.last_s;
    if (ctas) *ctas = h->c.last_ctas;
    return NBODY_OK;
}

int nbody_set_option(nbody_ctx *h, const char *key, int64_t value) {
    if (!h || !key) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (!strcmp(key, "diff_mode")) {
        if (value != 0 && value != 1) return NBODY_EINVAL;
        c->diff_mode = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "force_split")) {
        if (value < 0 || value > 65535) return NBODY_EINVAL;
        c->force_split = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "dt_criterion_order")) {
        if (value != 0 && value != 4 && value != 6 && value != 8) return NBODY_EINVAL;
        c->crit_order = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "force_lanes")) {
        if (value != 0 && !(value >= 1 && value <= 256 && (value & (value - 1)) == 0)) return NBODY_EINVAL;
        c->force_lanes = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "geometry_n_act")) {
        if (value < 0 || value > c->cap) return NBODY_EINVAL;
        c->geometry_n_act = value;
        return NBODY_OK;
    }
    if (!strcmp(key, "validate")) {
        if (value != 0 && value != 1) return NBODY_EINVAL;
        c->validate = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "corrector_order_limit")) {
        if (value != 0 && value != 1) return NBODY_EINVAL;
        c->limit_order = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "step_reject_ratio")) {
        if (value != 0 && (value < 2 || value > (1 << 20) || (value & (value - 1)) != 0)) return NBODY_EINVAL;
        c->reject_ratio = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "use_fused")) {
        if (value != 0 && value != 1) return NBODY_EINVAL;
        c->use_fused = (int)value;
        return NBODY_OK;
    }
    if (!strcmp(key, "use_graph")) {
        if (value != 0 && value != 1) return NBODY_EINVAL;
        c->use_graph = (int)value;
        return NBODY_OK;
    }
    return NBODY_EINVAL;
}

int nbody_predict(nbody_ctx *h, int64_t n, double t_now, int order, const double *t, const double *m,
                  const double *x, const double *v, const double *const a_derivs[6], void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n < 0 || n > h->c.cap) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (n > 0) {
        if (!t || !m || !x || !v || !a_derivs) return NBODY_EINVAL;
        NB_ALIGN8(t, m, x, v);
        for (int k = 0; k <= order - 3; ++k)
            if (!a_derivs[k] || misaligned(a_derivs[k], 8)) return NBODY_EINVAL;
    }
    DeviceGuard guard(c->device);
    c->n = n;
    c->n_pad = (n + kTileJ - 1) / kTileJ * kTileJ;
    c->pred_order = order;
    c->ds_valid = c->diff_mode == 1;
    if (n == 0) return NBODY_OK;
    c->launches += 1;
    return launch_predict(c, n, t_now, order, t, m, x, v, a_derivs, nullptr, (cudaStream_t)stream);
}

int nbody_force(nbody_ctx *h, const int32_t *active_idx, int64_t n_act, int order, double eps2, double *acc,
                double *jerk, double *snap, double *crackle, double *pot, void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n_act < 0) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (!(eps2 >= 0.0) || isinf(eps2)) return NBODY_EINVAL;
    if (eps2 > 0.0 && (float)eps2 < 1.17549435e-38f) return NBODY_EINVAL;  // would flush to 0 in the fp32 pair arithmetic
    if (c->n < 0 || order > c->pred_order) return NBODY_ESTATE;
    if (n_act > c->n) return NBODY_EINVAL;
    if (n_act == 0) return NBODY_OK;
    if (!active_idx || !acc || !jerk || !pot || (order >= 6 && !snap) || (order >= 8 && !crackle)) return NBODY_EINVAL;
    NB_ALIGN8(acc, jerk, snap, crackle, pot);
    if (misaligned(active_idx, 4)) return NBODY_EINVAL;
    if (c->diff_mode == 1 && !c->ds_valid) return NBODY_ESTATE;
    DeviceGuard guard(c->device);
    if (c->validate) {
        const int rc = validate_active(c, active_idx, n_act, c->n, nullptr, nullptr, 0.0, (cudaStream_t)stream);
        if (rc != NBODY_OK) return rc;
    }
    return launch_force(c, active_idx, n_act, order, (float)eps2, acc, jerk, snap, crackle, pot, (cudaStream_t)stream);
}

int nbody_force_static(nbody_ctx *h, const int32_t *active_idx, int64_t n_act, int order, double eps2, double *acc,
                       double *jerk, double *snap, double *crackle, double *pot, void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n_act < 0) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (!(eps2 >= 0.0) || isinf(eps2)) return NBODY_EINVAL;
    if (eps2 > 0.0 && (float)eps2 < 1.17549435e-38f) return NBODY_EINVAL;  // would flush to 0 in the fp32 pair arithmetic
    if (c->n < 0 || order > c->pred_order) return NBODY_ESTATE;
    if (n_act > c->n) return NBODY_EINVAL;
    DeviceGuard guard(c->device);
    if (n_act == 0)  // set-up only: resolves the static array's device address on this device
        return launch_force_static(c, nullptr, 0, order, (float)eps2, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);
    if (!active_idx || !acc || !jerk || !pot || (order >= 6 && !snap) || (order >= 8 && !crackle)) return NBODY_EINVAL;
    NB_ALIGN8(acc, jerk, snap, crackle, pot);
    if (misaligned(active_idx, 4)) return NBODY_EINVAL;
    if (c->diff_mode == 1 && !c->ds_valid) return NBODY_ESTATE;
    if (c->validate) {
        const int rc = validate_active(c, active_idx, n_act, c->n, nullptr, nullptr, 0.0, (cudaStream_t)stream);
        if (rc != NBODY_OK) return rc;
    }
    return launch_force_static(c, active_idx, n_act, order, (float)eps2, acc, jerk, snap, crackle, pot,
                               (cudaStream_t)stream);
}

int nbody_correct(nbody_ctx *h, const int32_t *active_idx, int64_t n_act, int order, double t_now, double eta,
                  double dt_min, double dt_max, double *t, double *dt, double *x, double *v,
                  double *const a_derivs[8], double *pot_state, const double *acc, const double *jerk,
                  const double *snap, const double *crackle, const double *pot, void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n_act < 0) return NBODY_EINVAL;
    Ctx *c = &h->c;
    int kmin, kmax;
    if (!(eta > 0.0) || !is_pow2(dt_min, &kmin) || !is_pow2(dt_max, &kmax) || dt_min > dt_max) return NBODY_EINVAL;
    if (!dt_range_ok(kmin, kmax, criterion_order(c, order) - 3)) return NBODY_EINVAL;
    if (n_act == 0) return NBODY_OK;
    if (!active_idx || !t || !dt || !x || !v || !a_derivs || !pot_state || !acc || !jerk || !pot) return NBODY_EINVAL;
    if ((order >= 6 && !snap) || (order >= 8 && !crackle)) return NBODY_EINVAL;
    NB_ALIGN8(t, dt, x, v, pot_state, acc, jerk, snap, crackle, pot);
    if (misaligned(active_idx, 4)) return NBODY_EINVAL;
    for (int k = 0; k < order; ++k)
        if (!a_derivs[k] || misaligned(a_derivs[k], 8)) return NBODY_EINVAL;
    DeviceGuard guard(c->device);
    if (c->validate) {
        const int rc = validate_active(c, active_idx, n_act, c->cap, t, dt, t_now, (cudaStream_t)stream);
        if (rc != NBODY_OK) return rc;
    }
    c->launches += 1;
    return launch_correct(c, active_idx, n_act, order, t_now, eta, dt_min, dt_max, kmin, kmax, t, dt, x, v, a_derivs,
                          pot_state, acc, jerk, snap, crackle, pot, nullptr, (cudaStream_t)stream);
}

int nbody_initial_dt(nbody_ctx *h, int64_t n, const double *acc, const double *jerk, double eta_s, double dt_min,
                     double dt_max, double *dt, void *stream) {
    if (!h || n < 0) return NBODY_EINVAL;
    int kmin, kmax;
    if (!(eta_s > 0.0) || !is_pow2(dt_min, &kmin) || !is_pow2(dt_max, &kmax) || dt_min > dt_max) return NBODY_EINVAL;
    if (!dt_range_ok(kmin, kmax, 1)) return NBODY_EINVAL;
    if (n == 0) return NBODY_OK;
    if (!acc || !jerk || !dt) return NBODY_EINVAL;
    NB_ALIGN8(acc, jerk, dt);
    Ctx *c = &h->c;
    DeviceGuard guard(c->device);
    k_initial_dt<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n, acc, jerk, eta_s, kmin, kmax, dt_min,
                                                                              dt_max, dt);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_next_block(nbody_ctx *h, int64_t n, const double *t, const double *dt, int32_t *active_idx,
                     double *t_next_host, int64_t *n_act_host, void *stream) {
    if (!h || n < 1 || n > h->c.cap || !t || !dt || !active_idx || !t_next_host || !n_act_host) return NBODY_EINVAL;
    NB_ALIGN8(t, dt);
    if (misaligned(active_idx, 4)) return NBODY_EINVAL;
    Ctx *c = &h->c;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    SelArgs A;
    fill_select(h, A, n, t, dt, active_idx, /*run_mode=*/0, n);
    k_select<<<select_grid(c, n), kSelThreads, select_smem(c, n), st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    NB_CUDA(c, cudaMemcpyAsync(c->h_ctl, c->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    *t_next_host = c->h_ctl->t_next;
    *n_act_host = (int64_t)c->h_ctl->n_act;
    return NBODY_OK;
}

int nbody_get_predicted(nbody_ctx *h, double *xp, float *vp, float *ap, float *jp, float *m32, void *stream) {
    if (!h || !xp || !vp || !m32) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (c->n < 0) return NBODY_ESTATE;
    if ((ap && c->pred_order < 6) || (jp && c->pred_order < 8)) return NBODY_EINVAL;
    if (c->n == 0) return NBODY_OK;
    DeviceGuard guard(c->device);
    const uint4 *q = c->jstore;
    k_unpack<<<(unsigned)((c->n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        q, q + c->cap_pad, q + 2 * c->cap_pad, q + 3 * c->cap_pad, c->n, c->pred_order, xp, vp, ap, jp, m32);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_nearest(nbody_ctx *h, const int32_t *active_idx, int64_t n_act, int32_t *nn_idx, double *nn_r2, void *stream) {
    if (!h || n_act < 0) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (c->n < 0) return NBODY_ESTATE;
    if (n_act > c->n) return NBODY_EINVAL;
    if (n_act == 0) return NBODY_OK;
    if (!active_idx || !nn_idx || !nn_r2) return NBODY_EINVAL;
    NB_ALIGN8(nn_r2);
    if (misaligned(active_idx, 4) || misaligned(nn_idx, 4)) return NBODY_EINVAL;
    if ((size_t)n_act * sizeof(unsigned long long) > c->partials_bytes) return NBODY_ENOMEM;  // keys live in the split scratch
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (c->validate) {
        const int rc = validate_active(c, active_idx, n_act, c->n, nullptr, nullptr, 0.0, st);
        if (rc != NBODY_OK) return rc;
    }
    unsigned long long *keys = reinterpret_cast<unsigned long long *>(c->partials);
    NB_CUDA(c, cudaMemsetAsync(keys, 0xff, (size_t)n_act * sizeof(unsigned long long), st));
    const int n_tiles = (int)((c->n + kNnTile - 1) / kNnTile);
    const long long i_tiles = (n_act + kNnTile - 1) / kNnTile;
    long long S = (4LL * c->sm_count + i_tiles - 1) / i_tiles;  // about four CTAs per SM in flight
    if (S > n_tiles) S = n_tiles;
    if (S > 65535) S = 65535;
    if (S < 1) S = 1;
    const uint4 *q = c->jstore;
    k_nearest<<<dim3((unsigned)i_tiles, (unsigned)S), kNnTile, 0, st>>>(q, q + c->cap_pad, c->n, active_idx, (int)n_act,
                                                                        n_tiles, (int)S, keys);
    NB_CUDA(c, cudaGetLastError());
    k_nearest_out<<<(unsigned)((n_act + 255) / 256), 256, 0, st>>>(keys, (int)n_act, nn_idx, nn_r2);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return NBODY_OK;
}

int nbody_rejected_steps(nbody_ctx *h, int reset, int64_t *count_host, void *stream) {
    if (!h || !count_host) return NBODY_EINVAL;
    Ctx *c = &h->c;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long v[2] = {0, 0};  // rejected, limited are adjacent in the control block
    NB_CUDA(c, cudaMemcpyAsync(v, &c->d_ctl->rejected, sizeof(v), cudaMemcpyDeviceToHost, st));
    if (reset) NB_CUDA(c, cudaMemsetAsync(&c->d_ctl->rejected, 0, sizeof(v), st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    count_host[0] = (int64_t)v[0];
    count_host[1] = (int64_t)v[1];
    return NBODY_OK;
}

// ---- row records for the multi-GPU exchange -----------------------------------------------------------------
static int rows_call(nbody_ctx *h, bool pack, const int32_t *idx, int64_t n_rows, int order, double *t, double *dt,
                     double *pot_state, double *x, double *v, double *const a_derivs[8], double *rec, void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n_rows < 0) return NBODY_EINVAL;
    if (n_rows == 0) return NBODY_OK;
    if (!idx || !t || !dt || !pot_state || !x || !v || !a_derivs || !rec) return NBODY_EINVAL;
    NB_ALIGN8(t, dt, pot_state, x, v, rec);
    RowArgs A;
    A.idx = idx; A.n_rows = n_rows; A.order = order; A.t = t; A.dt = dt; A.pot = pot_state; A.x = x; A.v = v; A.rec = rec;
    for (int k = 0; k < 8; ++k) {
        A.D[k] = k < order ? a_derivs[k] : nullptr;
        if (k < order && (!a_derivs[k] || misaligned(a_derivs[k], 8))) return NBODY_EINVAL;
    }
    Ctx *c = &h->c;
    DeviceGuard guard(c->device);
    long long blocks = (n_rows * (9 + 3 * order) + 255) / 256;
    if (blocks > 8LL * c->sm_count) blocks = 8LL * c->sm_count;
    if (pack) k_rows<true><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(A);
    else k_rows<false><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_pack_rows(nbody_ctx *h, const int32_t *idx, int64_t n_rows, int order, const double *t, const double *dt,
                    const double *pot_state, const double *x, const double *v, const double *const a_derivs[8],
                    double *rec, void *stream) {
    return rows_call(h, true, idx, n_rows, order, (double *)t, (double *)dt, (double *)pot_state, (double *)x, (double *)v,
                     (double *const *)a_derivs, rec, stream);
}

int nbody_unpack_rows(nbody_ctx *h, const int32_t *idx, int64_t n_rows, int order, double *t, double *dt,
                      double *pot_state, double *x, double *v, double *const a_derivs[8], const double *rec,
                      void *stream) {
    return rows_call(h, false, idx, n_rows, order, t, dt, pot_state, x, v, a_derivs, (double *)rec, stream);
}

// ---- device-driven block steps (a-1 .. a-4 without host round trips) ------------------------------------------
int nbody_run_blocks(nbody_ctx *h, int64_t n, int order, double eps2, double eta, double dt_min, double dt_max,
                     double t_end, int64_t max_blocks, int64_t max_n_act, double *t, double *dt, const double *m,
                     double *x, double *v, double *const a_derivs[8], double *pot_state, int32_t *active_idx,
                     double *acc, double *jerk, double *snap, double *crackle, double *pot, nbody_run_result *res,
                     void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n < 1 || n > h->c.cap || !res) return NBODY_EINVAL;
    Ctx *c = &h->c;
    int kmin, kmax;
    if (!(eta > 0.0) || !is_pow2(dt_min, &kmin) || !is_pow2(dt_max, &kmax) || dt_min > dt_max) return NBODY_EINVAL;
    if (!dt_range_ok(kmin, kmax, criterion_order(c, order) - 3)) return NBODY_EINVAL;
    if (!(eps2 >= 0.0) || isinf(eps2) || (eps2 > 0.0 && (float)eps2 < 1.17549435e-38f)) return NBODY_EINVAL;
    if (max_blocks < 0 || max_n_act < 1 || !(t_end == t_end)) return NBODY_EINVAL;
    if (!t || !dt || !m || !x || !v || !a_derivs || !pot_state || !active_idx || !acc || !jerk || !pot) return NBODY_EINVAL;
    if ((order >= 6 && !snap) || (order >= 8 && !crackle)) return NBODY_EINVAL;
    NB_ALIGN8(t, dt, m, x, v, pot_state, acc, jerk, snap, crackle, pot);
    if (misaligned(active_idx, 4)) return NBODY_EINVAL;
    for (int k = 0; k < order; ++k)
        if (!a_derivs[k] || misaligned(a_derivs[k], 8)) return NBODY_EINVAL;
    if (c->diff_mode != 0) return NBODY_ESTATE;  // the device-driven step is built for the literal difference mode
    DeviceGuard guard(c->device);
    cudaStream_t user = (cudaStream_t)stream, st = h->run_stream;
    memset(res, 0, sizeof(*res));

    // the private stream runs after everything the caller has queued on `stream`, and the caller's stream resumes
    // after the run (the legacy default stream cannot be captured into a graph)
    NB_CUDA(c, cudaEventRecord(h->ev_in, user));
    NB_CUDA(c, cudaStreamWaitEvent(st, h->ev_in, 0));

    // j-store bookkeeping of the ctx (what nbody_predict would set)
    c->n = n;
    c->n_pad = (n + kTileJ - 1) / kTileJ * kTileJ;
    c->pred_order = order;
    c->ds_valid = false;

    // run control
    Ctl *hc = c->h_ctl;
    memset(hc, 0, sizeof(Ctl));
    hc->t_end = t_end;
    hc->max_blocks = max_blocks;
    NB_CUDA(c, cudaMemcpyAsync(c->d_ctl, hc, sizeof(Ctl), cudaMemcpyHostToDevice, st));

    SelArgs SA, SF;
    fill_select(h, SA, n, t, dt, active_idx, /*run_mode=*/1, max_n_act);
    fill_select(h, SF, n, t, dt, active_idx, /*run_mode=*/2, max_n_act);
    const int sgrid = select_grid(c, n);
    const size_t ssmem = select_smem(c, n);
    CorrArgs CA;  // the corrector's arguments in control-block mode (shared by K_corr and the fused step)
    {
        CA.idx = active_idx; CA.n_act = 0; CA.t_now = 0.0; CA.eta = eta; CA.dt_min = dt_min; CA.dt_max = dt_max;
        CA.k_min = kmin; CA.k_max = kmax; CA.crit_order = criterion_order(c, order);
        CA.t = t; CA.dt = dt; CA.x = x; CA.v = v; CA.pot_state = pot_state;
        for (int k = 0; k < 8; ++k) CA.D[k] = k < order ? a_derivs[k] : nullptr;
        CA.acc = acc; CA.jerk = jerk; CA.snap = snap; CA.crk = crackle; CA.pot = pot;
        CA.ctl = c->d_ctl; CA.reject_ratio = c->reject_ratio; CA.n_rejected = &c->d_ctl->rejected;
        CA.limit_order = c->limit_order; CA.n_limited = &c->d_ctl->limited;
    }
    auto enqueue_step = [&](cudaStream_t s) -> int {  // general step: any block size
        k_select<<<sgrid, kSelThreads, ssmem, s>>>(SA);
        NB_CUDA(c, cudaGetLastError());
        int rc = launch_predict(c, n, 0.0, order, t, m, x, v, a_derivs, c->d_ctl, s);
        if (rc != NBODY_OK) return rc;
        rc = launch_force_dyn(c, active_idx, order, (float)eps2, acc, jerk, snap, crackle, pot, s);
        if (rc != NBODY_OK) return rc;
        // K_reduce and K_corr as two launches: one fused launch (a warp per particle, the corrector behind its reduce)
        // measured slower at every size (profiles/r02_latency.md)
        rc = launch_reduce_dyn(c, order, acc, jerk, snap, crackle, pot, s);
        if (rc != NBODY_OK) return rc;
        return launch_correct(c, active_idx, 0, order, 0.0, eta, dt_min, dt_max, kmin, kmax, t, dt, x, v, a_derivs,
                              pot_state, acc, jerk, snap, crackle, pot, c->d_ctl, s);
    };
    auto enqueue_fused = [&](cudaStream_t s) -> int {  // N1: blocks that fit one i-tile, two launches
        k_select<<<sgrid, kSelThreads, ssmem, s>>>(SF);
        NB_CUDA(c, cudaGetLastError());
        return launch_step_fused(c, order, (float)eps2, active_idx, t, m, x, v, a_derivs, CA, acc, jerk, snap, crackle,
                                 pot, s);
    };
    constexpr int kStepLaunches = 5;   // k_select, k_predict, k_force_dyn, k_reduce_dyn, k_correct
    constexpr int kFusedLaunches = 2;  // k_select, k_step_fused
    const bool fused = c->use_fused != 0;

    // CUDA graphs of the two step flavours, re-captured when any argument differs from the cached ones
    unsigned long long key[24] = {(unsigned long long)n, (unsigned long long)order, 0, 0, 0, 0,
                                  (unsigned long long)(uintptr_t)t, (unsigned long long)(uintptr_t)dt,
                                  (unsigned long long)(uintptr_t)m, (unsigned long long)(uintptr_t)x,
                                  (unsigned long long)(uintptr_t)v, (unsigned long long)(uintptr_t)pot_state,
                                  (unsigned long long)(uintptr_t)active_idx, (unsigned long long)(uintptr_t)acc,
                                  (unsigned long long)(uintptr_t)jerk, (unsigned long long)(uintptr_t)snap,
                                  (unsigned long long)(uintptr_t)crackle, (unsigned long long)(uintptr_t)pot,
                                  (unsigned long long)max_n_act,
                                  (unsigned long long)c->limit_order << 62 | (unsigned long long)c->reject_ratio << 40 |
                                      (unsigned long long)c->crit_order << 32 |
                                      (unsigned long long)c->force_lanes << 16 | (unsigned long long)c->force_split,
                                  0, 0, 0, 0};
    memcpy(&key[2], &eps2, 8); memcpy(&key[3], &eta, 8); memcpy(&key[4], &dt_min, 8); memcpy(&key[5], &dt_max, 8);
    for (int k = 0; k < order && k < 4; ++k) key[20 + k] = (unsigned long long)(uintptr_t)a_derivs[k];
    for (int k = 4; k < order; ++k) key[20 + (k & 3)] ^= (unsigned long long)(uintptr_t)a_derivs[k] * 0x9e3779b97f4a7c15ull;
    if (c->use_graph && (!c->graph_exec || memcmp(key, c->graph_key, sizeof(key)) != 0)) {
        for (cudaGraphExec_t *ge : {&c->graph_exec, &c->graph_small}) {
            if (*ge) cudaGraphExecDestroy(*ge);
            *ge = nullptr;
        }
        for (int which = 0; which < 2; ++which) {
            cudaGraph_t graph = nullptr;
            NB_CUDA(c, cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
            const int rc = which == 0 ? enqueue_step(st) : enqueue_fused(st);
            const cudaError_t e = cudaStreamEndCapture(st, &graph);
            if (rc != NBODY_OK) {
                if (graph) cudaGraphDestroy(graph);
                return rc;
            }
            NB_CUDA(c, e);
            const cudaError_t ei = cudaGraphInstantiate(which == 0 ? &c->graph_exec : &c->graph_small, graph, 0);
            cudaGraphDestroy(graph);
            NB_CUDA(c, ei);
        }
        memcpy(c->graph_key, key, sizeof(key));
    }
    auto step = [&](bool small) -> int {
        c->launches += small ? kFusedLaunches : kStepLaunches;
        if (c->use_graph) {
            const cudaError_t e = cudaGraphLaunch(small ? c->graph_small : c->graph_exec, st);
            return e == cudaSuccess ? NBODY_OK : cuda_fail(c, e);
        }
        return small ? enqueue_fused(st) : enqueue_step(st);
    };

    // batches of block steps between two looks at the control block.  With the fused step on, runs of blocks that
    // fit one i-tile go through it; a larger block stops such a batch (stop = 4) and is taken by the general step.
    int batch = 8;
    int rc = NBODY_OK;
    for (;;) {
        for (int b = 0; b < batch && rc == NBODY_OK; ++b) rc = step(fused);
        if (rc != NBODY_OK) break;
        cudaError_t e = cudaMemcpyAsync(hc, c->d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if (hc->stop == 4) {
            e = cudaMemsetAsync(&c->d_ctl->stop, 0, sizeof(int), st);
            if (e != cudaSuccess) { rc = cuda_fail(c, e); break; }
            rc = step(false);
            if (rc != NBODY_OK) break;
            if (batch > 8) batch /= 2;
            continue;
        }
        if (hc->stop) break;
        if (batch < 64) batch *= 2;
    }
    if (rc != NBODY_OK) {
        cudaStreamSynchronize(st);
        return rc;
    }
    res->blocks = (int64_t)hc->blocks;
    res->pairs = (int64_t)hc->pairs;
    res->t_next = hc->t_next;
    res->n_act_next = (int64_t)hc->n_act;
    res->stop_reason = hc->stop;
    res->rejected = (int64_t)hc->rejected;
    res->limited = (int64_t)hc->limited;
    for (int b = 0; b < 40; ++b) res->hist_log2[b] = (int64_t)hc->hist[b];
    NB_CUDA(c, cudaEventRecord(h->ev_out, st));
    NB_CUDA(c, cudaStreamWaitEvent(user, h->ev_out, 0));
    return NBODY_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// Host-buffer path (end-to-end measurement): H2D of the state, predict, force, D2H of the results.
// ---------------------------------------------------------------------------------------------------------
namespace {
// error exit of the *_host calls: drain the stream first, so that no copy from/to caller-owned host memory is in flight
inline int host_fail(Ctx *c, cudaStream_t st, int rc) {
    cudaStreamSynchronize(st);
    (void)c;
    return rc;
}
#define NB_CUDA_H(ctx, st, expr)                                               \
    do {                                                                       \
        cudaError_t e__ = (expr);                                              \
        if (e__ != cudaSuccess) return host_fail(ctx, st, ::nbody::cuda_fail(ctx, e__)); \
    } while (0)

int ensure_stage(Ctx *c, size_t need) {
    if (need <= c->stage_bytes) return NBODY_OK;
    NB_CUDA(c, cudaDeviceSynchronize());
    cudaFree(c->stage);
    c->stage = nullptr;
    c->stage_bytes = 0;
    NB_CUDA(c, cudaMalloc(&c->stage, need));
    c->stage_bytes = need;
    return NBODY_OK;
}
}  // namespace

extern "C" int nbody_force_host(nbody_ctx *h, int64_t n, double t_now, int order, const double *t, const double *m,
                                const double *x, const double *v, const double *const a_derivs[6],
                                const int32_t *active_idx, int64_t n_act, double eps2, double *acc, double *jerk,
                                double *snap, double *crackle, double *pot, int64_t *h2d_bytes, int64_t *d2h_bytes) {
    if (!h || (order != 4 && order != 6 && order != 8) || n < 1 || n > h->c.cap || n_act < 0 || n_act > n)
        return NBODY_EINVAL;
    if (!t || !m || !x || !v || !a_derivs || (n_act > 0 && (!active_idx || !acc || !jerk || !pot))) return NBODY_EINVAL;
    if (n_act > 0 && ((order >= 6 && !snap) || (order >= 8 && !crackle))) return NBODY_EINVAL;
    if (!(eps2 >= 0.0) || isinf(eps2) || (eps2 > 0.0 && (float)eps2 < 1.17549435e-38f)) return NBODY_EINVAL;
    const int nd = order - 2, K = order / 2;
    for (int k = 0; k < nd; ++k)
        if (!a_derivs[k]) return NBODY_EINVAL;
    Ctx *c = &h->c;
    DeviceGuard guard(c->device);
    // staging layout (doubles): t[n] m[n] x[3n] v[3n] D[nd][3n] | out: K x [3 n_act] + pot[n_act] | idx int32[n_act]
    const size_t in_d = (size_t)n * (2 + 6 + 3 * (size_t)nd);
    const size_t out_d = (size_t)n_act * (3 * (size_t)K + 1);
    const size_t need = (in_d + out_d) * sizeof(double) + (size_t)n_act * sizeof(int32_t) + 256;
    int rc = ensure_stage(c, need);
    if (rc != NBODY_OK) return rc;
    cudaStream_t st = 0;
    double *d = (double *)c->stage;
    double *dt_ = d, *dm = d + n, *dx = d + 2 * n, *dv = d + 5 * n;
    const double *dD[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int64_t up = 0, down = 0;
    NB_CUDA_H(c, st, cudaMemcpyAsync(dt_, t, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    NB_CUDA_H(c, st, cudaMemcpyAsync(dm, m, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    NB_CUDA_H(c, st, cudaMemcpyAsync(dx, x, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st));
    NB_CUDA_H(c, st, cudaMemcpyAsync(dv, v, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st));
    up += (int64_t)sizeof(double) * 8 * n;
    for (int k = 0; k < nd; ++k) {
        double *p = d + 8 * n + (size_t)k * 3 * n;
        NB_CUDA_H(c, st, cudaMemcpyAsync(p, a_derivs[k], sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st));
        dD[k] = p;
        up += (int64_t)sizeof(double) * 3 * n;
    }
    double *o = d + in_d;
    double *o_acc = o, *o_jerk = o + 3 * n_act, *o_snap = nullptr, *o_crk = nullptr;
    double *cur = o + 6 * n_act;
    if (order >= 6) { o_snap = cur; cur += 3 * n_act; }
    if (order >= 8) { o_crk = cur; cur += 3 * n_act; }
    double *o_pot = cur;
    int32_t *d_idx = (int32_t *)(o + out_d);
    rc = nbody_predict(h, n, t_now, order, dt_, dm, dx, dv, dD, st);
    if (rc != NBODY_OK) return host_fail(c, st, rc);
    if (n_act > 0) {
        NB_CUDA_H(c, st, cudaMemcpyAsync(d_idx, active_idx, sizeof(int32_t) * n_act, cudaMemcpyHostToDevice, st));
        up += (int64_t)sizeof(int32_t) * n_act;
        rc = nbody_force(h, d_idx, n_act, order, eps2, o_acc, o_jerk, o_snap, o_crk, o_pot, st);
        if (rc != NBODY_OK) return host_fail(c, st, rc);
        NB_CUDA_H(c, st, cudaMemcpyAsync(acc, o_acc, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        NB_CUDA_H(c, st, cudaMemcpyAsync(jerk, o_jerk, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        if (order >= 6) NB_CUDA_H(c, st, cudaMemcpyAsync(snap, o_snap, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        if (order >= 8) NB_CUDA_H(c, st, cudaMemcpyAsync(crackle, o_crk, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        NB_CUDA_H(c, st, cudaMemcpyAsync(pot, o_pot, sizeof(double) * n_act, cudaMemcpyDeviceToHost, st));
        down += (int64_t)sizeof(double) * n_act * (3 * K + 1);
    }
    NB_CUDA(c, cudaStreamSynchronize(st));
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return NBODY_OK;
}

// ---------------------------------------------------------------------------------------------------------
// One whole block step with HOST state (a-1 .. a-4): H2D of the state, selection, predict, force, correct,
// D2H of the updated state.  Same kernels as the device-pointer calls.
// ---------------------------------------------------------------------------------------------------------
extern "C" int nbody_step_host(nbody_ctx *h, int64_t n, int order, double eps2, double eta, double dt_min,
                               double dt_max, double *t, double *dt, const double *m, double *x, double *v,
                               double *const a_derivs[8], double *pot_state, double *t_next_host,
                               int64_t *n_act_host, int64_t *h2d_bytes, int64_t *d2h_bytes) {
    if (!h || (order != 4 && order != 6 && order != 8) || n < 1 || n > h->c.cap) return NBODY_EINVAL;
    if (!t || !dt || !m || !x || !v || !a_derivs || !pot_state || !t_next_host || !n_act_host) return NBODY_EINVAL;
    for (int k = 0; k < order; ++k)
        if (!a_derivs[k]) return NBODY_EINVAL;
    Ctx *c = &h->c;
    {  // every argument the inner calls would reject is rejected here, before the first copy is queued
        int kmin, kmax;
        if (!(eta > 0.0) || !is_pow2(dt_min, &kmin) || !is_pow2(dt_max, &kmax) || dt_min > dt_max) return NBODY_EINVAL;
        if (!dt_range_ok(kmin, kmax, criterion_order(c, order) - 3)) return NBODY_EINVAL;
        if (!(eps2 >= 0.0) || isinf(eps2) || (eps2 > 0.0 && (float)eps2 < 1.17549435e-38f)) return NBODY_EINVAL;
    }
    DeviceGuard guard(c->device);
    const int K = order / 2;
    // staging (doubles): t dt m pot [n] | x v [3n] | D[order][3n] | acc jerk snap crk [3n] fpot [n] | idx int32[n]
    const size_t nd = (size_t)n * (4 + 6 + 3 * (size_t)order + 12 + 1);
    const size_t need = nd * sizeof(double) + (size_t)n * sizeof(int32_t) + 256;
    int rc = ensure_stage(c, need);
    if (rc != NBODY_OK) return rc;
    cudaStream_t st = 0;
    double *d = (double *)c->stage;
    double *d_t = d, *d_dt = d + n, *d_m = d + 2 * n, *d_pot = d + 3 * n, *d_x = d + 4 * n, *d_v = d + 7 * n;
    double *d_D[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    for (int k = 0; k < order; ++k) d_D[k] = d + 10 * n + (size_t)k * 3 * n;
    double *o = d + 10 * n + (size_t)order * 3 * n;
    double *o_acc = o, *o_jerk = o + 3 * n, *o_snap = o + 6 * n, *o_crk = o + 9 * n, *o_pot = o + 12 * n;
    int32_t *d_idx = (int32_t *)(o + 13 * n);
    int64_t up = 0, down = 0;
    auto h2d = [&](double *dst, const double *src, size_t cnt) {
        up += (int64_t)(cnt * sizeof(double));
        return cudaMemcpyAsync(dst, src, cnt * sizeof(double), cudaMemcpyHostToDevice, st);
    };
    auto d2h = [&](double *dst, const double *src, size_t cnt) {
        down += (int64_t)(cnt * sizeof(double));
        return cudaMemcpyAsync(dst, src, cnt * sizeof(double), cudaMemcpyDeviceToHost, st);
    };
    NB_CUDA_H(c, st, h2d(d_t, t, n));
    NB_CUDA_H(c, st, h2d(d_dt, dt, n));
    NB_CUDA_H(c, st, h2d(d_m, m, n));
    NB_CUDA_H(c, st, h2d(d_pot, pot_state, n));
    NB_CUDA_H(c, st, h2d(d_x, x, 3 * n));
    NB_CUDA_H(c, st, h2d(d_v, v, 3 * n));
    for (int k = 0; k < order; ++k) NB_CUDA_H(c, st, h2d(d_D[k], a_derivs[k], 3 * n));
    double t_next = 0.0;
    int64_t n_act = 0;
    rc = nbody_next_block(h, n, d_t, d_dt, d_idx, &t_next, &n_act, st);
    if (rc != NBODY_OK) return host_fail(c, st, rc);
    rc = nbody_predict(h, n, t_next, order, d_t, d_m, d_x, d_v, d_D, st);
    if (rc != NBODY_OK) return host_fail(c, st, rc);
    rc = nbody_force(h, d_idx, n_act, order, eps2, o_acc, o_jerk, K >= 3 ? o_snap : nullptr, K >= 4 ? o_crk : nullptr,
                     o_pot, st);
    if (rc != NBODY_OK) return host_fail(c, st, rc);
    rc = nbody_correct(h, d_idx, n_act, order, t_next, eta, dt_min, dt_max, d_t, d_dt, d_x, d_v, d_D, d_pot, o_acc,
                       o_jerk, K >= 3 ? o_snap : nullptr, K >= 4 ? o_crk : nullptr, o_pot, st);
    if (rc != NBODY_OK) return host_fail(c, st, rc);
    NB_CUDA_H(c, st, d2h(t, d_t, n));
    NB_CUDA_H(c, st, d2h(dt, d_dt, n));
    NB_CUDA_H(c, st, d2h(pot_state, d_pot, n));
    NB_CUDA_H(c, st, d2h(x, d_x, 3 * n));
    NB_CUDA_H(c, st, d2h(v, d_v, 3 * n));
    for (int k = 0; k < order; ++k) NB_CUDA_H(c, st, d2h(a_derivs[k], d_D[k], 3 * n));
    NB_CUDA(c, cudaStreamSynchronize(st));
    *t_next_host = t_next;
    *n_act_host = n_act;
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return NBODY_OK;
}
