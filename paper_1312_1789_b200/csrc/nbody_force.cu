// libnbody.so, translation unit 2: K_force (a-3) and K_reduce (a-3b).
//
// K_force computes, for each active i, the sums of DESIGN.md R1 (= SURVEY.md c-1; the paper prints no formula,
// PAPER.md:15/:43 name the scheme, PAPER.md:31 the mixed precision) over the packed j-store:
//   - every thread owns TWO i-particles and runs the fp32 pair arithmetic on both at once with Blackwell's packed
//     f32x2 instructions (PTX fma/mul/add.f32x2 -> SASS FFMA2 / FMUL2 / FADD2): lane 0 = first i, lane 1 = second i.
//     The scalar form is limited by issue slots and by register-file bandwidth (a 3-source FFMA with two sources in
//     the same register bank takes 2 cycles); the packed form reads aligned 64-bit register pairs and halves the
//     instruction count of the fp32 part.  The j operand of a packed instruction is the broadcast pair {v, v},
//     which ptxas folds into a 32-bit broadcast register operand (SASS `Rn.F32`), so the j-store stays compact;
//   - j-tiles of kTileJ particles are staged plane by plane into shared memory by 1-D TMA bulk copies
//     (cp.async.bulk + mbarrier) through a 4-stage ring with per-stage full/empty mbarriers (no __syncthreads in
//     the loop); every pair-loop read is an LDS.128 broadcast;
//   - d = fl32(x_j - x_i) with the subtraction in fp64 (DIFF 0: DADD + F2F per lane) or double-single (DIFF 1:
//     packed fp32 adds of hi and lo parts); MUFU.RSQ per lane; fp32 partial sums over <= 64 consecutive j, then
//     fp64 accumulators, which live in shared memory (one slot per thread and component) to free registers (R10);
//   - the pair is cut into a head (differences, r^2, rsqrt: the LDS -> DADD -> F2F -> MUFU latency chain) and a
//     tail (the FFMA2 block); at order 8 the heads of two j are issued before their tails (no register spills);
//   - the self pair (R2) and the zero-mass pads above n are excluded by index, but the compare/select is only
//     executed by warps whose i-indices fall inside the current j-tile or whose tile holds pads (warp-uniform
//     branch), so the main loop is mask-free;
//   - a work item is (i-tile, j-split): IT = kThreads/JL i-lanes x JL j-lanes (2 IT i-particles): JL = 1 for big
//     blocks (every lane reads the same j: smem broadcast), JL up to 256 for tiny blocks; the j-lanes are reduced
//     through shared memory in fixed order; S > 1 j-splits write fp64 partials [S][NC][n_act] that K_reduce sums
//     in order.  k_force takes the geometry from the host (grid = i-tiles x S); k_force_dyn is the persistent
//     form of the same work items (grid = SMs) that reads n_act and the geometry from the device control block
//     (device-driven block step, nbody_run_blocks); k_reduce_dyn is K_reduce of that step (S, n_act from the control block).
#include <math.h>

#include <mutex>

#include "nbody_exact.cuh"
#include "nbody_internal.h"


namespace nbody {
namespace {


// ---- TMA / mbarrier primitives (PTX) -------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// ---- scalar helpers ------------------------------------------------------------------------------------
__device__ __forceinline__ double u2d(unsigned lo, unsigned hi) { return __hiloint2double((int)hi, (int)lo); }
__device__ __forceinline__ float u2f(unsigned u) { return __uint_as_float(u); }
// fp64 -> fp32, round to nearest even.  Written in PTX without .ftz: under -ftz=true the intrinsic would expand
// to F2F + DSETP + predicated FMUL (denormal flush), 2 extra instructions per coordinate.
__device__ __forceinline__ float d2f(double x) {
    float r;
    asm("cvt.rn.f32.f64 %0, %1;" : "=f"(r) : "d"(x));
    return r;
}
__device__ __forceinline__ float frsqrt(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---- packed f32x2 (one 64-bit register pair = {lane 0, lane 1}) -----------------------------------------
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float a, float b) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ f2 pku(unsigned a, unsigned b) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(a), "r"(b));
    return r;
}
// broadcast pair {v, v}: ptxas folds it into a 32-bit broadcast operand (Rn.F32) of the packed instruction
__device__ __forceinline__ f2 bc(unsigned v) { return pku(v, v); }
__device__ __forceinline__ void upk(f2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) {
    f2 r;
    asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b) {
    f2 r;
    asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
    f2 r;
    asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

template <int ORDER, int DIFF>
struct Geo {
    static constexpr int K = ORDER / 2;
    static constexpr int NC = 3 * K + 1;                        // components per i: 3K vectors + pot
    static constexpr int NQ = ORDER == 4 ? 3 : 4;               // planes staged per tile (Q0..Q3 | Q4, Q5, Q2, Q3)
    static constexpr int STAGES = 4;  // TMA ring depth
    static constexpr uint32_t STAGE_BYTES = NQ * kTileJ * 16;
    static constexpr size_t TILE_BYTES = (size_t)STAGES * STAGE_BYTES;
    static constexpr size_t ACC_BYTES = (size_t)2 * NC * kThreads * sizeof(double);
    static constexpr size_t SMEM = TILE_BYTES + ACC_BYTES + 128;  // + full/empty mbarriers
};

struct ForceArgs {
    const uint4 *q[4];  // planes in use: {Q0,Q1,Q2,Q3} (DIFF 0) or {Q4,Q5,Q2,Q3} (DIFF 1)
    const int32_t *idx;
    int n;              // particles in the j-store; entries [n, n_tiles * kTileJ) are pads, masked by index
    int n_act;          // host-geometry kernel only (k_force_dyn reads it from ctl)
    int n_tiles;
    int splits;         // host-geometry kernel only
    float eps2;
    double *out[5];     // acc, jerk, snap, crackle, pot (used when splits == 1)
    double *partials;   // [splits][NC][n_act]           (used when splits > 1)
    const Ctl *ctl;     // device control block (k_force_dyn)
};

template <int ORDER, int DIFF>
struct IPair {          // the thread's two i-particles
    double x[2][3];     // DIFF 0
    f2 nxh[3], nxl[3];  // DIFF 1: negated hi and lo parts
    f2 nv[3], na[3], nj[3];  // negated, so that a difference is one packed add
    int idx[2];
};

struct Consts {  // loop-invariant packed constants
    f2 eps2, m3, three, m4;
    int n;  // first pad index
};

// One j against the thread's two i-particles, in two parts.  head: d, r^2, rsqrt (LDS, DADD, F2F, FFMA2 x 3, MUFU: the
// long-latency chain); tail: everything else, accumulating into pa[0 .. 3K] (pot as +m/r, negated at the end).
// tq = base of the staged tile (plane p at tq + p * kTileJ), jt = index inside the tile.
struct Stage {
    f2 d[3];
    f2 rinv;
    unsigned m, vx;
};

template <int ORDER, int DIFF, bool MASK>
__device__ __forceinline__ void head(const IPair<ORDER, DIFF> &I, const uint4 *tq, int jt, int jglob, const Consts &C,
                                     Stage &S) {
    const uint4 qa = tq[jt];
    const uint4 qb = tq[kTileJ + jt];
    if (DIFF == 0) {
        const double xj = u2d(qa.x, qa.y), yj = u2d(qa.z, qa.w), zj = u2d(qb.x, qb.y);
        S.d[0] = pk(d2f(xj - I.x[0][0]), d2f(xj - I.x[1][0]));
        S.d[1] = pk(d2f(yj - I.x[0][1]), d2f(yj - I.x[1][1]));
        S.d[2] = pk(d2f(zj - I.x[0][2]), d2f(zj - I.x[1][2]));
    } else {
        S.d[0] = add2(add2(bc(qa.x), I.nxh[0]), add2(bc(qa.y), I.nxl[0]));
        S.d[1] = add2(add2(bc(qa.z), I.nxh[1]), add2(bc(qa.w), I.nxl[1]));
        S.d[2] = add2(add2(bc(qb.x), I.nxh[2]), add2(bc(qb.y), I.nxl[2]));
    }
    S.m = qb.z;
    S.vx = qb.w;
    f2 r2 = fma2(S.d[0], S.d[0], C.eps2);
    r2 = fma2(S.d[1], S.d[1], r2);
    r2 = fma2(S.d[2], S.d[2], r2);
    float r0, r1;
    upk(r2, r0, r1);
    r0 = frsqrt(r0);
    r1 = frsqrt(r1);
    if (MASK) {  // R2: the self pair is excluded by index; so are the pads above n
        r0 = (jglob == I.idx[0] || jglob >= C.n) ? 0.f : r0;
        r1 = (jglob == I.idx[1] || jglob >= C.n) ? 0.f : r1;
    }
    S.rinv = pk(r0, r1);
}

template <int ORDER, int DIFF>
__device__ __forceinline__ void tail(const IPair<ORDER, DIFF> &I, const uint4 *tq, int jt, const Consts &C,
                                     const Stage &S, f2 *pa) {
    const f2 *d = S.d;
    const f2 mj = bc(S.m);
    const uint4 qc = tq[2 * kTileJ + jt];  // Q2 = { vy, vz, ax, ay }
    f2 dv[3], dj[3], da[3];
    dv[0] = add2(bc(S.vx), I.nv[0]);
    dv[1] = add2(bc(qc.x), I.nv[1]);
    dv[2] = add2(bc(qc.y), I.nv[2]);
    f2 rv = mul2(d[0], dv[0]);
    rv = fma2(d[1], dv[1], rv);
    rv = fma2(d[2], dv[2], rv);
    const f2 rinv = S.rinv;
    const f2 rinv2 = mul2(rinv, rinv);
    const f2 mrinv = mul2(mj, rinv);
    const f2 q = mul2(mrinv, rinv2);
    const f2 alpha = mul2(rv, rinv2);
    constexpr int K = ORDER / 2;
    pa[3 * K] = add2(pa[3 * K], mrinv);
    const f2 c1 = mul2(C.m3, alpha);
    f2 Jp[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        Jp[c] = fma2(c1, d[c], dv[c]);
        pa[c] = fma2(q, d[c], pa[c]);
        pa[3 + c] = fma2(q, Jp[c], pa[3 + c]);
    }
    if (ORDER >= 6) {
        const uint4 qd = tq[3 * kTileJ + jt];  // Q3 = { az, jx, jy, jz }
        da[0] = add2(bc(qc.z), I.na[0]);
        da[1] = add2(bc(qc.w), I.na[1]);
        da[2] = add2(bc(qd.x), I.na[2]);
        f2 w = mul2(dv[0], dv[0]);
        w = fma2(dv[1], dv[1], w);
        w = fma2(dv[2], dv[2], w);
        w = fma2(d[0], da[0], w);
        w = fma2(d[1], da[1], w);
        w = fma2(d[2], da[2], w);
        const f2 beta = fma2(alpha, alpha, mul2(w, rinv2));
        const f2 c2 = add2(c1, c1);
        const f2 c3 = mul2(C.m3, beta);
        f2 Sp[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Sp[c] = fma2(c3, d[c], fma2(c2, Jp[c], da[c]));
            pa[6 + c] = fma2(q, Sp[c], pa[6 + c]);
        }
        if (ORDER >= 8) {
            dj[0] = add2(bc(qd.y), I.nj[0]);
            dj[1] = add2(bc(qd.z), I.nj[1]);
            dj[2] = add2(bc(qd.w), I.nj[2]);
            f2 va = mul2(dv[0], da[0]);
            va = fma2(dv[1], da[1], va);
            va = fma2(dv[2], da[2], va);
            f2 g = mul2(C.three, va);
            g = fma2(d[0], dj[0], g);
            g = fma2(d[1], dj[1], g);
            g = fma2(d[2], dj[2], g);
            const f2 t = fma2(mul2(C.m4, alpha), alpha, mul2(C.three, beta));
            const f2 gamma = fma2(alpha, t, mul2(g, rinv2));
            const f2 c4 = mul2(C.three, c1);  // -9 alpha
            const f2 c5 = mul2(C.three, c3);  // -9 beta
            const f2 c6 = mul2(C.m3, gamma);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const f2 Cp = fma2(c6, d[c], fma2(c5, Jp[c], fma2(c4, Sp[c], dj[c])));
                pa[9 + c] = fma2(q, Cp, pa[9 + c]);
            }
        }
    }
}

// fp32 partials -> the thread's fp64 accumulator slots in shared memory: acc[(2 c + lane) * kThreads + tid]
template <int NC>
__device__ __forceinline__ void flush(f2 (&pa)[NC], double *acc_mine) {
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        float a, b;
        upk(pa[c], a, b);
        acc_mine[(2 * c) * kThreads] += (double)a;
        acc_mine[(2 * c + 1) * kThreads] += (double)b;
        pa[c] = 0ull;
    }
}

template <int ORDER, int JL, int DIFF, bool MASK>
__device__ __forceinline__ void tile_compute(const IPair<ORDER, DIFF> &I, const uint4 *tq, int j0, int jl,
                                             const Consts &C, f2 (&pa)[3 * (ORDER / 2) + 1], double *acc_mine) {
    constexpr int JPT = kTileJ / JL;                 // j-particles per thread and tile
    constexpr int CH = JPT < 64 ? JPT : 64;          // fp32 partials are flushed to fp64 every <= 64 j (R10)
    constexpr int G0 = ORDER >= 6 ? 2 : 1;           // heads issued before their tails (measured: +2 % at orders 6, 8)
    constexpr int G = G0 < CH ? G0 : CH;
    constexpr int kUnroll = ORDER >= 6 ? 8 : 4;      // j-particles per unrolled group (measured per order)
#pragma unroll 1
    for (int jj0 = 0; jj0 < JPT; jj0 += CH) {
#pragma unroll(kUnroll / G)
        for (int u = 0; u < CH; u += G) {
            Stage S[G];
#pragma unroll
            for (int g = 0; g < G; ++g) {
                const int jt = (jj0 + u + g) * JL + jl;
                head<ORDER, DIFF, MASK>(I, tq, jt, j0 + jt, C, S[g]);
            }
#pragma unroll
            for (int g = 0; g < G; ++g) {
                const int jt = (jj0 + u + g) * JL + jl;
                tail<ORDER, DIFF>(I, tq, jt, C, S[g], pa);
            }
        }
        if (JPT >= 64) flush(pa, acc_mine);
    }
}

// One work item = (i-tile, j-split) of a force call.  `tile_run` counts the j-tiles this CTA has pushed through the
// ring since its mbarriers were initialised (stage and phase of tile g are g % STAGES and (g / STAGES) & 1), so a
// persistent CTA runs item after item on the same barriers.
// Epilogue of a work item with JL >= 128 j-lanes (few outputs, long sums; shared by force_item and fused_item, so every
// path sums in the same order): the fp64 accumulators of the JL j-lanes of each output are summed in a FIXED order by
// T = 4 (JL = 128) or 8 (JL = 256) adjacent threads -- thread t sums lanes l = t, t + T, ... in sequence, then a butterfly
// over the T threads -- pot is negated, and the result goes to the output arrays (S == 1) or to this split's row of the
// partials (S > 1).  (JL <= 64: one thread per output, lanes l = 0 .. JL-1 in sequence, written out at the call sites.)
template <int JL, int NC>
__device__ __forceinline__ void lane_sum_store(const ForceArgs &A, const double *acc_sm, int i_tile, int n_act,
                                               int splits, int split) {
    constexpr int IT = kThreads / JL;
    constexpr int NOUT = 2 * IT * NC;
    constexpr int T = JL >= 256 ? 8 : JL >= 128 ? 4 : 1;
    const int tid = threadIdx.x;
    for (int base = 0; base < NOUT * T; base += kThreads) {  // uniform trip count: the shuffles below see full warps
        const int q = base + tid;
        const int o = q / T, t = q % T;
        const int comp = o / (2 * IT), rem = o % (2 * IT);
        const int r = rem / IT, i_l = rem % IT;
        double sum = 0.0;
        if (o < NOUT) {
#pragma unroll 8
            for (int l = t; l < JL; l += T) sum += acc_sm[(2 * comp + r) * kThreads + l * IT + i_l];
        }
#pragma unroll
        for (int d = T / 2; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
        const int slot = i_tile * (2 * IT) + r * IT + i_l;
        if (o < NOUT && t == 0 && slot < n_act) {
            if (comp == NC - 1) sum = -sum;
            if (splits == 1) {
                if (comp == NC - 1) A.out[4][slot] = sum;
                else A.out[comp / 3][(size_t)slot * 3 + comp % 3] = sum;
            } else {
                A.partials[((size_t)split * NC + comp) * n_act + slot] = sum;
            }
        }
    }
}

template <int ORDER, int JL, int DIFF>
__device__ __forceinline__ void force_item(const ForceArgs &A, const int n_act, const int splits, const int i_tile,
                                           const int split, unsigned char *smem_raw, unsigned &tile_run) {
    typedef Geo<ORDER, DIFF> G;
    constexpr int NQ = G::NQ, NC = G::NC, STAGES = G::STAGES;
    constexpr int IT = kThreads / JL;    // threads per j-lane; the CTA owns 2 IT i-particles
    constexpr int JPT = kTileJ / JL;     // j-particles per thread and tile
    uint4 *tiles = reinterpret_cast<uint4 *>(smem_raw);
    double *acc_sm = reinterpret_cast<double *>(smem_raw + G::TILE_BYTES);
    const uint32_t bar0 = smem_u32(smem_raw + G::TILE_BYTES + G::ACC_BYTES);
    const int tid = threadIdx.x;
    const int il = JL == 1 ? tid : tid % IT, jl = JL == 1 ? 0 : tid / IT;  // JL = 1: uniform tile addresses (LDS [UR + imm])
    const int tile_lo = (int)((long long)A.n_tiles * split / splits);
    const int tile_hi = (int)((long long)A.n_tiles * (split + 1) / splits);
    const int ntile = tile_hi - tile_lo;
    const unsigned g0 = tile_run;

    auto issue = [&](int k) {  // k = tile number within this item's range
        const int s = (g0 + k) % STAGES;
        const uint32_t bar = bar0 + 8 * s;
        mbar_expect_tx(bar, G::STAGE_BYTES);
        const size_t off = (size_t)(tile_lo + k) * kTileJ;
#pragma unroll
        for (int p = 0; p < NQ; ++p)
            bulk_g2s(smem_u32(tiles + (s * NQ + p) * kTileJ), A.q[p] + off, kTileJ * 16, bar);
    };
    if (tid == 0) {  // every stage is free here: the previous item ended with a __syncthreads after its last tile
        for (int k = 0; k < STAGES - 1 && k < ntile; ++k) issue(k);
    }

    // ---- the thread's two i-particles into registers (gathered from the same j-store: R4) ----
    IPair<ORDER, DIFF> I;
    float nv[2][3], na[2][3], nj[2][3], xh[2][3], xl[2][3];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int slot = i_tile * (2 * IT) + r * IT + il;
        const bool valid = slot < n_act;
        const int gi = A.idx[valid ? slot : n_act - 1];
        I.idx[r] = valid ? gi : -1;
        const uint4 qa = __ldg(A.q[0] + gi), qb = __ldg(A.q[1] + gi), qc = __ldg(A.q[2] + gi);
        if (DIFF == 0) {
            I.x[r][0] = u2d(qa.x, qa.y);
            I.x[r][1] = u2d(qa.z, qa.w);
            I.x[r][2] = u2d(qb.x, qb.y);
        } else {
            xh[r][0] = -u2f(qa.x); xl[r][0] = -u2f(qa.y);
            xh[r][1] = -u2f(qa.z); xl[r][1] = -u2f(qa.w);
            xh[r][2] = -u2f(qb.x); xl[r][2] = -u2f(qb.y);
        }
        nv[r][0] = -u2f(qb.w);
        nv[r][1] = -u2f(qc.x);
        nv[r][2] = -u2f(qc.y);
        if (ORDER >= 6) {
            const uint4 qd = __ldg(A.q[3] + gi);
            na[r][0] = -u2f(qc.z);
            na[r][1] = -u2f(qc.w);
            na[r][2] = -u2f(qd.x);
            nj[r][0] = -u2f(qd.y);
            nj[r][1] = -u2f(qd.z);
            nj[r][2] = -u2f(qd.w);
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        I.nv[c] = pk(nv[0][c], nv[1][c]);
        if (ORDER >= 6) I.na[c] = pk(na[0][c], na[1][c]);
        if (ORDER >= 8) I.nj[c] = pk(nj[0][c], nj[1][c]);
        if (DIFF == 1) {
            I.nxh[c] = pk(xh[0][c], xh[1][c]);
            I.nxl[c] = pk(xl[0][c], xl[1][c]);
        }
    }
    Consts C;
    C.eps2 = pk(A.eps2, A.eps2);
    C.m3 = pk(-3.f, -3.f);
    C.three = pk(3.f, 3.f);
    C.m4 = pk(-4.f, -4.f);
    C.n = A.n;
    f2 pa[NC];
    double *acc_mine = acc_sm + tid;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        pa[c] = 0ull;
        acc_mine[(2 * c) * kThreads] = 0.0;
        acc_mine[(2 * c + 1) * kThreads] = 0.0;
    }

    // ---- main loop over this item's j-tiles ----
    int since = 0;
#pragma unroll 1
    for (int k = 0; k < ntile; ++k) {
        const unsigned g = g0 + k;
        const int s = g % STAGES;
        if (tid == 0 && k + STAGES - 1 < ntile) {  // tile g+STAGES-1 goes into the stage tile g-1 used
            if (g >= 1) mbar_wait(bar0 + 8 * (STAGES + (g - 1) % STAGES), (uint32_t)(((g - 1) / STAGES) & 1));
            issue(k + STAGES - 1);
        }
        mbar_wait(bar0 + 8 * s, (uint32_t)((g / STAGES) & 1));
        const uint4 *tq = tiles + s * NQ * kTileJ;
        const int j0 = (tile_lo + k) * kTileJ;
        const bool mine = (unsigned)(I.idx[0] - j0) < (unsigned)kTileJ || (unsigned)(I.idx[1] - j0) < (unsigned)kTileJ;
        if (__any_sync(0xffffffffu, mine) || j0 + kTileJ > A.n)
            tile_compute<ORDER, JL, DIFF, true>(I, tq, j0, jl, C, pa, acc_mine);
        else
            tile_compute<ORDER, JL, DIFF, false>(I, tq, j0, jl, C, pa, acc_mine);
        if (JPT < 64) {
            if (++since == 64 / JPT) {
                since = 0;
                flush(pa, acc_mine);
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (STAGES + s));
    }
    tile_run = g0 + ntile;
    flush(pa, acc_mine);
    __syncthreads();

    // ---- epilogue: fixed-order sum over the JL j-lanes, pot = - Sum m/r ----
    if constexpr (JL >= 128) {
        lane_sum_store<JL, NC>(A, acc_sm, i_tile, n_act, splits, split);
    } else {  // one thread per output, lanes in sequence (kept as written: the big-block kernels are tuned around it)
        for (int o = tid; o < 2 * IT * NC; o += kThreads) {
            const int comp = o / (2 * IT), rem = o % (2 * IT);
            const int r = rem / IT, i_l = rem % IT;
            double sum = 0.0;
#pragma unroll 8
            for (int l = 0; l < JL; ++l) sum += acc_sm[(2 * comp + r) * kThreads + l * IT + i_l];
            const int slot = i_tile * (2 * IT) + r * IT + i_l;
            if (slot < n_act) {
                if (comp == NC - 1) sum = -sum;
                if (splits == 1) {
                    if (comp == NC - 1) A.out[4][slot] = sum;
                    else A.out[comp / 3][(size_t)slot * 3 + comp % 3] = sum;
                } else {
                    A.partials[((size_t)split * NC + comp) * n_act + slot] = sum;
                }
            }
        }
    }
}

template <int ORDER, int DIFF>
__device__ __forceinline__ void init_ring(unsigned char *smem_raw) {
    typedef Geo<ORDER, DIFF> G;
    const uint32_t bar0 = smem_u32(smem_raw + G::TILE_BYTES + G::ACC_BYTES);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < G::STAGES; ++s) {
            mbar_init(bar0 + 8 * s, 1);                             // full[s]: the TMA transaction
            mbar_init(bar0 + 8 * (G::STAGES + s), kThreads / 32);   // empty[s]: one arrival per warp
        }
        mbar_fence_init();
    }
    __syncthreads();
}

// host-geometry form: grid = (i-tiles, j-splits), one work item per CTA
template <int ORDER, int JL, int DIFF>
__global__ void __launch_bounds__(kThreads, 1) k_force(const ForceArgs A) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    init_ring<ORDER, DIFF>(smem_raw);
    unsigned tile_run = 0;
    force_item<ORDER, JL, DIFF>(A, A.n_act, A.splits, blockIdx.x, blockIdx.y, smem_raw, tile_run);
}

// device-driven form: persistent CTAs (grid = SMs) walk the work items of the block whose size and geometry the
// selection kernel left in the control block; a stopped run is a no-op.
template <int ORDER>
__global__ void __launch_bounds__(kThreads, 1) k_force_dyn(const ForceArgs A) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const Ctl *ctl = A.ctl;
    if (ctl->stop) return;
    const int n_act = (int)ctl->n_act, jl = ctl->jl, splits = ctl->splits;
    const long long items = ctl->i_tiles * splits;
    init_ring<ORDER, 0>(smem_raw);
    unsigned tile_run = 0;
    for (long long w = blockIdx.x; w < items; w += gridDim.x) {
        const int i_tile = (int)(w % ctl->i_tiles), split = (int)(w / ctl->i_tiles);
        switch (jl) {
            case 1: force_item<ORDER, 1, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 2: force_item<ORDER, 2, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 4: force_item<ORDER, 4, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 8: force_item<ORDER, 8, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 16: force_item<ORDER, 16, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 32: force_item<ORDER, 32, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 64: force_item<ORDER, 64, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            case 128: force_item<ORDER, 128, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
            default: force_item<ORDER, 256, 0>(A, n_act, splits, i_tile, split, smem_raw, tile_run); break;
        }
        __syncthreads();  // the epilogue has read the accumulators before the next item clears them
    }
}

// K_reduce (a-3b): out = Sum over the S j-splits of partial[s], in a FIXED order that depends on S only (so the result is
// bit-reproducible and the same for every caller that uses the same S):
//   S <= 8 : one thread per output, s = 0 .. S-1 in sequence;
//   S  > 8 : one warp per output, lane l sums s = l, l + 32, ... in sequence, then a fixed butterfly over the lanes.
__device__ __forceinline__ void reduce_store(double s, long long o, int nc, int n_act, double *acc, double *jerk,
                                             double *snap, double *crk, double *pot) {
    const int comp = (int)(o / n_act), slot = (int)(o % n_act);
    if (comp == nc - 1) pot[slot] = s;
    else {
        double *dst = comp < 3 ? acc : comp < 6 ? jerk : comp < 9 ? snap : crk;
        dst[(size_t)slot * 3 + comp % 3] = s;
    }
}

__device__ __forceinline__ void reduce_body(const double *partials, int splits, int nc, int n_act, double *acc,
                                            double *jerk, double *snap, double *crk, double *pot, const long long tid,
                                            const long long nthr) {
    const long long tot = (long long)nc * n_act;
    if (splits <= 8) {
        for (long long o = tid; o < tot; o += nthr) {
            double v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = k < splits ? __ldcg(partials + (size_t)k * tot + o) : 0.0;
            double s = v[0];
#pragma unroll
            for (int k = 1; k < 8; ++k)
                if (k < splits) s += v[k];
            reduce_store(s, o, nc, n_act, acc, jerk, snap, crk, pot);
        }
    } else {
        const int lane = threadIdx.x & 31;
        for (long long o = tid >> 5; o < tot; o += nthr >> 5) {
            double s = 0.0;
#pragma unroll 4
            for (int k = lane; k < splits; k += 32) s += __ldcg(partials + (size_t)k * tot + o);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
            if (lane == 0) reduce_store(s, o, nc, n_act, acc, jerk, snap, crk, pot);
        }
    }
}

__global__ void __launch_bounds__(256) k_reduce(const double *partials, int splits, int nc, int n_act, double *acc,
                                                double *jerk, double *snap, double *crk, double *pot) {
    reduce_body(partials, splits, nc, n_act, acc, jerk, snap, crk, pot,
                (long long)blockIdx.x * blockDim.x + threadIdx.x, (long long)gridDim.x * blockDim.x);
}

// K_reduce of the device-driven step: S and n_act from the control block (a stopped run and an unsplit block are no-ops)
__global__ void __launch_bounds__(256) k_reduce_dyn(const Ctl *ctl, const double *partials, int nc, double *acc,
                                                    double *jerk, double *snap, double *crk, double *pot) {
    if (ctl->stop || ctl->splits == 1) return;
    reduce_body(partials, ctl->splits, nc, (int)ctl->n_act, acc, jerk, snap, crk, pot,
                (long long)blockIdx.x * blockDim.x + threadIdx.x, (long long)gridDim.x * blockDim.x);
}

// ---------------------------------------------------------------------------------------------------------
// N1 -- the fused small-block step ("real core-halo density structure ... block
// time-steps": most block steps of such a system move a handful of particles).  For a block that fits one i-tile
// (n_act <= 2 kThreads / JL, i.e. <= 1024) the j-store round trip is dropped: every persistent CTA owns one j-split,
// pulls the RAW fp64 Taylor state of its j-tiles into shared memory by TMA (two stages), its threads run the bit-exact
// Horner predictor (predict_particle, the code of K_pred; two threads per particle, each its own polynomials) and leave
// the packed quads of the tile in shared memory, then all 512 threads run the ordinary pair loop on it.  Every j is predicted exactly
// once in the whole grid; the i-particles are predicted by their own threads (the same arithmetic, so the self
// differences are still exactly zero, R4).  The last CTA to finish sums the j-split partials (K_reduce's fixed tree)
// and runs the corrector (correct_one, the code of K_corr) for the block: one launch instead of four.
// Results are bit-identical to K_pred + K_force + K_reduce + K_corr.
// ---------------------------------------------------------------------------------------------------------
struct FusedArgs {
    ForceArgs F;                    // idx, n, n_tiles, eps2, out, partials, ctl (q[] unused)
    const double *t, *m, *x, *v;    // raw state: the predictor's inputs
    const double *D[6];
    CorrArgs C;                     // corrector arguments (control-block mode)
    int tma_ok;                     // every raw array is 16-byte aligned: full tiles come in by TMA
};

template <int ORDER>
struct FGeo {
    static constexpr int K = ORDER / 2, NC = 3 * K + 1, ND = ORDER - 2;
    static constexpr int NQ = ORDER == 4 ? 3 : 4;
    static constexpr int RSTAGES = 2;
    static constexpr uint32_t RAW_DOUBLES = kTileJ * (2 + 3 * (2 + ND));  // t, m, x[3], v[3], D_k[3]
    static constexpr uint32_t RAW_BYTES = RAW_DOUBLES * 8;
    static constexpr size_t PRED_BYTES = (size_t)NQ * kTileJ * 16;
    static constexpr size_t ACC_BYTES = (size_t)2 * NC * kThreads * sizeof(double);
    static constexpr size_t SMEM = RSTAGES * (size_t)RAW_BYTES + PRED_BYTES + ACC_BYTES + 128;
};

template <int ORDER, int JL>
__device__ __forceinline__ void fused_item(const FusedArgs &A, const int n_act, const int splits, const int split,
                                           const double t_now, unsigned char *smem_raw, unsigned &tile_run) {
    typedef FGeo<ORDER> G;
    constexpr int NC = G::NC, ND = G::ND, RST = G::RSTAGES;
    constexpr int IT = kThreads / JL, JPT = kTileJ / JL;
    double *raw = reinterpret_cast<double *>(smem_raw);
    uint4 *pred = reinterpret_cast<uint4 *>(smem_raw + RST * (size_t)G::RAW_BYTES);
    double *acc_sm = reinterpret_cast<double *>(smem_raw + RST * (size_t)G::RAW_BYTES + G::PRED_BYTES);
    const uint32_t bar0 = smem_u32(smem_raw + RST * (size_t)G::RAW_BYTES + G::PRED_BYTES + G::ACC_BYTES);
    const int tid = threadIdx.x;
    const int il = JL == 1 ? tid : tid % IT, jl = JL == 1 ? 0 : tid / IT;
    const ForceArgs &F = A.F;
    const int tile_lo = (int)((long long)F.n_tiles * split / splits);
    const int tile_hi = (int)((long long)F.n_tiles * (split + 1) / splits);
    const int ntile = tile_hi - tile_lo;
    // a tile comes in by TMA iff it is full and the arrays are aligned; only the last tile of the array can be ragged
    auto by_tma = [&](int k) { return A.tma_ok && (tile_lo + k + 1) * kTileJ <= F.n; };
    auto issue = [&](int k, unsigned g) {  // tile k of this item is TMA tile number g of this CTA
        const int s = g % RST;
        const uint32_t bar = bar0 + 8 * s;
        mbar_expect_tx(bar, G::RAW_BYTES);
        const size_t b = (size_t)(tile_lo + k) * kTileJ;
        double *dst = raw + (size_t)s * G::RAW_DOUBLES;
        bulk_g2s(smem_u32(dst), A.t + b, kTileJ * 8, bar);
        bulk_g2s(smem_u32(dst + kTileJ), A.m + b, kTileJ * 8, bar);
        bulk_g2s(smem_u32(dst + 2 * kTileJ), A.x + 3 * b, kTileJ * 24, bar);
        bulk_g2s(smem_u32(dst + 5 * kTileJ), A.v + 3 * b, kTileJ * 24, bar);
#pragma unroll
        for (int d = 0; d < ND; ++d) bulk_g2s(smem_u32(dst + (8 + 3 * d) * kTileJ), A.D[d] + 3 * b, kTileJ * 24, bar);
    };
    unsigned g_issue = tile_run, g_use = tile_run;  // TMA tiles issued / consumed so far by this CTA
    if (tid == 0 && ntile > 0 && by_tma(0)) issue(0, g_issue);
    if (ntile > 0 && by_tma(0)) ++g_issue;

    // ---- the thread's two i-particles: predicted here from the raw state (same arithmetic as for the j: R4) ----
    IPair<ORDER, 0> I;
    float nv[2][3], na[2][3], nj[2][3];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int slot = r * IT + il;
        const bool valid = slot < n_act;
        const long long gi = F.idx[valid ? slot : n_act - 1];
        I.idx[r] = valid ? (int)gi : -1;
        const double *Dp[6];
#pragma unroll
        for (int d = 0; d < ND; ++d) Dp[d] = A.D[d] + 3 * gi;
        double xp[3];
        float vp[3], ap[3], jp[3];
        predict_particle<ORDER>(d_sub(t_now, A.t[gi]), A.x + 3 * gi, A.v + 3 * gi, Dp, xp, vp, ap, jp);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            I.x[r][c] = xp[c];
            nv[r][c] = -vp[c];
            na[r][c] = -ap[c];
            nj[r][c] = -jp[c];
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        I.nv[c] = pk(nv[0][c], nv[1][c]);
        if (ORDER >= 6) I.na[c] = pk(na[0][c], na[1][c]);
        if (ORDER >= 8) I.nj[c] = pk(nj[0][c], nj[1][c]);
    }
    Consts C;
    C.eps2 = pk(F.eps2, F.eps2);
    C.m3 = pk(-3.f, -3.f);
    C.three = pk(3.f, 3.f);
    C.m4 = pk(-4.f, -4.f);
    C.n = F.n;
    f2 pa[NC];
    double *acc_mine = acc_sm + tid;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        pa[c] = 0ull;
        acc_mine[(2 * c) * kThreads] = 0.0;
        acc_mine[(2 * c + 1) * kThreads] = 0.0;
    }

    int since = 0;
#pragma unroll 1
    for (int k = 0; k < ntile; ++k) {
        const int j0 = (tile_lo + k) * kTileJ;
        const bool tma_k = by_tma(k);
        // producer: the raw data of tile k+1 goes into the other stage, which tile k-1's predictors have released
        if (k + 1 < ntile && by_tma(k + 1)) {
            if (tid == 0) {
                if (g_issue >= RST)
                    mbar_wait(bar0 + 8 * (RST + (g_issue - RST) % RST), (uint32_t)(((g_issue - RST) / RST) & 1));
                issue(k + 1, g_issue);
            }
            ++g_issue;
        }
        // ---- predict phase: particle j0 + p is predicted by TWO threads (warps 0-7: x_p and j_p, warps 8-15: v_p, a_p
        //      and the mass), each writing its own bytes of the packed tile ----
        {
            const int p = tid & (kTileJ - 1), part = tid / kTileJ;
            const bool real = j0 + p < F.n;
            const double *st = nullptr;
            if (tma_k) {
                const int s = g_use % RST;
                mbar_wait(bar0 + 8 * s, (uint32_t)((g_use / RST) & 1));
                st = raw + (size_t)s * G::RAW_DOUBLES;
            }
            // the particle's raw state: shared memory (TMA tile) or global memory (ragged last tile / unaligned arrays)
            const double *tp = tma_k ? st + p : A.t + (j0 + p);
            const double *mp = tma_k ? st + kTileJ + p : A.m + (j0 + p);
            const double *xq = tma_k ? st + 2 * kTileJ + 3 * p : A.x + 3 * (size_t)(j0 + p);
            const double *vq = tma_k ? st + 5 * kTileJ + 3 * p : A.v + 3 * (size_t)(j0 + p);
            const double *Dp[6];
#pragma unroll
            for (int d = 0; d < ND; ++d) Dp[d] = tma_k ? st + (8 + 3 * d) * kTileJ + 3 * p : A.D[d] + 3 * (size_t)(j0 + p);
            double xp[3] = {kPadPos, kPadPos, kPadPos};
            float vp[3] = {0.f, 0.f, 0.f}, ap[3] = {0.f, 0.f, 0.f}, jp[3] = {0.f, 0.f, 0.f}, m32 = 0.f;
            unsigned *w = reinterpret_cast<unsigned *>(pred);  // word view: quad q of plane P at w[4 * (P * kTileJ + q)]
            if (part == 0) {
                if (real) predict_particle<ORDER, true, false, false, true>(d_sub(t_now, *tp), xq, vq, Dp, xp, vp, ap, jp);
                pred[p] = pack_dd(xp[0], xp[1]);
                *reinterpret_cast<double *>(w + 4 * (kTileJ + p)) = xp[2];
                if (ORDER >= 6) {
                    w[4 * (3 * kTileJ + p) + 1] = __float_as_uint(jp[0]);
                    w[4 * (3 * kTileJ + p) + 2] = __float_as_uint(jp[1]);
                    w[4 * (3 * kTileJ + p) + 3] = __float_as_uint(jp[2]);
                }
            } else {
                if (real) {
                    predict_particle<ORDER, false, true, true, false>(d_sub(t_now, *tp), xq, vq, Dp, xp, vp, ap, jp);
                    m32 = __double2float_rn(*mp);
                }
                w[4 * (kTileJ + p) + 2] = __float_as_uint(m32);
                w[4 * (kTileJ + p) + 3] = __float_as_uint(vp[0]);
                pred[2 * kTileJ + p] = pack_ffff(vp[1], vp[2], ap[0], ap[1]);
                if (ORDER >= 6) w[4 * (3 * kTileJ + p)] = __float_as_uint(ap[2]);
            }
            if (tma_k) {
                __syncwarp();
                if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (RST + (g_use % RST)));  // this warp is done with the raw stage
            }
        }
        if (tma_k) ++g_use;
        __syncthreads();
        // ---- pair loop on the predicted tile ----
        const bool mine = (unsigned)(I.idx[0] - j0) < (unsigned)kTileJ || (unsigned)(I.idx[1] - j0) < (unsigned)kTileJ;
        if (__any_sync(0xffffffffu, mine) || j0 + kTileJ > F.n)
            tile_compute<ORDER, JL, 0, true>(I, pred, j0, jl, C, pa, acc_mine);
        else
            tile_compute<ORDER, JL, 0, false>(I, pred, j0, jl, C, pa, acc_mine);
        if (JPT < 64) {
            if (++since == 64 / JPT) {
                since = 0;
                flush(pa, acc_mine);
            }
        }
        __syncthreads();  // the tile buffer is free for the next predict phase
    }
    tile_run = g_use;
    flush(pa, acc_mine);
    __syncthreads();

    // ---- epilogue: force_item's, for i-tile 0 ----
    if constexpr (JL >= 128) {
        lane_sum_store<JL, NC>(F, acc_sm, 0, n_act, splits, split);
    } else {
        for (int o = tid; o < 2 * IT * NC; o += kThreads) {
            const int comp = o / (2 * IT), rem = o % (2 * IT);
            const int r = rem / IT, i_l = rem % IT;
            double sum = 0.0;
#pragma unroll 8
            for (int l = 0; l < JL; ++l) sum += acc_sm[(2 * comp + r) * kThreads + l * IT + i_l];
            const int slot = r * IT + i_l;
            if (slot < n_act) {
                if (comp == NC - 1) sum = -sum;
                if (splits == 1) {
                    if (comp == NC - 1) F.out[4][slot] = sum;
                    else F.out[comp / 3][(size_t)slot * 3 + comp % 3] = sum;
                } else {
                    F.partials[((size_t)split * NC + comp) * n_act + slot] = sum;
                }
            }
        }
    }
}

template <int ORDER>
__global__ void __launch_bounds__(kThreads, 1) k_step_fused(const FusedArgs A) {
    typedef FGeo<ORDER> G;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ int s_last;
    Ctl *ctl = const_cast<Ctl *>(A.F.ctl);
    if (ctl->stop || ctl->i_tiles != 1) return;  // (the selection stops a fused run in front of a larger block)
    const int n_act = (int)ctl->n_act, jl = ctl->jl, splits = ctl->splits;
    const double t_now = ctl->t_next;
    const int tid = threadIdx.x;
    const uint32_t bar0 = smem_u32(smem_raw + G::RSTAGES * (size_t)G::RAW_BYTES + G::PRED_BYTES + G::ACC_BYTES);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < G::RSTAGES; ++s) {
            mbar_init(bar0 + 8 * s, 1);                              // full[s]: the TMA transaction
            mbar_init(bar0 + 8 * (G::RSTAGES + s), kThreads / 32);   // empty[s]: one arrival per warp
        }
        mbar_fence_init();
    }
    __syncthreads();
    unsigned tile_run = 0;
    for (int w = blockIdx.x; w < splits; w += gridDim.x) {
        switch (jl) {
            case 1: fused_item<ORDER, 1>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 2: fused_item<ORDER, 2>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 4: fused_item<ORDER, 4>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 8: fused_item<ORDER, 8>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 16: fused_item<ORDER, 16>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 32: fused_item<ORDER, 32>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 64: fused_item<ORDER, 64>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            case 128: fused_item<ORDER, 128>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
            default: fused_item<ORDER, 256>(A, n_act, splits, w, t_now, smem_raw, tile_run); break;
        }
        __syncthreads();
    }
    // ---- the last CTA to get here sums the split partials and corrects the block ----
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned ticket = atomicAdd(&ctl->tickets[0], 1u);
        s_last = ticket == gridDim.x - 1;
        if (s_last) ctl->tickets[0] = 0;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const ForceArgs &F = A.F;
    if (splits > 1) {
        reduce_body(F.partials, splits, G::NC, n_act, F.out[0], F.out[1], F.out[2], F.out[3], F.out[4], tid, kThreads);
        __threadfence_block();
        __syncthreads();
    }
    for (long long ia = tid; ia < n_act; ia += kThreads) correct_one<ORDER>(A.C, ia, t_now);
}

typedef void (*force_fn)(const ForceArgs);

template <int ORDER, int DIFF>
force_fn pick(int jl) {
    switch (jl) {
        case 1: return k_force<ORDER, 1, DIFF>;
        case 2: return k_force<ORDER, 2, DIFF>;
        case 4: return k_force<ORDER, 4, DIFF>;
        case 8: return k_force<ORDER, 8, DIFF>;
        case 16: return k_force<ORDER, 16, DIFF>;
        case 32: return k_force<ORDER, 32, DIFF>;
        case 64: return k_force<ORDER, 64, DIFF>;
        case 128: return k_force<ORDER, 128, DIFF>;
        default: return k_force<ORDER, 256, DIFF>;
    }
}

force_fn pick_fn(int order, int diff, int jl) {
    if (diff == 0) {
        if (order == 4) return pick<4, 0>(jl);
        if (order == 6) return pick<6, 0>(jl);
        return pick<8, 0>(jl);
    }
    if (order == 4) return pick<4, 1>(jl);
    if (order == 6) return pick<6, 1>(jl);
    return pick<8, 1>(jl);
}

force_fn pick_dyn(int order) {
    return order == 4 ? k_force_dyn<4> : order == 6 ? k_force_dyn<6> : k_force_dyn<8>;
}

size_t smem_for(int order, int diff) {
    if (diff == 0) return order == 4 ? Geo<4, 0>::SMEM : order == 6 ? Geo<6, 0>::SMEM : Geo<8, 0>::SMEM;
    return order == 4 ? Geo<4, 1>::SMEM : order == 6 ? Geo<6, 1>::SMEM : Geo<8, 1>::SMEM;
}

void fill_args(Ctx *c, ForceArgs &A, const int32_t *active_idx, float eps2, double *acc, double *jerk, double *snap,
               double *crackle, double *pot) {
    const uint4 *base = c->jstore;
    A.q[0] = base + (size_t)(c->diff_mode ? 4 : 0) * c->cap_pad;
    A.q[1] = base + (size_t)(c->diff_mode ? 5 : 1) * c->cap_pad;
    A.q[2] = base + (size_t)2 * c->cap_pad;
    A.q[3] = base + (size_t)3 * c->cap_pad;
    A.idx = active_idx;
    A.n = (int)c->n;
    A.n_act = 0;
    A.n_tiles = (int)(c->n_pad / kTileJ);
    A.splits = 1;
    A.eps2 = eps2;
    A.out[0] = acc; A.out[1] = jerk; A.out[2] = snap; A.out[3] = crackle; A.out[4] = pot;
    A.partials = c->partials;
    A.ctl = c->d_ctl;
}

}  // namespace

int force_static_init(Ctx *c) {
    const int orders[3] = {4, 6, 8};
    for (int o = 0; o < 3; ++o) {
        for (int diff = 0; diff < 2; ++diff)
            for (int j = 0; j < kNumLanes; ++j)
                NB_CUDA(c, cudaFuncSetAttribute((const void *)pick_fn(orders[o], diff, lane_variant(j)),
                                                cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)smem_for(orders[o], diff)));
        NB_CUDA(c, cudaFuncSetAttribute((const void *)pick_dyn(orders[o]), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem_for(orders[o], 0)));
    }
    NB_CUDA(c, cudaFuncSetAttribute((const void *)k_step_fused<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FGeo<4>::SMEM));
    NB_CUDA(c, cudaFuncSetAttribute((const void *)k_step_fused<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FGeo<6>::SMEM));
    NB_CUDA(c, cudaFuncSetAttribute((const void *)k_step_fused<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FGeo<8>::SMEM));
    return NBODY_OK;
}

int launch_step_fused(Ctx *c, int order, float eps2, const int32_t *active_idx, const double *t, const double *m,
                      const double *x, const double *v, const double *const a_derivs[8], const CorrArgs &corr,
                      double *acc, double *jerk, double *snap, double *crackle, double *pot, cudaStream_t st) {
    FusedArgs A;
    fill_args(c, A.F, active_idx, eps2, acc, jerk, snap, crackle, pot);
    A.t = t; A.m = m; A.x = x; A.v = v;
    bool aligned = ((uintptr_t)t | (uintptr_t)m | (uintptr_t)x | (uintptr_t)v) % 16 == 0;
    for (int k = 0; k < 6; ++k) {
        A.D[k] = k <= order - 3 ? a_derivs[k] : nullptr;
        if (A.D[k] && (uintptr_t)A.D[k] % 16 != 0) aligned = false;
    }
    A.C = corr;
    A.tma_ok = aligned ? 1 : 0;
    if (order == 4) k_step_fused<4><<<c->sm_count, kThreads, FGeo<4>::SMEM, st>>>(A);
    else if (order == 6) k_step_fused<6><<<c->sm_count, kThreads, FGeo<6>::SMEM, st>>>(A);
    else k_step_fused<8><<<c->sm_count, kThreads, FGeo<8>::SMEM, st>>>(A);
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int launch_force(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2, double *acc, double *jerk,
                 double *snap, double *crackle, double *pot, cudaStream_t st) {
    const int K = order / 2, NC = 3 * K + 1;
    ForceArgs A;
    fill_args(c, A, active_idx, eps2, acc, jerk, snap, crackle, pot);
    // geometry: j-lanes and j-splits from the size of the whole block (an i-sharded rank passes its slice as n_act
    // and the block size as the "geometry_n_act" option, so every rank sums in the order of the unsharded call)
    const int64_t n_geo = c->geometry_n_act ? c->geometry_n_act : n_act;
    if (n_act > n_geo) return NBODY_EINVAL;
    const ForceGeo g = force_geometry(n_geo, A.n_tiles, c->sm_count, c->force_lanes, c->force_split, c->partial_rows);
    const int64_t i_tiles = (n_act + g.i_per_cta - 1) / g.i_per_cta;
    if (g.splits > 1 && (int64_t)g.splits * n_act > c->partial_rows) return NBODY_EINVAL;  // forced split beyond the scratch
    A.n_act = (int)n_act;
    A.splits = g.splits;
    const dim3 grid((unsigned)i_tiles, (unsigned)g.splits);
    pick_fn(order, c->diff_mode, g.jl)<<<grid, kThreads, smem_for(order, c->diff_mode), st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    if (g.splits > 1) {
        const long long tot = (long long)NC * n_act;
        long long blocks = g.splits <= 8 ? (tot + 255) / 256 : (tot + 7) / 8;  // thread or warp per output
        if (blocks > 8LL * c->sm_count) blocks = 8LL * c->sm_count;
        k_reduce<<<(unsigned)blocks, 256, 0, st>>>(c->partials, g.splits, NC, (int)n_act, acc, jerk, snap, crackle, pot);
        c->launches += 1;
        NB_CUDA(c, cudaGetLastError());
    }
    c->last_r = 2;
    c->last_jl = g.jl;
    c->last_s = g.splits;
    c->last_ctas = i_tiles * g.splits;
    return NBODY_OK;
}

int launch_force_dyn(Ctx *c, const int32_t *active_idx, int order, float eps2, double *acc, double *jerk, double *snap,
                     double *crackle, double *pot, cudaStream_t st) {
    ForceArgs A;
    fill_args(c, A, active_idx, eps2, acc, jerk, snap, crackle, pot);
    pick_dyn(order)<<<c->sm_count, kThreads, smem_for(order, 0), st>>>(A);
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int launch_reduce_dyn(Ctx *c, int order, double *acc, double *jerk, double *snap, double *crackle, double *pot,
                      cudaStream_t st) {
    k_reduce_dyn<<<c->sm_count, 256, 0, st>>>(c->d_ctl, c->partials, 3 * (order / 2) + 1, acc, jerk, snap, crackle, pot);
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

// ---- allocation-free K_force: the j-split scratch in static device memory (include/nbody.h, nbody_force_static) ----
// For callers that may not allocate (and that do not want the launch to touch ctx-owned scratch): the [S][NC][n_act] fp64
// partials of a j-split launch go to this file-scope array instead of Ctx::partials.  Every GPU that loads libnbody.so
// holds the array (NBODY_FORCE_STATIC_SCRATCH_BYTES = 16 MiB) until the process exits.  All calls on a device share it,
// so two nbody_force_static launches that overlap on the GPU (different streams) race; launches on one stream do not.
// Nothing in it has to start at zero: K_force writes every entry (split, component, slot < n_act) that K_reduce of the
// same call reads, so the previous call's contents are never seen.
static __device__ __align__(256) double g_force_static_scratch[NBODY_FORCE_STATIC_SCRATCH_BYTES / sizeof(double)];

namespace {

constexpr int kMaxDevices = 64;
double *g_static_scratch_ptr[kMaxDevices] = {nullptr};  // device address of the array, per device (host code cannot
std::mutex g_static_scratch_mutex;                      // use the symbol's name: that is a host-side stand-in)

// Set-up, once per device, with that device current (the caller holds a DeviceGuard): resolve the device address.
int static_scratch_address(Ctx *c, double **out) {
    if (c->device < 0 || c->device >= kMaxDevices) return NBODY_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_scratch_mutex);
    if (!g_static_scratch_ptr[c->device]) {
        double *ptr = nullptr;
        NB_CUDA(c, cudaGetSymbolAddress((void **)&ptr, g_force_static_scratch));
        if (!ptr) return NBODY_ECUDA;
        g_static_scratch_ptr[c->device] = ptr;
    }
    *out = g_static_scratch_ptr[c->device];
    return NBODY_OK;
}

}  // namespace

// launch_force with the split partials in the static array: same kernels, same geometry rule (so the same bits as
// launch_force for the same options), no allocation, Ctx::partials untouched.  n_act == 0 only resolves the address.
int launch_force_static(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2, double *acc, double *jerk,
                        double *snap, double *crackle, double *pot, cudaStream_t st) {
    double *scratch = nullptr;
    const int rc = static_scratch_address(c, &scratch);
    if (rc != NBODY_OK) return rc;
    if (n_act == 0) return NBODY_OK;
    const int K = order / 2, NC = 3 * K + 1;
    ForceArgs A;
    fill_args(c, A, active_idx, eps2, acc, jerk, snap, crackle, pot);
    A.partials = scratch;
    const int64_t n_geo = c->geometry_n_act ? c->geometry_n_act : n_act;
    if (n_act > n_geo) return NBODY_EINVAL;
    const ForceGeo g = force_geometry(n_geo, A.n_tiles, c->sm_count, c->force_lanes, c->force_split, c->partial_rows);
    const int64_t i_tiles = (n_act + g.i_per_cta - 1) / g.i_per_cta;
    if (g.splits > 1 &&
        (uint64_t)g.splits * (uint64_t)NC * (uint64_t)n_act * sizeof(double) > (uint64_t)NBODY_FORCE_STATIC_SCRATCH_BYTES)
        return NBODY_ESCRATCH;  // beyond the static array: nothing was launched
    A.n_act = (int)n_act;
    A.splits = g.splits;
    const dim3 grid((unsigned)i_tiles, (unsigned)g.splits);
    pick_fn(order, c->diff_mode, g.jl)<<<grid, kThreads, smem_for(order, c->diff_mode), st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    if (g.splits > 1) {
        const long long tot = (long long)NC * n_act;
        long long blocks = g.splits <= 8 ? (tot + 255) / 256 : (tot + 7) / 8;  // thread or warp per output
        if (blocks > 8LL * c->sm_count) blocks = 8LL * c->sm_count;
        k_reduce<<<(unsigned)blocks, 256, 0, st>>>(scratch, g.splits, NC, (int)n_act, acc, jerk, snap, crackle, pot);
        c->launches += 1;
        NB_CUDA(c, cudaGetLastError());
    }
    c->last_r = 2;
    c->last_jl = g.jl;
    c->last_s = g.splits;
    c->last_ctas = i_tiles * g.splits;
    return NBODY_OK;
}

}  // namespace nbody
