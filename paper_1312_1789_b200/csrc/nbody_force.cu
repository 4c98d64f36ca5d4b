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
//     (cp.async.bulk + mbarrier) through a ring; every pair-loop read is an LDS.128 broadcast;
//   - d = fl32(x_j - x_i) with the subtraction in fp64 (DIFF 0: DADD + F2F per lane) or double-single (DIFF 1:
//     packed fp32 adds of hi and lo parts); MUFU.RSQ per lane; fp32 partial sums over <= 64 consecutive j, then
//     fp64 accumulators, which live in shared memory (one slot per thread and component) to free registers (R10);
//   - the self pair is excluded by index (R2), but the compare/select is only executed by warps whose i-indices
//     fall inside the current j-tile (warp-uniform branch), so the main loop is mask-free;
//   - a CTA is IT = 256/JL i-lanes x JL j-lanes (2 IT i-particles): JL = 1 for big blocks (every lane reads the
//     same j: smem broadcast), JL up to 256 for tiny blocks; the j-lanes are reduced through shared memory in
//     fixed order; gridDim.y = S j-splits; S > 1 writes fp64 partials [S][NC][n_act] that K_reduce sums in order.
#include <math.h>

#include "nbody_internal.h"

#ifndef NB_UNROLL
#define NB_UNROLL 4
#endif
#ifndef NB_NOBAR
#define NB_NOBAR 1  // 1 = no __syncthreads per tile: stages are released through per-stage "empty" mbarriers (+1.5 %)
#endif
#ifndef NB_MINB
#define NB_MINB 1  // resident CTAs per SM the register budget is sized for (1 x 512 threads measured 5 % faster than 2 x 256)
#endif

namespace nbody {
namespace {

constexpr int kUnroll = NB_UNROLL;  // j-particles per unrolled group of the pair loop

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
    int n_act;
    int n_tiles;
    int splits;
    float eps2;
    double *out[5];    // acc, jerk, snap, crackle, pot (used when splits == 1)
    double *partials;  // [splits][NC][n_act]           (used when splits > 1)
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
};

// One j against the thread's two i-particles; accumulates into pa[0 .. 3K] (pot as +m/r, negated at the end).
// tq = base of the staged tile (plane p at tq + p * kTileJ), jt = index inside the tile.
template <int ORDER, int DIFF, bool MASK>
__device__ __forceinline__ void pair2(const IPair<ORDER, DIFF> &I, const uint4 *tq, int jt, int jglob,
                                      const Consts &C, f2 *pa) {
    f2 d[3];
    const uint4 qa = tq[jt];           // Q0 = { x, y } (f64)           | Q4 = { xhi, xlo, yhi, ylo }
    const uint4 qb = tq[kTileJ + jt];  // Q1 = { z (f64), m, vx }       | Q5 = { zhi, zlo, m, vx }
    if (DIFF == 0) {
        const double xj = u2d(qa.x, qa.y), yj = u2d(qa.z, qa.w), zj = u2d(qb.x, qb.y);
        d[0] = pk(d2f(xj - I.x[0][0]), d2f(xj - I.x[1][0]));
        d[1] = pk(d2f(yj - I.x[0][1]), d2f(yj - I.x[1][1]));
        d[2] = pk(d2f(zj - I.x[0][2]), d2f(zj - I.x[1][2]));
    } else {
        d[0] = add2(add2(bc(qa.x), I.nxh[0]), add2(bc(qa.y), I.nxl[0]));
        d[1] = add2(add2(bc(qa.z), I.nxh[1]), add2(bc(qa.w), I.nxl[1]));
        d[2] = add2(add2(bc(qb.x), I.nxh[2]), add2(bc(qb.y), I.nxl[2]));
    }
    const f2 mj = bc(qb.z);
    const uint4 qc = tq[2 * kTileJ + jt];  // Q2 = { vy, vz, ax, ay }
    f2 dv[3], dj[3];
    dv[0] = add2(bc(qb.w), I.nv[0]);
    dv[1] = add2(bc(qc.x), I.nv[1]);
    dv[2] = add2(bc(qc.y), I.nv[2]);
    f2 da[3];
    f2 r2 = fma2(d[0], d[0], C.eps2);
    r2 = fma2(d[1], d[1], r2);
    r2 = fma2(d[2], d[2], r2);
    f2 rv = mul2(d[0], dv[0]);
    rv = fma2(d[1], dv[1], rv);
    rv = fma2(d[2], dv[2], rv);
    float r0, r1;
    upk(r2, r0, r1);
    r0 = frsqrt(r0);
    r1 = frsqrt(r1);
    if (MASK) {
        r0 = (jglob == I.idx[0]) ? 0.f : r0;
        r1 = (jglob == I.idx[1]) ? 0.f : r1;
    }
    const f2 rinv = pk(r0, r1);
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
            // gamma = g / s2 + alpha (3 beta - 4 alpha^2)
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
    constexpr int JPT = kTileJ / JL;
    constexpr int CH = JPT < 64 ? JPT : 64;
#pragma unroll 1
    for (int jj0 = 0; jj0 < JPT; jj0 += CH) {
#pragma unroll kUnroll
        for (int u = 0; u < CH; ++u) {
            const int jt = (jj0 + u) * JL + jl;
            pair2<ORDER, DIFF, MASK>(I, tq, jt, j0 + jt, C, pa);
        }
        if (JPT >= 64) flush(pa, acc_mine);
    }
}

template <int ORDER, int JL, int DIFF>
__global__ void __launch_bounds__(kThreads, NB_MINB) k_force(const ForceArgs A) {
    typedef Geo<ORDER, DIFF> G;
    constexpr int NQ = G::NQ, NC = G::NC, STAGES = G::STAGES;
    constexpr int IT = kThreads / JL;    // threads per j-lane; the CTA owns 2 IT i-particles
    constexpr int JPT = kTileJ / JL;     // j-particles per thread and tile
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint4 *tiles = reinterpret_cast<uint4 *>(smem_raw);
    double *acc_sm = reinterpret_cast<double *>(smem_raw + G::TILE_BYTES);
    const uint32_t bar0 = smem_u32(smem_raw + G::TILE_BYTES + G::ACC_BYTES);
    const int tid = threadIdx.x;
    const int il = tid % IT, jl = tid / IT;
    const int tile_lo = (int)((long long)A.n_tiles * blockIdx.y / A.splits);
    const int tile_hi = (int)((long long)A.n_tiles * (blockIdx.y + 1) / A.splits);
    const int ntile = tile_hi - tile_lo;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar0 + 8 * s, 1);                          // full[s]: the TMA transaction
            mbar_init(bar0 + 8 * (STAGES + s), kThreads / 32);   // empty[s]: one arrival per warp
        }
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int k) {  // k = tile number within this CTA's range
        const int s = k % STAGES;
        const uint32_t bar = bar0 + 8 * s;
        mbar_expect_tx(bar, G::STAGE_BYTES);
        const size_t off = (size_t)(tile_lo + k) * kTileJ;
#pragma unroll
        for (int p = 0; p < NQ; ++p)
            bulk_g2s(smem_u32(tiles + (s * NQ + p) * kTileJ), A.q[p] + off, kTileJ * 16, bar);
    };
    if (tid == 0) {
        for (int k = 0; k < STAGES - 1 && k < ntile; ++k) issue(k);
    }

    // ---- the thread's two i-particles into registers (gathered from the same j-store: R4) ----
    IPair<ORDER, DIFF> I;
    float nv[2][3], na[2][3], nj[2][3], xh[2][3], xl[2][3];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int slot = blockIdx.x * (2 * IT) + r * IT + il;
        const bool valid = slot < A.n_act;
        const int gi = A.idx[valid ? slot : A.n_act - 1];
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
    f2 pa[NC];
    double *acc_mine = acc_sm + tid;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        pa[c] = 0ull;
        acc_mine[(2 * c) * kThreads] = 0.0;
        acc_mine[(2 * c + 1) * kThreads] = 0.0;
    }

    // ---- main loop over this CTA's j-tiles ----
    int since = 0;
#pragma unroll 1
    for (int k = 0; k < ntile; ++k) {
        const int s = k % STAGES;
#if NB_NOBAR
        if (tid == 0 && k + STAGES - 1 < ntile) {  // tile k+STAGES-1 goes into the stage tile k-1 used
            if (k >= 1) mbar_wait(bar0 + 8 * (STAGES + (k - 1) % STAGES), (uint32_t)(((k - 1) / STAGES) & 1));
            issue(k + STAGES - 1);
        }
#else
        __syncthreads();  // every warp is done with tile k-1, whose stage is refilled now
        if (tid == 0 && k + STAGES - 1 < ntile) issue(k + STAGES - 1);
#endif
        mbar_wait(bar0 + 8 * s, (uint32_t)((k / STAGES) & 1));
        const uint4 *tq = tiles + s * NQ * kTileJ;
        const int j0 = (tile_lo + k) * kTileJ;
        const bool mine = (unsigned)(I.idx[0] - j0) < (unsigned)kTileJ || (unsigned)(I.idx[1] - j0) < (unsigned)kTileJ;
        if (__any_sync(0xffffffffu, mine))
            tile_compute<ORDER, JL, DIFF, true>(I, tq, j0, jl, C, pa, acc_mine);
        else
            tile_compute<ORDER, JL, DIFF, false>(I, tq, j0, jl, C, pa, acc_mine);
        if (JPT < 64) {
            if (++since == 64 / JPT) {
                since = 0;
                flush(pa, acc_mine);
            }
        }
#if NB_NOBAR
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(bar0 + 8 * (STAGES + s));
#endif
    }
    flush(pa, acc_mine);
    __syncthreads();

    // ---- epilogue: fixed-order sum over the JL j-lanes, pot = - Sum m/r ----
    for (int o = tid; o < 2 * IT * NC; o += kThreads) {
        const int comp = o / (2 * IT), rem = o % (2 * IT);
        const int r = rem / IT, i_l = rem % IT;
        double sum = 0.0;
#pragma unroll 1
        for (int l = 0; l < JL; ++l) sum += acc_sm[(2 * comp + r) * kThreads + l * IT + i_l];
        const int slot = blockIdx.x * (2 * IT) + r * IT + i_l;
        if (slot < A.n_act) {
            if (comp == NC - 1) sum = -sum;
            if (A.splits == 1) {
                if (comp == NC - 1) A.out[4][slot] = sum;
                else A.out[comp / 3][(size_t)slot * 3 + comp % 3] = sum;
            } else {
                A.partials[((size_t)blockIdx.y * NC + comp) * A.n_act + slot] = sum;
            }
        }
    }
}

// K_reduce (a-3b): out = Sum_{s = 0 .. S-1} partial[s] in that order.
__global__ void __launch_bounds__(256) k_reduce(const double *partials, int splits, int nc, int n_act, double *acc,
                                                double *jerk, double *snap, double *crk, double *pot) {
    const long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long tot = (long long)nc * n_act;
    if (o >= tot) return;
    double s = 0.0;
    for (int k = 0; k < splits; ++k) s += partials[(size_t)k * tot + o];
    const int comp = (int)(o / n_act), slot = (int)(o % n_act);
    if (comp == nc - 1) pot[slot] = s;
    else {
        double *dst = comp < 3 ? acc : comp < 6 ? jerk : comp < 9 ? snap : crk;
        dst[(size_t)slot * 3 + comp % 3] = s;
    }
}

typedef void (*force_fn)(const ForceArgs);

template <int ORDER, int DIFF>
force_fn pick(int jl) {
    switch (jl) {
        case 1: return k_force<ORDER, 1, DIFF>;
        case 2: return k_force<ORDER, 2, DIFF>;
        case 4: return k_force<ORDER, 4, DIFF>;
        case 8: return k_force<ORDER, 8, DIFF>;
        case 32: return k_force<ORDER, 32, DIFF>;
        default: return k_force<ORDER, 128, DIFF>;
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

size_t smem_for(int order, int diff) {
    if (diff == 0) return order == 4 ? Geo<4, 0>::SMEM : order == 6 ? Geo<6, 0>::SMEM : Geo<8, 0>::SMEM;
    return order == 4 ? Geo<4, 1>::SMEM : order == 6 ? Geo<6, 1>::SMEM : Geo<8, 1>::SMEM;
}

constexpr int kNumLanes = 6;
const int kLanes[kNumLanes] = {1, 2, 4, 8, 32, 128};

}  // namespace

int force_static_init(Ctx *c) {
    const int orders[3] = {4, 6, 8};
    for (int diff = 0; diff < 2; ++diff)
        for (int o = 0; o < 3; ++o)
            for (int j = 0; j < kNumLanes; ++j)
                NB_CUDA(c, cudaFuncSetAttribute((const void *)pick_fn(orders[o], diff, kLanes[j]),
                                                cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)smem_for(orders[o], diff)));
    return NBODY_OK;
}

int launch_force(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2, double *acc, double *jerk,
                 double *snap, double *crackle, double *pot, cudaStream_t st) {
    const int K = order / 2, NC = 3 * K + 1;
    const int n_tiles = (int)(c->n_pad / kTileJ);
    // geometry: j-lanes (a CTA owns 2 * 256 / JL i-particles), i-tiles, j-splits
    int jl;
    if (c->force_lanes) jl = c->force_lanes;
    else {  // the most j-lanes whose CTA still holds all active particles (2 * kThreads / JL i-slots)
        jl = 1;
        for (int k = kNumLanes - 1; k >= 1; --k)
            if ((int64_t)2 * kThreads / kLanes[k] >= n_act) { jl = kLanes[k]; break; }
    }
    const int i_per_cta = 2 * (kThreads / jl);
    const int64_t i_tiles = (n_act + i_per_cta - 1) / i_per_cta;
    // j-splits: the chip holds `slots` CTAs at once (2 per SM); a launch of i_tiles * S CTAs takes
    // ceil(i_tiles * S / slots) waves of (n_tiles / S + fixed per-CTA cost) tile-times.  Pick the S that minimises it:
    // small blocks get S ~ slots / i_tiles (fill the chip), mid-size blocks get a CTA count that is close to a
    // multiple of `slots` (no half-empty last wave), big blocks (>= 8 waves) run unsplit.
    const int64_t slots = NB_MINB * (int64_t)c->sm_count;
    int64_t S = 1;
    if (c->force_split) {
        S = c->force_split;
    } else if (i_tiles < 8 * slots) {
        const double fixed = 3.0;  // prologue + epilogue + reduce, in tile-times
        double best = 1e300, cost1 = 0.0;
        const int64_t s_max = n_tiles < 4 * slots ? n_tiles : 4 * slots;
        for (int64_t s = 1; s <= s_max; ++s) {
            const int64_t waves = (i_tiles * s + slots - 1) / slots;
            const double cost = (double)waves * ((double)((n_tiles + s - 1) / s) + fixed);
            if (s == 1) cost1 = cost;
            if (cost < best * (1.0 - 1e-9)) {
                best = cost;
                S = s;
            }
        }
        if (best > 0.97 * cost1) S = 1;  // a split costs S x NC x n_act doubles of scratch: only for a real gain
    }
    if (S > n_tiles) S = n_tiles;
    if (S > 65535) S = 65535;
    if (S < 1) S = 1;
    if (S > 1) {
        const size_t need = sizeof(double) * (size_t)S * NC * (size_t)n_act;
        if (need > c->partials_bytes) {
            NB_CUDA(c, cudaStreamSynchronize(st));
            cudaFree(c->partials);
            c->partials = nullptr;
            c->partials_bytes = 0;
            NB_CUDA(c, cudaMalloc(&c->partials, need));
            c->partials_bytes = need;
        }
    }
    ForceArgs A;
    const uint4 *base = c->jstore;
    A.q[0] = base + (size_t)(c->diff_mode ? 4 : 0) * c->cap_pad;
    A.q[1] = base + (size_t)(c->diff_mode ? 5 : 1) * c->cap_pad;
    A.q[2] = base + (size_t)2 * c->cap_pad;
    A.q[3] = base + (size_t)3 * c->cap_pad;
    A.idx = active_idx;
    A.n_act = (int)n_act;
    A.n_tiles = n_tiles;
    A.splits = (int)S;
    A.eps2 = eps2;
    A.out[0] = acc; A.out[1] = jerk; A.out[2] = snap; A.out[3] = crackle; A.out[4] = pot;
    A.partials = c->partials;
    const dim3 grid((unsigned)i_tiles, (unsigned)S);
    pick_fn(order, c->diff_mode, jl)<<<grid, kThreads, smem_for(order, c->diff_mode), st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    if (S > 1) {
        const long long tot = (long long)NC * n_act;
        k_reduce<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(c->partials, (int)S, NC, (int)n_act, acc, jerk, snap,
                                                                 crackle, pot);
        c->launches += 1;
        NB_CUDA(c, cudaGetLastError());
    }
    c->last_r = 2;
    c->last_jl = jl;
    c->last_s = (int)S;
    c->last_ctas = i_tiles * S;
    return NBODY_OK;
}

}  // namespace nbody
