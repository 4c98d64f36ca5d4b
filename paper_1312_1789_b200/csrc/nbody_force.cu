// libnbody.so, translation unit 2: K_force (a-3), K_reduce (a-3b) and the peak micro-probes.
//
// K_force computes, for each active i, the sums of DESIGN.md R1 (= SURVEY.md c-1; the paper prints no formula,
// PAPER.md:15/:43 name the scheme, PAPER.md:31 the mixed precision) over the packed j-store:
//   - i-particles live in registers (R per thread), j-tiles of kTileJ particles are staged plane by plane into
//     shared memory by 1-D TMA bulk copies (cp.async.bulk + mbarrier) through a kStages-deep ring;
//   - d = fl32(x_j - x_i) with the subtraction in fp64 (DIFF 0) or double-single (DIFF 1); all pair arithmetic
//     fp32 with MUFU.RSQ; fp32 partial sums over <= 64 consecutive j, then fp64 accumulators (R10);
//   - the self pair is excluded by index (R2), but the compare/select is only executed by warps whose
//     i-indices fall inside the current j-tile (warp-uniform branch), so the main loop is mask-free;
//   - a CTA is IT = 256/JL i-lanes x JL j-lanes: JL = 1 for big blocks (every lane reads the same j: smem
//     broadcast), JL up to 256 for tiny blocks (lanes share one i and stride over j), reduced through smem;
//   - gridDim.y = S j-splits; S > 1 writes fp64 partials [S][NC][n_act] that K_reduce sums in fixed order.
#include <math.h>

#include "nbody_internal.h"

namespace nbody {
namespace {

// ---- TMA / mbarrier primitives (PTX) -------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
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
struct IPart {  // one i-particle in registers
    double x[3];
    float xh[3], xl[3];
    float v[3], a[3], j[3];
    int idx;
};

// One pair: accumulates into pa[0 .. 3K] (pot as +m/r, negated at the end).
template <int ORDER, int DIFF, bool MASK>
__device__ __forceinline__ void pair(const IPart<ORDER, DIFF> &I, const uint4 &qa, const uint4 &qb, const uint4 &qc,
                                     const uint4 &qd, int jglob, float eps2, float *pa) {
    float d[3], dv[3], da[3], dj[3];
    float mj;
    if (DIFF == 0) {
        d[0] = d2f(u2d(qa.x, qa.y) - I.x[0]);
        d[1] = d2f(u2d(qa.z, qa.w) - I.x[1]);
        d[2] = d2f(u2d(qb.x, qb.y) - I.x[2]);
    } else {
        d[0] = (u2f(qa.x) - I.xh[0]) + (u2f(qa.y) - I.xl[0]);
        d[1] = (u2f(qa.z) - I.xh[1]) + (u2f(qa.w) - I.xl[1]);
        d[2] = (u2f(qb.x) - I.xh[2]) + (u2f(qb.y) - I.xl[2]);
    }
    mj = u2f(qb.z);
    dv[0] = u2f(qb.w) - I.v[0];
    dv[1] = u2f(qc.x) - I.v[1];
    dv[2] = u2f(qc.y) - I.v[2];
    float r2 = fmaf(d[0], d[0], eps2);
    r2 = fmaf(d[1], d[1], r2);
    r2 = fmaf(d[2], d[2], r2);
    float rv = d[0] * dv[0];
    rv = fmaf(d[1], dv[1], rv);
    rv = fmaf(d[2], dv[2], rv);
    float rinv = frsqrt(r2);
    if (MASK) rinv = (jglob == I.idx) ? 0.f : rinv;
    const float rinv2 = rinv * rinv;
    const float mrinv = mj * rinv;
    const float q = mrinv * rinv2;
    const float alpha = rv * rinv2;
    constexpr int K = ORDER / 2;
    pa[3 * K] += mrinv;
    const float c1 = -3.f * alpha;
    float Jp[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        Jp[c] = fmaf(c1, d[c], dv[c]);
        pa[c] = fmaf(q, d[c], pa[c]);
        pa[3 + c] = fmaf(q, Jp[c], pa[3 + c]);
    }
    if (ORDER >= 6) {
        da[0] = u2f(qc.z) - I.a[0];
        da[1] = u2f(qc.w) - I.a[1];
        da[2] = u2f(qd.x) - I.a[2];
        float w = dv[0] * dv[0];
        w = fmaf(dv[1], dv[1], w);
        w = fmaf(dv[2], dv[2], w);
        w = fmaf(d[0], da[0], w);
        w = fmaf(d[1], da[1], w);
        w = fmaf(d[2], da[2], w);
        const float beta = fmaf(alpha, alpha, w * rinv2);
        const float c2 = c1 + c1;
        const float c3 = -3.f * beta;
        float Sp[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Sp[c] = fmaf(c3, d[c], fmaf(c2, Jp[c], da[c]));
            pa[6 + c] = fmaf(q, Sp[c], pa[6 + c]);
        }
        if (ORDER >= 8) {
            dj[0] = u2f(qd.y) - I.j[0];
            dj[1] = u2f(qd.z) - I.j[1];
            dj[2] = u2f(qd.w) - I.j[2];
            float va = dv[0] * da[0];
            va = fmaf(dv[1], da[1], va);
            va = fmaf(dv[2], da[2], va);
            float g = 3.f * va;
            g = fmaf(d[0], dj[0], g);
            g = fmaf(d[1], dj[1], g);
            g = fmaf(d[2], dj[2], g);
            // gamma = g / s2 + alpha (3 beta - 4 alpha^2)
            const float t = fmaf(-4.f * alpha, alpha, 3.f * beta);
            const float gamma = fmaf(alpha, t, g * rinv2);
            const float c4 = 3.f * c1;   // -9 alpha
            const float c5 = 3.f * c3;   // -9 beta
            const float c6 = -3.f * gamma;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float Cp = fmaf(c6, d[c], fmaf(c5, Jp[c], fmaf(c4, Sp[c], dj[c])));
                pa[9 + c] = fmaf(q, Cp, pa[9 + c]);
            }
        }
    }
}

template <int ORDER, int R, int JL, int DIFF, bool MASK>
__device__ __forceinline__ void tile_compute(const IPart<ORDER, DIFF> (&I)[R], const uint4 *tq, int j0, int jl,
                                             float eps2, float (&pa)[R][3 * (ORDER / 2) + 1],
                                             double (&acc)[R][3 * (ORDER / 2) + 1]) {
    constexpr int NQ = ORDER == 4 ? 3 : 4;
    constexpr int NC = 3 * (ORDER / 2) + 1;
    constexpr int JPT = kTileJ / JL;
    constexpr int CH = JPT < 64 ? JPT : 64;
#pragma unroll 1
    for (int jj0 = 0; jj0 < JPT; jj0 += CH) {
#pragma unroll 4
        for (int u = 0; u < CH; ++u) {
            const int jt = (jj0 + u) * JL + jl;
            const uint4 qa = tq[jt];
            const uint4 qb = tq[kTileJ + jt];
            const uint4 qc = tq[2 * kTileJ + jt];
            uint4 qd = make_uint4(0, 0, 0, 0);
            if (NQ == 4) qd = tq[3 * kTileJ + jt];
#pragma unroll
            for (int r = 0; r < R; ++r) pair<ORDER, DIFF, MASK>(I[r], qa, qb, qc, qd, j0 + jt, eps2, pa[r]);
        }
        if (JPT >= 64) {
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    acc[r][c] += (double)pa[r][c];
                    pa[r][c] = 0.f;
                }
        }
    }
}

template <int ORDER, int R, int JL, int DIFF>
__global__ void __launch_bounds__(kThreads, 2) k_force(const ForceArgs A) {
    constexpr int NQ = ORDER == 4 ? 3 : 4;
    constexpr int K = ORDER / 2;
    constexpr int NC = 3 * K + 1;
    constexpr int IT = kThreads / JL;
    constexpr int JPT = kTileJ / JL;
    constexpr uint32_t kStageBytes = NQ * kTileJ * 16;
    static_assert(JL == 1 || R == 1, "j-lanes only with one i per thread");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint4 *tiles = reinterpret_cast<uint4 *>(smem_raw);
    const uint32_t bar0 = smem_u32(smem_raw + kStages * kStageBytes);
    const int tid = threadIdx.x;
    const int il = tid % IT, jl = tid / IT;
    const int tile_lo = (int)((long long)A.n_tiles * blockIdx.y / A.splits);
    const int tile_hi = (int)((long long)A.n_tiles * (blockIdx.y + 1) / A.splits);
    const int ntile = tile_hi - tile_lo;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int k) {  // k = tile number within this CTA's range
        const int s = k % kStages;
        const uint32_t bar = bar0 + 8 * s;
        mbar_expect_tx(bar, kStageBytes);
        const size_t off = (size_t)(tile_lo + k) * kTileJ;
#pragma unroll
        for (int p = 0; p < NQ; ++p)
            bulk_g2s(smem_u32(tiles + (s * NQ + p) * kTileJ), A.q[p] + off, kTileJ * 16, bar);
    };
    if (tid == 0) {
        for (int k = 0; k < kStages - 1 && k < ntile; ++k) issue(k);
    }

    // ---- i-particles into registers ----
    IPart<ORDER, DIFF> I[R];
    float pa[R][NC];
    double acc[R][NC];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int slot = blockIdx.x * (IT * R) + r * IT + il;
        const bool valid = slot < A.n_act;
        const int gi = A.idx[valid ? slot : A.n_act - 1];
        I[r].idx = valid ? gi : -1;
        const uint4 qa = __ldg(A.q[0] + gi), qb = __ldg(A.q[1] + gi), qc = __ldg(A.q[2] + gi);
        if (DIFF == 0) {
            I[r].x[0] = u2d(qa.x, qa.y);
            I[r].x[1] = u2d(qa.z, qa.w);
            I[r].x[2] = u2d(qb.x, qb.y);
        } else {
            I[r].xh[0] = u2f(qa.x); I[r].xl[0] = u2f(qa.y);
            I[r].xh[1] = u2f(qa.z); I[r].xl[1] = u2f(qa.w);
            I[r].xh[2] = u2f(qb.x); I[r].xl[2] = u2f(qb.y);
        }
        I[r].v[0] = u2f(qb.w);
        I[r].v[1] = u2f(qc.x);
        I[r].v[2] = u2f(qc.y);
        if (ORDER >= 6) {
            const uint4 qd = __ldg(A.q[3] + gi);
            I[r].a[0] = u2f(qc.z);
            I[r].a[1] = u2f(qc.w);
            I[r].a[2] = u2f(qd.x);
            I[r].j[0] = u2f(qd.y);
            I[r].j[1] = u2f(qd.z);
            I[r].j[2] = u2f(qd.w);
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            pa[r][c] = 0.f;
            acc[r][c] = 0.0;
        }
    }

    // ---- main loop over this CTA's j-tiles ----
    int since = 0;
#pragma unroll 1
    for (int k = 0; k < ntile; ++k) {
        const int s = k % kStages;
        __syncthreads();  // every warp is done with tile k-1, whose stage is refilled now
        if (tid == 0 && k + kStages - 1 < ntile) issue(k + kStages - 1);
        mbar_wait(bar0 + 8 * s, (uint32_t)((k / kStages) & 1));
        const uint4 *tq = tiles + s * NQ * kTileJ;
        const int j0 = (tile_lo + k) * kTileJ;
        bool mine = false;
#pragma unroll
        for (int r = 0; r < R; ++r) mine |= (unsigned)(I[r].idx - j0) < (unsigned)kTileJ;
        if (__any_sync(0xffffffffu, mine))
            tile_compute<ORDER, R, JL, DIFF, true>(I, tq, j0, jl, A.eps2, pa, acc);
        else
            tile_compute<ORDER, R, JL, DIFF, false>(I, tq, j0, jl, A.eps2, pa, acc);
        if (JPT < 64) {
            if (++since == 64 / JPT) {
                since = 0;
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        acc[r][c] += (double)pa[r][c];
                        pa[r][c] = 0.f;
                    }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[r][c] += (double)pa[r][c];
        acc[r][NC - 1] = -acc[r][NC - 1];  // pot = - Sum m/r
    }

    // ---- epilogue ----
    auto store = [&](int comp, int slot, double val) {
        if (A.splits == 1) {
            if (comp == NC - 1) A.out[4][slot] = val;
            else A.out[comp / 3][(size_t)slot * 3 + comp % 3] = val;
        } else {
            A.partials[((size_t)blockIdx.y * NC + comp) * A.n_act + slot] = val;
        }
    };
    if (JL == 1) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int slot = blockIdx.x * (IT * R) + r * IT + il;
            if (slot < A.n_act) {
#pragma unroll
                for (int c = 0; c < NC; ++c) store(c, slot, acc[r][c]);
            }
        }
    } else {
        __syncthreads();  // tiles are dead: reuse them as the reduction buffer red[jl][comp][il]
        double *red = reinterpret_cast<double *>(smem_raw);
#pragma unroll
        for (int c = 0; c < NC; ++c) red[(jl * NC + c) * IT + il] = acc[0][c];
        __syncthreads();
        for (int o = tid; o < IT * NC; o += kThreads) {
            const int comp = o / IT, i_l = o % IT;
            double sum = 0.0;
            for (int l = 0; l < JL; ++l) sum += red[(l * NC + comp) * IT + i_l];
            const int slot = blockIdx.x * IT + i_l;
            if (slot < A.n_act) store(comp, slot, sum);
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

template <int ORDER>
constexpr size_t force_smem() {
    return (size_t)kStages * (ORDER == 4 ? 3 : 4) * kTileJ * 16 + 8 * kStages + 64;
}

typedef void (*force_fn)(const ForceArgs);

template <int ORDER, int DIFF>
force_fn pick(int r, int jl) {
    if (r == 2) return k_force<ORDER, 2, 1, DIFF>;
    switch (jl) {
        case 1: return k_force<ORDER, 1, 1, DIFF>;
        case 4: return k_force<ORDER, 1, 4, DIFF>;
        case 16: return k_force<ORDER, 1, 16, DIFF>;
        case 64: return k_force<ORDER, 1, 64, DIFF>;
        default: return k_force<ORDER, 1, 256, DIFF>;
    }
}

force_fn pick_fn(int order, int diff, int r, int jl) {
    if (diff == 0) {
        if (order == 4) return pick<4, 0>(r, jl);
        if (order == 6) return pick<6, 0>(r, jl);
        return pick<8, 0>(r, jl);
    }
    if (order == 4) return pick<4, 1>(r, jl);
    if (order == 6) return pick<6, 1>(r, jl);
    return pick<8, 1>(r, jl);
}

size_t smem_for(int order) { return order == 4 ? force_smem<4>() : force_smem<6>(); }

}  // namespace

int force_static_init(Ctx *c) {
    const int orders[3] = {4, 6, 8};
    const int jls[5] = {1, 4, 16, 64, 256};
    for (int diff = 0; diff < 2; ++diff)
        for (int o = 0; o < 3; ++o) {
            NB_CUDA(c, cudaFuncSetAttribute((const void *)pick_fn(orders[o], diff, 2, 1),
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_for(orders[o])));
            for (int j = 0; j < 5; ++j)
                NB_CUDA(c, cudaFuncSetAttribute((const void *)pick_fn(orders[o], diff, 1, jls[j]),
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_for(orders[o])));
        }
    return NBODY_OK;
}

int launch_force(Ctx *c, const int32_t *active_idx, int64_t n_act, int order, float eps2, double *acc, double *jerk,
                 double *snap, double *crackle, double *pot, cudaStream_t st) {
    const int K = order / 2, NC = 3 * K + 1;
    const int n_tiles = (int)(c->n_pad / kTileJ);
    // geometry: i per thread, j-lanes, i-tiles, j-splits
    int r, jl;
    if (c->force_lanes) {
        r = 1;
        jl = c->force_lanes;
    } else if (n_act > 256) {
        r = 2;
        jl = 1;
    } else {
        r = 1;
        jl = n_act > 64 ? 1 : n_act > 16 ? 4 : n_act > 4 ? 16 : n_act > 1 ? 64 : 256;
    }
    const int i_per_cta = (kThreads / jl) * r;
    const int64_t i_tiles = (n_act + i_per_cta - 1) / i_per_cta;
    const int64_t target = 2 * (int64_t)c->sm_count;  // 2 resident CTAs per SM
    int64_t S = c->force_split ? c->force_split : (i_tiles >= target ? 1 : (target + i_tiles - 1) / i_tiles);
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
    pick_fn(order, c->diff_mode, r, jl)<<<grid, kThreads, smem_for(order), st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    if (S > 1) {
        const long long tot = (long long)NC * n_act;
        k_reduce<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(c->partials, (int)S, NC, (int)n_act, acc, jerk, snap,
                                                                 crackle, pot);
        c->launches += 1;
        NB_CUDA(c, cudaGetLastError());
    }
    c->last_r = r;
    c->last_jl = jl;
    c->last_s = (int)S;
    c->last_ctas = i_tiles * S;
    return NBODY_OK;
}

}  // namespace nbody
