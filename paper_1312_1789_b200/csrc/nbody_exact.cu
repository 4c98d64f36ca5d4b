// libnbody.so, translation unit 1: context management and the fp64 bit-exact kernels
//   K_pred (a-2), K_corr (a-4), initial dt, block selection (a-1), j-store export, host-buffer path.
// Compiled with -fmad=false; in addition every fp64 operation whose rounding matters is written with the
// __d*_rn intrinsics, which are never contracted, so the results equal a plain IEEE evaluation in the
// stated order (R12).  The formulas restate DESIGN.md section 3 (R5..R9); the paper
// itself names the scheme only.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "nbody_internal.h"

using namespace nbody;

namespace {

__device__ __forceinline__ double dadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double dsub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double dmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double ddiv(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double dsqrt(double a) { return __dsqrt_rn(a); }

// exact 2^e for e in the normal range
__device__ __forceinline__ double pow2i(int e) { return __longlong_as_double((long long)(e + 1023) << 52); }

struct PredArgs {
    const double *t, *m, *x, *v;
    const double *D[6];
    uint4 *q[kPlanes];
    double t_now;
    long long n, n_pad;
    int write_ds;
};

__device__ __forceinline__ uint4 pack_dd(double a, double b) {
    uint4 r;
    long long ia = __double_as_longlong(a), ib = __double_as_longlong(b);
    r.x = (unsigned)(ia & 0xffffffffll);
    r.y = (unsigned)((unsigned long long)ia >> 32);
    r.z = (unsigned)(ib & 0xffffffffll);
    r.w = (unsigned)((unsigned long long)ib >> 32);
    return r;
}
__device__ __forceinline__ uint4 pack_dff(double a, float b, float c) {
    uint4 r;
    long long ia = __double_as_longlong(a);
    r.x = (unsigned)(ia & 0xffffffffll);
    r.y = (unsigned)((unsigned long long)ia >> 32);
    r.z = __float_as_uint(b);
    r.w = __float_as_uint(c);
    return r;
}
__device__ __forceinline__ uint4 pack_ffff(float a, float b, float c, float d) {
    return make_uint4(__float_as_uint(a), __float_as_uint(b), __float_as_uint(c), __float_as_uint(d));
}

// K_pred: one thread per j-store slot (particles, then pads).  R5: Horner, innermost first, c_k = tau / k.
template <int ORDER>
__global__ void __launch_bounds__(256) k_predict(PredArgs A) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.n_pad) return;
    double xp[3];
    float vp[3], ap[3] = {0.f, 0.f, 0.f}, jp[3] = {0.f, 0.f, 0.f}, m32 = 0.f;
    if (i < A.n) {
        constexpr int ND = ORDER - 2;
        const double tau = dsub(A.t_now, A.t[i]);
        double c[9];
#pragma unroll
        for (int k = 1; k <= 8; ++k) c[k] = ddiv(tau, (double)k);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const long long q = 3 * i + d;
            double Dk[ND];
#pragma unroll
            for (int k = 0; k < ND; ++k) Dk[k] = A.D[k][q];
            double s = Dk[ND - 1];
#pragma unroll
            for (int k = ND - 1; k >= 1; --k) s = dadd(Dk[k - 1], dmul(c[k + 2], s));
            const double vq = A.v[q];
            xp[d] = dadd(A.x[q], dmul(tau, dadd(vq, dmul(c[2], s))));
            s = Dk[ND - 1];
#pragma unroll
            for (int k = ND - 1; k >= 1; --k) s = dadd(Dk[k - 1], dmul(c[k + 1], s));
            vp[d] = __double2float_rn(dadd(vq, dmul(tau, s)));
            if (ORDER >= 6) {
                s = Dk[ND - 1];
#pragma unroll
                for (int k = ND - 1; k >= 1; --k) s = dadd(Dk[k - 1], dmul(c[k], s));
                ap[d] = __double2float_rn(s);
            }
            if (ORDER >= 8) {
                s = Dk[ND - 1];
#pragma unroll
                for (int k = ND - 1; k >= 2; --k) s = dadd(Dk[k - 1], dmul(c[k - 1], s));
                jp[d] = __double2float_rn(s);
            }
        }
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
            lo[d] = __double2float_rn(dsub(xp[d], (double)hi[d]));
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

}  // namespace

// ---------------------------------------------------------------------------------------------------------
// K_corr (a-4): R6 corrector, R7 interpolated derivatives, R8 criterion, R9 quantisation.
// ---------------------------------------------------------------------------------------------------------
namespace {

#define P_(a, b) dadd((a), (b))
#define S_(a, b) dsub((a), (b))
#define M_(a, b) dmul((a), (b))
#define Q_(a, b) ddiv((a), (b))

__device__ __forceinline__ double nrm3(const double *a) {
    return dsqrt(P_(P_(M_(a[0], a[0]), M_(a[1], a[1])), M_(a[2], a[2])));
}

// R9 step 1: largest k in [k_lo, k_hi] with Ap * 2^(k q) <= A1 * E, else k_lo - 1 (NaN: every comparison false).
__device__ __forceinline__ int floor_log2_ratio(double A1, double Ap, double E, int q, int k_lo, int k_hi) {
    const double rhs = M_(A1, E);
    int k = k_hi;
    while (k >= k_lo && !(M_(Ap, pow2i(k * q)) <= rhs)) --k;
    return k;
}

// R8 + R9 for one particle; d[k] = a^(k)(t1), k = 0..p-1
template <int ORDER>
__device__ __forceinline__ double new_dt(const double (*d)[3], double t1, double dt_old, double eta, int k_min,
                                         int k_max, double dt_min, double dt_max) {
    constexpr int p = ORDER, q = p - 3;
    const double n0 = nrm3(d[0]), n1 = nrm3(d[1]), n2 = nrm3(d[2]);
    const double m3 = nrm3(d[p - 3]), m2 = nrm3(d[p - 2]), m1 = nrm3(d[p - 1]);
    const double A1 = dsqrt(P_(M_(n0, n2), M_(n1, n1)));
    const double Ap = dsqrt(P_(M_(m3, m1), M_(m2, m2)));
    double E = 1.0;
#pragma unroll
    for (int k = 0; k < q; ++k) E = M_(E, eta);
    const int k = floor_log2_ratio(A1, Ap, E, q, k_min - 1, k_max + 1);
    double dt_new = pow2i(k);
    const double two_old = M_(2.0, dt_old);
    if (dt_new > two_old) dt_new = two_old;
    if (dt_new == two_old) {
        const double r = Q_(t1, dt_new);  // exact: dt_new is a power of two
        if (r != rint(r)) dt_new = dt_old;
    }
    if (dt_new > dt_max) dt_new = dt_max;
    if (dt_new < dt_min) dt_new = dt_min;
    return dt_new;
}

struct CorrArgs {
    const int32_t *idx;
    long long n_act;
    double t_now, eta, dt_min, dt_max;
    int k_min, k_max;
    int crit_order;  // R8b: criterion evaluated on the lowest crit_order derivatives (<= ORDER)
    double *t, *dt, *x, *v, *D[8], *pot_state;
    const double *acc, *jerk, *snap, *crk, *pot;
};

template <int ORDER>
__global__ void __launch_bounds__(128) k_correct(CorrArgs A) {
    const long long ia = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ia >= A.n_act) return;
    const long long i = A.idx[ia];
    const double h = A.dt[i];
    const double h2 = M_(h, h), h3 = M_(h2, h), h4 = M_(h3, h), h5 = M_(h4, h), h6 = M_(h5, h), h7 = M_(h6, h);
    double dn[8][3];
    double cbar[3] = {0.0, 0.0, 0.0};  // R8b, p = 6: mean crackle over the step, (s1 - s0) / h
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const long long q = 3 * i + c, qa = 3 * ia + c;
        const double x0 = A.x[q], v0 = A.v[q];
        const double a0 = A.D[0][q], j0 = A.D[1][q];
        const double a1 = A.acc[qa], j1 = A.jerk[qa];
        const double dl = S_(a0, a1);
        const double hh = Q_(h, 2.0);
        double v1, x1;
        if (ORDER == 4) {
            const double w = Q_(h2, 12.0);
            v1 = P_(v0, P_(M_(hh, P_(a0, a1)), M_(w, S_(j0, j1))));
            x1 = P_(x0, P_(M_(hh, P_(v0, v1)), M_(w, S_(a0, a1))));
            const double A2 = Q_(M_(2.0, P_(P_(M_(3.0, dl), M_(h, j0)), M_(M_(2.0, h), j1))), h2);
            const double A3 = Q_(M_(6.0, P_(P_(M_(2.0, dl), M_(h, j0)), M_(h, j1))), h3);
            dn[0][c] = a1; dn[1][c] = j1; dn[2][c] = A2; dn[3][c] = A3;
        } else if (ORDER == 6) {
            const double s0 = A.D[2][q], s1 = A.snap[qa];
            const double w2 = Q_(h2, 10.0), w3 = Q_(h3, 120.0);
            v1 = P_(v0, P_(M_(hh, P_(a0, a1)), P_(M_(w2, S_(j0, j1)), M_(w3, P_(s0, s1)))));
            x1 = P_(x0, P_(M_(hh, P_(v0, v1)), P_(M_(w2, S_(a0, a1)), M_(w3, P_(j0, j1)))));
            const double A3 = Q_(M_(-3.0, S_(P_(P_(P_(M_(20.0, dl), M_(M_(8.0, h), j0)), M_(M_(12.0, h), j1)), M_(h2, s0)), M_(M_(3.0, h2), s1))), h3);
            const double A4 = Q_(M_(-12.0, S_(P_(P_(P_(M_(30.0, dl), M_(M_(14.0, h), j0)), M_(M_(16.0, h), j1)), M_(M_(2.0, h2), s0)), M_(M_(3.0, h2), s1))), h4);
            const double A5 = Q_(M_(-60.0, S_(P_(P_(P_(M_(12.0, dl), M_(M_(6.0, h), j0)), M_(M_(6.0, h), j1)), M_(h2, s0)), M_(h2, s1))), h5);
            dn[0][c] = a1; dn[1][c] = j1; dn[2][c] = s1; dn[3][c] = A3; dn[4][c] = A4; dn[5][c] = A5;
            cbar[c] = Q_(S_(s1, s0), h);
        } else {
            const double s0 = A.D[2][q], s1 = A.snap[qa];
            const double c0 = A.D[3][q], c1 = A.crk[qa];
            const double w2 = Q_(M_(3.0, h2), 28.0), w3 = Q_(h3, 84.0), w4 = Q_(h4, 1680.0);
            v1 = P_(v0, P_(M_(hh, P_(a0, a1)), P_(M_(w2, S_(j0, j1)), P_(M_(w3, P_(s0, s1)), M_(w4, S_(c0, c1))))));
            x1 = P_(x0, P_(M_(hh, P_(v0, v1)), P_(M_(w2, S_(a0, a1)), P_(M_(w3, P_(j0, j1)), M_(w4, S_(s0, s1))))));
#define HERM8(k0, kj0, kj1, ks0, ks1, kc0, kc1)                                                                     \
    P_(P_(S_(P_(P_(P_(M_(k0, dl), M_(M_(kj0, h), j0)), M_(M_(kj1, h), j1)), M_(M_(ks0, h2), s0)), M_(M_(ks1, h2), s1)), \
          kc0),                                                                                                   \
       kc1)
            const double A4 = Q_(M_(4.0, HERM8(210.0, 90.0, 120.0, 15.0, 30.0, M_(h3, c0), M_(M_(4.0, h3), c1))), h4);
            const double A5 = Q_(M_(60.0, HERM8(168.0, 78.0, 90.0, 14.0, 20.0, M_(h3, c0), M_(M_(2.0, h3), c1))), h5);
            const double A6 = Q_(M_(120.0, HERM8(420.0, 204.0, 216.0, 39.0, 45.0, M_(M_(3.0, h3), c0), M_(M_(4.0, h3), c1))), h6);
            const double A7 = Q_(M_(840.0, HERM8(120.0, 60.0, 60.0, 12.0, 12.0, M_(h3, c0), M_(h3, c1))), h7);
#undef HERM8
            dn[0][c] = a1; dn[1][c] = j1; dn[2][c] = s1; dn[3][c] = c1;
            dn[4][c] = A4; dn[5][c] = A5; dn[6][c] = A6; dn[7][c] = A7;
        }
        A.x[q] = x1;
        A.v[q] = v1;
    }
    double dt_new;
    if (ORDER == 6 && A.crit_order == 4) {  // only directly computed derivatives enter the step decision
        double d4[4][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            d4[0][c] = dn[0][c]; d4[1][c] = dn[1][c]; d4[2][c] = dn[2][c]; d4[3][c] = cbar[c];
        }
        dt_new = new_dt<4>(d4, A.t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    } else if (ORDER >= 8 && A.crit_order == 4)
        dt_new = new_dt<4>(dn, A.t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    else if (ORDER >= 8 && A.crit_order == 6)
        dt_new = new_dt<6>(dn, A.t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    else
        dt_new = new_dt<ORDER>(dn, A.t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
#pragma unroll
    for (int k = 0; k < ORDER; ++k)
#pragma unroll
        for (int c = 0; c < 3; ++c) A.D[k][3 * i + c] = dn[k][c];
    A.pot_state[i] = A.pot[ia];
    A.t[i] = A.t_now;
    A.dt[i] = dt_new;
}

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
// Block selection (a-1, R9c): min of t + dt, then order-preserving compaction of the particles due at it.
// ---------------------------------------------------------------------------------------------------------
namespace {

constexpr int kSelThreads = 256;
constexpr int kSelPerThread = 8;
constexpr int kSelBlock = kSelThreads * kSelPerThread;  // particles per selection CTA

// order-preserving map double -> uint64 (total order of finite values)
__device__ __forceinline__ unsigned long long dkey(double v) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dunkey(unsigned long long k) {
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

__global__ void k_sel_init(unsigned long long *min_key, long long *n_act) {
    *min_key = ~0ull;
    *n_act = 0;
}

__global__ void __launch_bounds__(kSelThreads) k_sel_min(long long n, const double *t, const double *dt,
                                                         unsigned long long *min_key) {
    unsigned long long k = ~0ull;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long ki = dkey(dadd(t[i], dt[i]));
        k = ki < k ? ki : k;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other < k ? other : k;
    }
    __shared__ unsigned long long sm[kSelThreads / 32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = k;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kSelThreads / 32; ++w) k = sm[w] < k ? sm[w] : k;
        atomicMin(min_key, k);
    }
}

// counts[b] = number of due particles in chunk b
__global__ void __launch_bounds__(kSelThreads) k_sel_count(long long n, const double *t, const double *dt,
                                                           const unsigned long long *min_key, int *counts) {
    const unsigned long long key = *min_key;
    const long long base = (long long)blockIdx.x * kSelBlock + (long long)threadIdx.x * kSelPerThread;
    int c = 0;
#pragma unroll
    for (int u = 0; u < kSelPerThread; ++u) {
        const long long i = base + u;
        if (i < n && dkey(dadd(t[i], dt[i])) == key) ++c;
    }
    c = __reduce_add_sync(0xffffffffu, c);
    __shared__ int sm[kSelThreads / 32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        int s = 0;
        for (int w = 0; w < kSelThreads / 32; ++w) s += sm[w];
        counts[blockIdx.x] = s;
    }
}

// exclusive scan of counts[0..nb) in place by one CTA; total -> *n_act, t_next -> ret[0]
__global__ void __launch_bounds__(1024) k_sel_scan(int nb, int *counts, long long *n_act,
                                                   const unsigned long long *min_key, double *ret) {
    __shared__ int sm[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < nb ? counts[i] : 0;
        sm[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const int add = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
            __syncthreads();
            sm[threadIdx.x] += add;
            __syncthreads();
        }
        if (i < nb) counts[i] = carry + sm[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry += sm[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *n_act = carry;
        ret[0] = dunkey(*min_key);
        ret[1] = (double)carry;
    }
}

__global__ void __launch_bounds__(kSelThreads) k_sel_write(long long n, const double *t, const double *dt,
                                                           const unsigned long long *min_key, const int *offsets,
                                                           int32_t *active_idx) {
    const unsigned long long key = *min_key;
    const long long base = (long long)blockIdx.x * kSelBlock + (long long)threadIdx.x * kSelPerThread;
    unsigned flags = 0;
    int c = 0;
#pragma unroll
    for (int u = 0; u < kSelPerThread; ++u) {
        const long long i = base + u;
        if (i < n && dkey(dadd(t[i], dt[i])) == key) {
            flags |= 1u << u;
            ++c;
        }
    }
    // exclusive scan of c over the CTA (thread order == index order)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
    }
    __shared__ int wsum[kSelThreads / 32];
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    int woff = 0;
    for (int w = 0; w < warp; ++w) woff += wsum[w];
    int pos = offsets[blockIdx.x] + woff + incl - c;
#pragma unroll
    for (int u = 0; u < kSelPerThread; ++u)
        if (flags & (1u << u)) active_idx[pos++] = (int32_t)(base + u);
}

bool is_pow2(double x, int *e) {
    if (!(x > 0.0) || isinf(x)) return false;
    int ex;
    const double f = frexp(x, &ex);
    *e = ex - 1;
    return f == 0.5;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------------------
struct nbody_ctx {
    Ctx c;
};

extern "C" {

int nbody_abi_version(void) { return 1; }

const char *nbody_strerror(int code) {
    switch (code) {
        case NBODY_OK: return "ok";
        case NBODY_EINVAL: return "invalid argument";
        case NBODY_ESTATE: return "invalid call order (predict first; force order <= predict order)";
        case NBODY_ECUDA: return "CUDA runtime error (see nbody_last_cuda_error)";
        case NBODY_ENOMEM: return "out of memory";
        default: return "unknown nbody error code";
    }
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
    int rc = NBODY_OK;
    do {
        cudaError_t e;
        if ((e = cudaSetDevice(device)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        cudaDeviceProp prop;
        if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        c->sm_count = prop.multiProcessorCount;
        c->cap = n_capacity;
        c->cap_pad = (n_capacity + kTileJ - 1) / kTileJ * kTileJ;
        if ((e = cudaMalloc(&c->jstore, sizeof(uint4) * kPlanes * c->cap_pad)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        c->counts_cap = (c->cap + kSelBlock - 1) / kSelBlock + 1;
        if ((e = cudaMalloc(&c->d_counts, sizeof(int) * c->counts_cap)) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_min_key, sizeof(unsigned long long))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMalloc(&c->d_nact, sizeof(long long))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        if ((e = cudaMallocHost(&c->h_pinned, 4 * sizeof(double))) != cudaSuccess) { rc = cuda_fail(c, e); break; }
        rc = force_static_init(c);
        if (rc != NBODY_OK) break;
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
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    cudaFree(c->jstore);
    cudaFree(c->partials);
    cudaFree(c->d_counts);
    cudaFree(c->d_min_key);
    cudaFree(c->d_nact);
    cudaFree(c->stage);
    if (c->h_pinned) cudaFreeHost(c->h_pinned);
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
        if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 && value != 32 && value != 128) return NBODY_EINVAL;
        c->force_lanes = (int)value;
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
        for (int k = 0; k <= order - 3; ++k)
            if (!a_derivs[k]) return NBODY_EINVAL;
    }
    c->n = n;
    c->n_pad = (n + kTileJ - 1) / kTileJ * kTileJ;
    c->pred_order = order;
    c->ds_valid = c->diff_mode == 1;
    if (n == 0) return NBODY_OK;
    PredArgs A;
    A.t = t; A.m = m; A.x = x; A.v = v;
    for (int k = 0; k < 6; ++k) A.D[k] = k <= order - 3 ? a_derivs[k] : nullptr;
    for (int p = 0; p < kPlanes; ++p) A.q[p] = c->jstore + (size_t)p * c->cap_pad;
    A.t_now = t_now;
    A.n = n;
    A.n_pad = c->n_pad;
    A.write_ds = c->ds_valid ? 1 : 0;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = (unsigned)((c->n_pad + 255) / 256);
    if (order == 4) k_predict<4><<<grid, 256, 0, st>>>(A);
    else if (order == 6) k_predict<6><<<grid, 256, 0, st>>>(A);
    else k_predict<8><<<grid, 256, 0, st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_force(nbody_ctx *h, const int32_t *active_idx, int64_t n_act, int order, double eps2, double *acc,
                double *jerk, double *snap, double *crackle, double *pot, void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n_act < 0) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (!(eps2 >= 0.0) || isinf(eps2)) return NBODY_EINVAL;
    if (c->n < 0 || order > c->pred_order) return NBODY_ESTATE;
    if (n_act > c->n) return NBODY_EINVAL;
    if (n_act == 0) return NBODY_OK;
    if (!active_idx || !acc || !jerk || !pot || (order >= 6 && !snap) || (order >= 8 && !crackle)) return NBODY_EINVAL;
    if (c->diff_mode == 1 && !c->ds_valid) return NBODY_ESTATE;
    return launch_force(c, active_idx, n_act, order, (float)eps2, acc, jerk, snap, crackle, pot, (cudaStream_t)stream);
}

int nbody_correct(nbody_ctx *h, const int32_t *active_idx, int64_t n_act, int order, double t_now, double eta,
                  double dt_min, double dt_max, double *t, double *dt, double *x, double *v,
                  double *const a_derivs[8], double *pot_state, const double *acc, const double *jerk,
                  const double *snap, const double *crackle, const double *pot, void *stream) {
    if (!h || (order != 4 && order != 6 && order != 8) || n_act < 0) return NBODY_EINVAL;
    Ctx *c = &h->c;
    int kmin, kmax;
    if (!(eta > 0.0) || !is_pow2(dt_min, &kmin) || !is_pow2(dt_max, &kmax) || dt_min > dt_max) return NBODY_EINVAL;
    if (kmin < -900 || kmax > 900) return NBODY_EINVAL;
    if (n_act == 0) return NBODY_OK;
    if (!active_idx || !t || !dt || !x || !v || !a_derivs || !pot_state || !acc || !jerk || !pot) return NBODY_EINVAL;
    if ((order >= 6 && !snap) || (order >= 8 && !crackle)) return NBODY_EINVAL;
    for (int k = 0; k < order; ++k)
        if (!a_derivs[k]) return NBODY_EINVAL;
    CorrArgs A;
    A.idx = active_idx; A.n_act = n_act; A.t_now = t_now; A.eta = eta; A.dt_min = dt_min; A.dt_max = dt_max;
    A.k_min = kmin; A.k_max = kmax;
    // 0 = automatic: R8b (pc = 4) for p >= 6, where the order-p criterion collapses under fp32 force noise
    A.crit_order = c->crit_order ? (c->crit_order < order ? c->crit_order : order) : (order >= 6 ? 4 : order);
    A.t = t; A.dt = dt; A.x = x; A.v = v; A.pot_state = pot_state;
    for (int k = 0; k < 8; ++k) A.D[k] = k < order ? a_derivs[k] : nullptr;
    A.acc = acc; A.jerk = jerk; A.snap = snap; A.crk = crackle; A.pot = pot;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = (unsigned)((n_act + 127) / 128);
    if (order == 4) k_correct<4><<<grid, 128, 0, st>>>(A);
    else if (order == 6) k_correct<6><<<grid, 128, 0, st>>>(A);
    else k_correct<8><<<grid, 128, 0, st>>>(A);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_initial_dt(nbody_ctx *h, int64_t n, const double *acc, const double *jerk, double eta_s, double dt_min,
                     double dt_max, double *dt, void *stream) {
    if (!h || n < 0) return NBODY_EINVAL;
    int kmin, kmax;
    if (!(eta_s > 0.0) || !is_pow2(dt_min, &kmin) || !is_pow2(dt_max, &kmax) || dt_min > dt_max) return NBODY_EINVAL;
    if (n == 0) return NBODY_OK;
    if (!acc || !jerk || !dt) return NBODY_EINVAL;
    Ctx *c = &h->c;
    k_initial_dt<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n, acc, jerk, eta_s, kmin, kmax, dt_min,
                                                                              dt_max, dt);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_next_block(nbody_ctx *h, int64_t n, const double *t, const double *dt, int32_t *active_idx,
                     double *t_next_host, int64_t *n_act_host, void *stream) {
    if (!h || n < 1 || n > h->c.cap || !t || !dt || !active_idx || !t_next_host || !n_act_host) return NBODY_EINVAL;
    Ctx *c = &h->c;
    cudaStream_t st = (cudaStream_t)stream;
    const int nb = (int)((n + kSelBlock - 1) / kSelBlock);
    k_sel_init<<<1, 1, 0, st>>>(c->d_min_key, c->d_nact);
    const int gmin = nb < 4 * c->sm_count ? nb : 4 * c->sm_count;
    k_sel_min<<<gmin, kSelThreads, 0, st>>>(n, t, dt, c->d_min_key);
    k_sel_count<<<nb, kSelThreads, 0, st>>>(n, t, dt, c->d_min_key, c->d_counts);
    k_sel_scan<<<1, 1024, 0, st>>>(nb, c->d_counts, c->d_nact, c->d_min_key, c->h_pinned);
    k_sel_write<<<nb, kSelThreads, 0, st>>>(n, t, dt, c->d_min_key, c->d_counts, active_idx);
    c->launches += 5;
    NB_CUDA(c, cudaGetLastError());
    NB_CUDA(c, cudaStreamSynchronize(st));
    *t_next_host = c->h_pinned[0];
    *n_act_host = (int64_t)c->h_pinned[1];
    return NBODY_OK;
}

int nbody_get_predicted(nbody_ctx *h, double *xp, float *vp, float *ap, float *jp, float *m32, void *stream) {
    if (!h || !xp || !vp || !m32) return NBODY_EINVAL;
    Ctx *c = &h->c;
    if (c->n < 0) return NBODY_ESTATE;
    if ((ap && c->pred_order < 6) || (jp && c->pred_order < 8)) return NBODY_EINVAL;
    if (c->n == 0) return NBODY_OK;
    const uint4 *q = c->jstore;
    k_unpack<<<(unsigned)((c->n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        q, q + c->cap_pad, q + 2 * c->cap_pad, q + 3 * c->cap_pad, c->n, c->pred_order, xp, vp, ap, jp, m32);
    c->launches += 1;
    NB_CUDA(c, cudaGetLastError());
    return NBODY_OK;
}

int nbody_probe_peak(nbody_ctx *h, int kind, int millis, double *tera_ops_host) {
    if (!h || !tera_ops_host || kind < 0 || kind > 6 || millis < 1 || millis > 20000) return NBODY_EINVAL;
    return probe_peak(&h->c, kind, millis, tera_ops_host);
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// Host-buffer path (end-to-end measurement): H2D of the state, predict, force, D2H of the results.
// ---------------------------------------------------------------------------------------------------------
extern "C" int nbody_force_host(nbody_ctx *h, int64_t n, double t_now, int order, const double *t, const double *m,
                                const double *x, const double *v, const double *const a_derivs[6],
                                const int32_t *active_idx, int64_t n_act, double eps2, double *acc, double *jerk,
                                double *snap, double *crackle, double *pot, int64_t *h2d_bytes, int64_t *d2h_bytes) {
    if (!h || (order != 4 && order != 6 && order != 8) || n < 1 || n > h->c.cap || n_act < 0 || n_act > n)
        return NBODY_EINVAL;
    if (!t || !m || !x || !v || !a_derivs || (n_act > 0 && (!active_idx || !acc || !jerk || !pot))) return NBODY_EINVAL;
    if (n_act > 0 && ((order >= 6 && !snap) || (order >= 8 && !crackle))) return NBODY_EINVAL;
    const int nd = order - 2, K = order / 2;
    for (int k = 0; k < nd; ++k)
        if (!a_derivs[k]) return NBODY_EINVAL;
    Ctx *c = &h->c;
    NB_CUDA(c, cudaSetDevice(c->device));
    // staging layout (doubles): t[n] m[n] x[3n] v[3n] D[nd][3n] | out: K x [3 n_act] + pot[n_act] | idx int32[n_act]
    const size_t in_d = (size_t)n * (2 + 6 + 3 * (size_t)nd);
    const size_t out_d = (size_t)n_act * (3 * (size_t)K + 1);
    const size_t need = (in_d + out_d) * sizeof(double) + (size_t)n_act * sizeof(int32_t) + 256;
    if (need > c->stage_bytes) {
        NB_CUDA(c, cudaDeviceSynchronize());
        cudaFree(c->stage);
        c->stage = nullptr;
        c->stage_bytes = 0;
        NB_CUDA(c, cudaMalloc(&c->stage, need));
        c->stage_bytes = need;
    }
    cudaStream_t st = 0;
    double *d = (double *)c->stage;
    double *dt_ = d, *dm = d + n, *dx = d + 2 * n, *dv = d + 5 * n;
    const double *dD[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int64_t up = 0, down = 0;
    NB_CUDA(c, cudaMemcpyAsync(dt_, t, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    NB_CUDA(c, cudaMemcpyAsync(dm, m, sizeof(double) * n, cudaMemcpyHostToDevice, st));
    NB_CUDA(c, cudaMemcpyAsync(dx, x, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st));
    NB_CUDA(c, cudaMemcpyAsync(dv, v, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st));
    up += (int64_t)sizeof(double) * 8 * n;
    for (int k = 0; k < nd; ++k) {
        double *p = d + 8 * n + (size_t)k * 3 * n;
        NB_CUDA(c, cudaMemcpyAsync(p, a_derivs[k], sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st));
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
    int rc = nbody_predict(h, n, t_now, order, dt_, dm, dx, dv, dD, st);
    if (rc != NBODY_OK) return rc;
    if (n_act > 0) {
        NB_CUDA(c, cudaMemcpyAsync(d_idx, active_idx, sizeof(int32_t) * n_act, cudaMemcpyHostToDevice, st));
        up += (int64_t)sizeof(int32_t) * n_act;
        rc = nbody_force(h, d_idx, n_act, order, eps2, o_acc, o_jerk, o_snap, o_crk, o_pot, st);
        if (rc != NBODY_OK) return rc;
        NB_CUDA(c, cudaMemcpyAsync(acc, o_acc, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        NB_CUDA(c, cudaMemcpyAsync(jerk, o_jerk, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        if (order >= 6) NB_CUDA(c, cudaMemcpyAsync(snap, o_snap, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        if (order >= 8) NB_CUDA(c, cudaMemcpyAsync(crackle, o_crk, sizeof(double) * 3 * n_act, cudaMemcpyDeviceToHost, st));
        NB_CUDA(c, cudaMemcpyAsync(pot, o_pot, sizeof(double) * n_act, cudaMemcpyDeviceToHost, st));
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
    NB_CUDA(c, cudaSetDevice(c->device));
    const int K = order / 2;
    // staging (doubles): t dt m pot [n] | x v [3n] | D[order][3n] | acc jerk snap crk [3n] fpot [n] | idx int32[n]
    const size_t nd = (size_t)n * (4 + 6 + 3 * (size_t)order + 12 + 1);
    const size_t need = nd * sizeof(double) + (size_t)n * sizeof(int32_t) + 256;
    if (need > c->stage_bytes) {
        NB_CUDA(c, cudaDeviceSynchronize());
        cudaFree(c->stage);
        c->stage = nullptr;
        c->stage_bytes = 0;
        NB_CUDA(c, cudaMalloc(&c->stage, need));
        c->stage_bytes = need;
    }
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
    NB_CUDA(c, h2d(d_t, t, n));
    NB_CUDA(c, h2d(d_dt, dt, n));
    NB_CUDA(c, h2d(d_m, m, n));
    NB_CUDA(c, h2d(d_pot, pot_state, n));
    NB_CUDA(c, h2d(d_x, x, 3 * n));
    NB_CUDA(c, h2d(d_v, v, 3 * n));
    for (int k = 0; k < order; ++k) NB_CUDA(c, h2d(d_D[k], a_derivs[k], 3 * n));
    double t_next = 0.0;
    int64_t n_act = 0;
    int rc = nbody_next_block(h, n, d_t, d_dt, d_idx, &t_next, &n_act, st);
    if (rc != NBODY_OK) return rc;
    rc = nbody_predict(h, n, t_next, order, d_t, d_m, d_x, d_v, d_D, st);
    if (rc != NBODY_OK) return rc;
    rc = nbody_force(h, d_idx, n_act, order, eps2, o_acc, o_jerk, K >= 3 ? o_snap : nullptr, K >= 4 ? o_crk : nullptr,
                     o_pot, st);
    if (rc != NBODY_OK) return rc;
    rc = nbody_correct(h, d_idx, n_act, order, t_next, eta, dt_min, dt_max, d_t, d_dt, d_x, d_v, d_D, d_pot, o_acc,
                       o_jerk, K >= 3 ? o_snap : nullptr, K >= 4 ? o_crk : nullptr, o_pot, st);
    if (rc != NBODY_OK) return rc;
    NB_CUDA(c, d2h(t, d_t, n));
    NB_CUDA(c, d2h(dt, d_dt, n));
    NB_CUDA(c, d2h(pot_state, d_pot, n));
    NB_CUDA(c, d2h(x, d_x, 3 * n));
    NB_CUDA(c, d2h(v, d_v, 3 * n));
    for (int k = 0; k < order; ++k) NB_CUDA(c, d2h(a_derivs[k], d_D[k], 3 * n));
    NB_CUDA(c, cudaStreamSynchronize(st));
    *t_next_host = t_next;
    *n_act_host = n_act;
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return NBODY_OK;
}
