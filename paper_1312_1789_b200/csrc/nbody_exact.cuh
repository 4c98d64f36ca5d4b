// Device code shared by the translation units of libnbody.so: the bit-exact fp64 pieces (R12) -- Taylor predictor of
// one particle (R5), Hermite corrector + time step of one particle (R6..R9, R8b, R14) -- used by the stand-alone
// kernels K_pred / K_corr (nbody_exact.cu) and by the fused small-block kernel (nbody_force.cu).  Every fp64 operation
// whose rounding matters is an __d*_rn intrinsic (never contracted, whatever -fmad says), in the oracle's order.
#pragma once
#include "nbody_internal.h"

namespace nbody {

__device__ __forceinline__ double d_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double d_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double d_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double d_div(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double d_sqrt(double a) { return __dsqrt_rn(a); }

// exact 2^e for e in the normal range [-1022, 1023] (the callers validate (|k| + 1) q <= 1022 on the host)
__device__ __forceinline__ double pow2i(int e) { return __longlong_as_double((long long)(e + 1023) << 52); }

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


// R5 for one particle: tau = t_now - t_i; x3, v3 and Dp[k] point at the particle's three components of x, v and
// a^(k) (k = 0 .. ORDER-3).  Horner, innermost first, c_k = tau / k.  Outputs: x_p (fp64), v_p, a_p, j_p rounded to fp32.
// The four polynomials are independent chains; DO_X .. DO_J select which of them this thread evaluates (the fused
// small-block kernel splits a particle over two threads), the arithmetic of each is the same whoever evaluates it.
template <int ORDER, bool DO_X = true, bool DO_V = true, bool DO_A = true, bool DO_J = true>
__device__ __forceinline__ void predict_particle(const double tau, const double *x3, const double *v3,
                                                 const double *const *Dp, double (&xp)[3], float (&vp)[3],
                                                 float (&ap)[3], float (&jp)[3]) {
    constexpr int ND = ORDER - 2;
    // c_k = fl(tau / k), as the oracle's IEEE division gives it: dividing by 2, 4, 8 is an exact scaling, and
    // fl(tau / 6) = fl(tau / 3) / 2 because halving commutes with rounding (no underflow: |tau| >= 2^-1000 or 0), so only
    // k = 3, 5, 7 need a real division (a division is ~45 instructions on the fp64 pipe: they dominated the predictor).
    double c[9];
    c[1] = tau;
    c[2] = d_mul(tau, 0.5);
    c[3] = d_div(tau, 3.0);
    c[4] = d_mul(tau, 0.25);
    c[5] = d_div(tau, 5.0);
    c[6] = d_mul(c[3], 0.5);
    c[7] = d_div(tau, 7.0);
    c[8] = d_mul(tau, 0.125);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double Dk[ND];
#pragma unroll
        for (int k = 0; k < ND; ++k) Dk[k] = Dp[k][d];
        double s;
        if (DO_X) {
            s = Dk[ND - 1];
#pragma unroll
            for (int k = ND - 1; k >= 1; --k) s = d_add(Dk[k - 1], d_mul(c[k + 2], s));
            xp[d] = d_add(x3[d], d_mul(tau, d_add(v3[d], d_mul(c[2], s))));
        }
        if (DO_V) {
            s = Dk[ND - 1];
#pragma unroll
            for (int k = ND - 1; k >= 1; --k) s = d_add(Dk[k - 1], d_mul(c[k + 1], s));
            vp[d] = __double2float_rn(d_add(v3[d], d_mul(tau, s)));
        }
        if (DO_A) {
            ap[d] = 0.f;
            if (ORDER >= 6) {
                s = Dk[ND - 1];
#pragma unroll
                for (int k = ND - 1; k >= 1; --k) s = d_add(Dk[k - 1], d_mul(c[k], s));
                ap[d] = __double2float_rn(s);
            }
        }
        if (DO_J) {
            jp[d] = 0.f;
            if (ORDER >= 8) {
                s = Dk[ND - 1];
#pragma unroll
                for (int k = ND - 1; k >= 2; --k) s = d_add(Dk[k - 1], d_mul(c[k - 1], s));
                jp[d] = __double2float_rn(s);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// K_corr (a-4) for one particle: R6 corrector, R7 interpolated derivatives, R8 / R8b criterion, R9 quantisation,
// R14 a-posteriori step rejection.
// ---------------------------------------------------------------------------------------------------------
#define P_(a, b) d_add((a), (b))
#define S_(a, b) d_sub((a), (b))
#define M_(a, b) d_mul((a), (b))
#define Q_(a, b) d_div((a), (b))

__device__ __forceinline__ double nrm3(const double *a) {
    return d_sqrt(P_(P_(M_(a[0], a[0]), M_(a[1], a[1])), M_(a[2], a[2])));
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
    const double A1 = d_sqrt(P_(M_(n0, n2), M_(n1, n1)));
    const double Ap = d_sqrt(P_(M_(m3, m1), M_(m2, m2)));
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
    const Ctl *ctl;  // device-driven step: n_act and t_now from the control block (else NULL)
    int reject_ratio;               // R14 (SURVEY c-9b analogue): 0 = off
    unsigned long long *n_rejected; // device counter of refused steps
    int limit_order;                // R15 (oracle c-6b): corrector order limiter, 0 = off
    unsigned long long *n_limited;  // device counter of order-limited steps
};

// R6 for one component at a chosen order m2 = 2, 4, 6, 8 (2 = trapezoid), in the oracle's operation order (c-6b).
__device__ __forceinline__ void corrector_xv(int m2, double h, double x0, double v0, double a0, double a1, double j0,
                                             double j1, double s0, double s1, double c0, double c1, double &x1, double &v1) {
    const double h2 = M_(h, h), h3 = M_(h2, h), h4 = M_(h3, h);
    const double hh = Q_(h, 2.0);
    double v, x;
    if (m2 == 2) {
        v = P_(v0, M_(hh, P_(a0, a1)));
        x = P_(x0, M_(hh, P_(v0, v)));
    } else if (m2 == 4) {
        const double w = Q_(h2, 12.0);
        v = P_(v0, P_(M_(hh, P_(a0, a1)), M_(w, S_(j0, j1))));
        x = P_(x0, P_(M_(hh, P_(v0, v)), M_(w, S_(a0, a1))));
    } else if (m2 == 6) {
        const double w2 = Q_(h2, 10.0), w3 = Q_(h3, 120.0);
        v = P_(v0, P_(M_(hh, P_(a0, a1)), P_(M_(w2, S_(j0, j1)), M_(w3, P_(s0, s1)))));
        x = P_(x0, P_(M_(hh, P_(v0, v)), P_(M_(w2, S_(a0, a1)), M_(w3, P_(j0, j1)))));
    } else {
        const double w2 = Q_(M_(3.0, h2), 28.0), w3 = Q_(h3, 84.0), w4 = Q_(h4, 1680.0);
        v = P_(v0, P_(M_(hh, P_(a0, a1)), P_(M_(w2, S_(j0, j1)), P_(M_(w3, P_(s0, s1)), M_(w4, S_(c0, c1))))));
        x = P_(x0, P_(M_(hh, P_(v0, v)), P_(M_(w2, S_(a0, a1)), P_(M_(w3, P_(j0, j1)), M_(w4, S_(s0, s1))))));
    }
    x1 = x;
    v1 = v;
}

template <int ORDER>
__device__ __forceinline__ void correct_one(const CorrArgs &A, long long ia, double t_now);

template <int ORDER>
__global__ void __launch_bounds__(128) k_correct(CorrArgs A) {
    long long n_act = A.n_act;
    double t_now = A.t_now;
    if (A.ctl) {
        if (A.ctl->stop) return;
        n_act = A.ctl->n_act;
        t_now = A.ctl->t_next;
    }
    for (long long ia = (long long)blockIdx.x * blockDim.x + threadIdx.x; ia < n_act;
         ia += (long long)gridDim.x * blockDim.x)
        correct_one<ORDER>(A, ia, t_now);
}

template <int ORDER>
__device__ __forceinline__ void correct_one(const CorrArgs &A, const long long ia, const double t_now) {
    const long long i = A.idx[ia];
    const double h = A.dt[i];
    const double h2 = M_(h, h), h3 = M_(h2, h), h4 = M_(h3, h), h5 = M_(h4, h), h6 = M_(h5, h), h7 = M_(h6, h);
    double dn[8][3], xn[3], vn[3];
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
        xn[c] = x1;
        vn[c] = v1;
    }
    double dt_new;
    if (ORDER == 6 && A.crit_order == 4) {  // only directly computed derivatives enter the step decision
        double d4[4][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            d4[0][c] = dn[0][c]; d4[1][c] = dn[1][c]; d4[2][c] = dn[2][c]; d4[3][c] = cbar[c];
        }
        dt_new = new_dt<4>(d4, t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    } else if (ORDER >= 8 && A.crit_order == 4)
        dt_new = new_dt<4>(dn, t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    else if (ORDER >= 8 && A.crit_order == 6)
        dt_new = new_dt<6>(dn, t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    else
        dt_new = new_dt<ORDER>(dn, t_now, h, A.eta, A.k_min, A.k_max, A.dt_min, A.dt_max);
    if (A.limit_order) {  // R15 (oracle c-6b): use the highest corrector order whose quadrature terms do not grow
        constexpr int K = ORDER / 2;
        const double w[4] = {Q_(h, 2.0), ORDER == 4 ? Q_(h2, 12.0) : ORDER == 6 ? Q_(h2, 10.0) : Q_(M_(3.0, h2), 28.0),
                             ORDER == 6 ? Q_(h3, 120.0) : Q_(h3, 84.0), Q_(h4, 1680.0)};
        double T[4][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const long long q = 3 * i + c, qa = 3 * ia + c;
            T[0][c] = M_(w[0], P_(A.D[0][q], A.acc[qa]));
            T[1][c] = M_(w[1], S_(A.D[1][q], A.jerk[qa]));
            T[2][c] = K >= 3 ? M_(w[2], P_(A.D[2][q], A.snap[qa])) : 0.0;
            T[3][c] = K >= 4 ? M_(w[3], S_(A.D[3][q], A.crk[qa])) : 0.0;
        }
        // level 0: the first end-point correction U_1 = h/2 (a1 - a0) against U_0 = h a0
        double U0[3], U1[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            U0[c] = M_(h, A.D[0][3 * i + c]);
            U1[c] = M_(w[0], S_(A.acc[3 * ia + c], A.D[0][3 * i + c]));
        }
        int M = nrm3(U1) <= nrm3(U0) ? 1 : 0;
        while (M >= 1 && M < K && nrm3(T[M]) <= nrm3(T[M - 1])) ++M;
        if (M == 0) {  // the end point is not to be trusted at all: the particle's own Taylor prediction (R5, fp64)
            constexpr int ND = ORDER - 2;
            double ck[9];
#pragma unroll
            for (int k = 1; k <= 8; ++k) ck[k] = Q_(h, (double)k);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const long long q = 3 * i + c;
                double sx = A.D[ND - 1][q], sv = A.D[ND - 1][q];
#pragma unroll
                for (int k = ND - 1; k >= 1; --k) sx = P_(A.D[k - 1][q], M_(ck[k + 2], sx));
#pragma unroll
                for (int k = ND - 1; k >= 1; --k) sv = P_(A.D[k - 1][q], M_(ck[k + 1], sv));
                xn[c] = P_(A.x[q], M_(h, P_(A.v[q], M_(ck[2], sx))));
                vn[c] = P_(A.v[q], M_(h, sv));
            }
            atomicAdd(A.n_limited, 1ull);
        } else if (M < K) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const long long q = 3 * i + c, qa = 3 * ia + c;
                corrector_xv(2 * M, h, A.x[q], A.v[q], A.D[0][q], A.acc[qa], A.D[1][q], A.jerk[qa],
                             K >= 3 ? A.D[2][q] : 0.0, K >= 3 ? A.snap[qa] : 0.0, K >= 4 ? A.D[3][q] : 0.0,
                             K >= 4 ? A.crk[qa] : 0.0, xn[c], vn[c]);
            }
            atomicAdd(A.n_limited, 1ull);
        }
    }
    if (A.reject_ratio >= 2) {  // R14: the end-point criterion says the step was >= R times too long: do not take it
        const double R = (double)A.reject_ratio;
        const double hr = Q_(h, R);
        if (M_(dt_new, R) <= h && hr >= A.dt_min) {
            A.dt[i] = hr;
            atomicAdd(A.n_rejected, 1ull);
            return;
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        A.x[3 * i + c] = xn[c];
        A.v[3 * i + c] = vn[c];
    }
#pragma unroll
    for (int k = 0; k < ORDER; ++k)
#pragma unroll
        for (int c = 0; c < 3; ++c) A.D[k][3 * i + c] = dn[k][c];
    A.pot_state[i] = A.pot[ia];
    A.t[i] = t_now;
    A.dt[i] = dt_new;
}


#undef P_
#undef S_
#undef M_
#undef Q_

}  // namespace nbody
