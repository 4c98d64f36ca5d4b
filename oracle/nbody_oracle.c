/*
 * oracle/nbody_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the hot path of the block-time-step Hermite
 * direct N-body method benchmarked in arXiv:1312.1789 (PAPER.md:15 abstract:
 * "individual hierarchically block time-steps with the high (4th, 6th and 8th)
 * order Hermite integration schemes"; section 2; Fig. 1
 * "mixed (fp32 + fp64) precision").  The paper prints no formula; the method
 * statement followed here is SURVEY.md section 8(c) (items c-1 ... c-11), which
 * restates the textbook Hermite scheme.  Every function cites its item.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code with
 * paper_1312_1789_b200/csrc (the CUDA path) and neither includes the other.
 *
 * Everything is IEEE fp64, compiled with -O2 -ffp-contract=off (no FMA
 * contraction, no -ffast-math), operations in the order written, so that the
 * predictor / corrector / time-step results are reproducible bit for bit.
 * OpenMP parallelises over particles only; each particle's arithmetic is serial.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): worked example W3 (40-digit
 * mpmath differentiation of the softened acceleration along cubic orbits),
 * mpmath brute force on N <= 8, circular two-body closed form, Sum m a = 0 ...
 * Sum m c = 0, Plummer W -> -1/2, polynomial exactness of predictor /
 * corrector / interpolated derivatives, exponential dt pin eta/lambda,
 * quantisation against exact rational arithmetic (ties and one-ulp near-ties
 * included), the c-8b mean-crackle criterion against its closed form for
 * a(t) = a0 e^(lambda t) (50-digit mpmath), convergence slopes 4/6/8 (table B2),
 * Kepler closure, energy conservation; oracle_nearest (c-17) on a chain with
 * closed-form neighbours, against an fp64 brute force, on ties and on a
 * difference only fp64 resolves.  Parity unpinned: nothing.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------ *
 * c-5  Predictor.  tau = t_now - t_i ; D_k = a^(k)(t_i), k = 0 .. p-3.
 *   x_p = x + v tau + Sum_k D_k tau^(k+2)/(k+2)!
 *   v_p = v +         Sum_k D_k tau^(k+1)/(k+1)!
 *   a_p =             Sum_k D_k tau^k/k!              (p >= 6)
 *   j_p =             Sum_{k>=1} D_k tau^(k-1)/(k-1)! (p == 8)
 * Horner, innermost term first, with c_k = tau / k (IEEE division).
 * D[k] points to a^(k) as [n][3]; outputs [n][3] (ap / jp may be NULL).
 * ------------------------------------------------------------------------ */
void oracle_predict(int64_t n, double t_now, int order,
                    const double *t, const double *x, const double *v,
                    const double *const *D,
                    double *xp, double *vp, double *ap, double *jp)
{
    const int nd = order - 2;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double tau = t_now - t[i];
        double c[9];
        for (int k = 1; k <= 8; ++k) c[k] = tau / (double)k;
        for (int d = 0; d < 3; ++d) {
            const int64_t q = 3 * i + d;
            double s;
            /* position */
            s = D[nd - 1][q];
            for (int k = nd - 1; k >= 1; --k) s = D[k - 1][q] + c[k + 2] * s;
            xp[q] = x[q] + tau * (v[q] + c[2] * s);
            /* velocity */
            s = D[nd - 1][q];
            for (int k = nd - 1; k >= 1; --k) s = D[k - 1][q] + c[k + 1] * s;
            vp[q] = v[q] + tau * s;
            /* acceleration */
            if (order >= 6 && ap) {
                s = D[nd - 1][q];
                for (int k = nd - 1; k >= 1; --k) s = D[k - 1][q] + c[k] * s;
                ap[q] = s;
            }
            /* jerk */
            if (order >= 8 && jp) {
                s = D[nd - 1][q];
                for (int k = nd - 1; k >= 2; --k) s = D[k - 1][q] + c[k - 1] * s;
                jp[q] = s;
            }
        }
    }
}

/* ------------------------------------------------------------------------ *
 * c-1 .. c-4  Force with derivatives: the plain definition, summed over all
 * j != i (excluded BY INDEX, c-2), G = 1, pot negative (c-3).  All inputs are
 * the predicted values at the block time; the i-particle is one of them (c-4).
 *   r = x_j - x_i, v = v_j - v_i, a = a_j - a_i (p>=6), j = j_j - j_i (p=8)
 *   s2 = r.r + eps2 ; q = m_j / s2^(3/2)
 *   alpha = (r.v)/s2
 *   beta  = (v.v + r.a)/s2 + alpha^2
 *   gamma = (3 v.a + r.j)/s2 + alpha (3 beta - 4 alpha^2)
 *   A = q r ; J = q v - 3 alpha A ; S = q a - 6 alpha J - 3 beta A
 *   C = q j - 9 alpha S - 9 beta J - 3 gamma A ; pot = - Sum m_j / sqrt(s2)
 * order 4: acc, jerk, pot ; 6: + snap ; 8: + crackle.  Outputs in active-list
 * order, [n_act][3] / [n_act].  ap may be NULL for order 4, jp for order < 8.
 * ------------------------------------------------------------------------ */
void oracle_force(int64_t n, const double *m,
                  const double *xp, const double *vp, const double *ap, const double *jp,
                  const int32_t *active_idx, int64_t n_act, int order, double eps2,
                  double *acc, double *jerk, double *snap, double *crackle, double *pot)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t ia = 0; ia < n_act; ++ia) {
        const int64_t i = active_idx[ia];
        double A[3] = {0, 0, 0}, J[3] = {0, 0, 0}, S[3] = {0, 0, 0}, C[3] = {0, 0, 0}, P = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double r[3], v[3], a[3] = {0, 0, 0}, jj[3] = {0, 0, 0};
            for (int d = 0; d < 3; ++d) {
                r[d] = xp[3 * j + d] - xp[3 * i + d];
                v[d] = vp[3 * j + d] - vp[3 * i + d];
                if (order >= 6) a[d] = ap[3 * j + d] - ap[3 * i + d];
                if (order >= 8) jj[d] = jp[3 * j + d] - jp[3 * i + d];
            }
            const double s2 = (r[0] * r[0] + r[1] * r[1] + r[2] * r[2]) + eps2;
            const double rinv = 1.0 / sqrt(s2);
            const double q = m[j] * rinv * rinv * rinv;
            const double rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
            const double alpha = rv / s2;
            double Ap[3], Jp[3], Sp[3];
            P -= m[j] * rinv;
            for (int d = 0; d < 3; ++d) {
                Ap[d] = q * r[d];
                Jp[d] = q * v[d] - 3.0 * alpha * Ap[d];
                A[d] += Ap[d];
                J[d] += Jp[d];
            }
            if (order >= 6) {
                const double vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
                const double ra = r[0] * a[0] + r[1] * a[1] + r[2] * a[2];
                const double beta = (vv + ra) / s2 + alpha * alpha;
                for (int d = 0; d < 3; ++d) {
                    Sp[d] = q * a[d] - 6.0 * alpha * Jp[d] - 3.0 * beta * Ap[d];
                    S[d] += Sp[d];
                }
                if (order >= 8) {
                    const double va = v[0] * a[0] + v[1] * a[1] + v[2] * a[2];
                    const double rj = r[0] * jj[0] + r[1] * jj[1] + r[2] * jj[2];
                    const double gamma = (3.0 * va + rj) / s2 + alpha * (3.0 * beta - 4.0 * alpha * alpha);
                    for (int d = 0; d < 3; ++d)
                        C[d] += q * jj[d] - 9.0 * alpha * Sp[d] - 9.0 * beta * Jp[d] - 3.0 * gamma * Ap[d];
                }
            }
        }
        for (int d = 0; d < 3; ++d) {
            acc[3 * ia + d] = A[d];
            jerk[3 * ia + d] = J[d];
            if (order >= 6 && snap) snap[3 * ia + d] = S[d];
            if (order >= 8 && crackle) crackle[3 * ia + d] = C[d];
        }
        pot[ia] = P;
    }
}

/* ------------------------------------------------------------------------ *
 * c-16  Conditioning of the sums of c-1 (diagnostic for the parity reports, SURVEY.md
 * 7.2 H5): for each active i the sums over j != i of the Euclidean NORMS of
 * the pair terms, abs_k[ia] = Sum_j |term^(k)_ij| (k = 0 acc, 1 jerk, 2 snap,
 * 3 crackle; entries above the order are left untouched), so that
 * kappa_k = abs_k / |Sum_j term^(k)_ij| >= 1 measures the cancellation in the
 * sum a mixed-precision evaluation has to survive.  Same pair formulas as
 * oracle_force (c-1), same exclusion by index.
 * ------------------------------------------------------------------------ */
void oracle_force_abs(int64_t n, const double *m,
                      const double *xp, const double *vp, const double *ap, const double *jp,
                      const int32_t *active_idx, int64_t n_act, int order, double eps2,
                      double *abs_acc, double *abs_jerk, double *abs_snap, double *abs_crackle)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t ia = 0; ia < n_act; ++ia) {
        const int64_t i = active_idx[ia];
        double sA = 0.0, sJ = 0.0, sS = 0.0, sC = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double r[3], v[3], a[3] = {0, 0, 0}, jj[3] = {0, 0, 0};
            for (int d = 0; d < 3; ++d) {
                r[d] = xp[3 * j + d] - xp[3 * i + d];
                v[d] = vp[3 * j + d] - vp[3 * i + d];
                if (order >= 6) a[d] = ap[3 * j + d] - ap[3 * i + d];
                if (order >= 8) jj[d] = jp[3 * j + d] - jp[3 * i + d];
            }
            const double s2 = (r[0] * r[0] + r[1] * r[1] + r[2] * r[2]) + eps2;
            const double rinv = 1.0 / sqrt(s2);
            const double q = m[j] * rinv * rinv * rinv;
            const double alpha = (r[0] * v[0] + r[1] * v[1] + r[2] * v[2]) / s2;
            double Ap[3], Jp[3], Sp[3], Cp[3];
            for (int d = 0; d < 3; ++d) {
                Ap[d] = q * r[d];
                Jp[d] = q * v[d] - 3.0 * alpha * Ap[d];
            }
            sA += sqrt((Ap[0] * Ap[0] + Ap[1] * Ap[1]) + Ap[2] * Ap[2]);
            sJ += sqrt((Jp[0] * Jp[0] + Jp[1] * Jp[1]) + Jp[2] * Jp[2]);
            if (order >= 6) {
                const double vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
                const double ra = r[0] * a[0] + r[1] * a[1] + r[2] * a[2];
                const double beta = (vv + ra) / s2 + alpha * alpha;
                for (int d = 0; d < 3; ++d) Sp[d] = q * a[d] - 6.0 * alpha * Jp[d] - 3.0 * beta * Ap[d];
                sS += sqrt((Sp[0] * Sp[0] + Sp[1] * Sp[1]) + Sp[2] * Sp[2]);
                if (order >= 8) {
                    const double va = v[0] * a[0] + v[1] * a[1] + v[2] * a[2];
                    const double rj = r[0] * jj[0] + r[1] * jj[1] + r[2] * jj[2];
                    const double gamma = (3.0 * va + rj) / s2 + alpha * (3.0 * beta - 4.0 * alpha * alpha);
                    for (int d = 0; d < 3; ++d)
                        Cp[d] = q * jj[d] - 9.0 * alpha * Sp[d] - 9.0 * beta * Jp[d] - 3.0 * gamma * Ap[d];
                    sC += sqrt((Cp[0] * Cp[0] + Cp[1] * Cp[1]) + Cp[2] * Cp[2]);
                }
            }
        }
        abs_acc[ia] = sA;
        abs_jerk[ia] = sJ;
        if (order >= 6 && abs_snap) abs_snap[ia] = sS;
        if (order >= 8 && abs_crackle) abs_crackle[ia] = sC;
    }
}

/* Euclidean norm, fixed order ((x^2 + y^2) + z^2) then IEEE sqrt. */
/* ------------------------------------------------------------------------
 * c-17 (this build's reading R16 of SURVEY 8(f) N4 "nearest-neighbour output";
 * not in PAPER.md, which names the Ahmad-Cohen neighbour scheme of its second
 * code only): for every active particle the index of the nearest
 * OTHER particle (excluded by index, as in c-1) at the predicted positions, and
 * the squared distance to it.  The distance decides an integer (the argmin), so
 * its precision is fixed and is the force kernel's (c-12): each component of
 * the difference is formed in fp64 and rounded to fp32, and
 *     r2 = fma(dz, dz, fma(dy, dy, dx * dx))      in fp32, in this order;
 * ties go to the lowest index.  n == 1: index -1, r2 = +inf.
 * nn_r2 holds the fp32 value (as a double).
 * ------------------------------------------------------------------------ */
void oracle_nearest(int64_t n, const double *xp, const int32_t *active_idx, int64_t n_act,
                    int32_t *nn_idx, double *nn_r2)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t ia = 0; ia < n_act; ++ia) {
        const int64_t i = active_idx[ia];
        float best = INFINITY;
        int32_t who = -1;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const float dx = (float)(xp[3 * j + 0] - xp[3 * i + 0]);
            const float dy = (float)(xp[3 * j + 1] - xp[3 * i + 1]);
            const float dz = (float)(xp[3 * j + 2] - xp[3 * i + 2]);
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            if (r2 < best) {
                best = r2;
                who = (int32_t)j;
            }
        }
        nn_idx[ia] = who;
        nn_r2[ia] = (double)best;
    }
}

static double nrm3(const double *a)
{
    return sqrt((a[0] * a[0] + a[1] * a[1]) + a[2] * a[2]);
}

/* Exact 2^k for k in the normal range. */
static double pow2i(int k)
{
    return ldexp(1.0, k);
}

/* exact integer log2 of a power of two (returns 0 and sets *ok = 0 otherwise) */
static int log2_exact(double x, int *ok)
{
    int e;
    double f = frexp(x, &e); /* x = f 2^e, f in [0.5,1) */
    *ok = (x > 0.0 && f == 0.5);
    return e - 1;
}

/* ------------------------------------------------------------------------ *
 * c-9 step 1.  Largest integer k with  Ap * 2^(k q) <= A1 * E  (i.e. 2^k <=
 * eta (A1/Ap)^(1/q)), searched downwards from k_hi; returns k_lo - 1 when no
 * k in [k_lo, k_hi] satisfies it (NaN lands here: comparisons are false).
 * Multiplying by a power of two is exact, so this is floor(log2 dt_crit)
 * without pow/log.
 * ------------------------------------------------------------------------ */
static int floor_log2_ratio(double A1, double Ap, double E, int q, int k_lo, int k_hi)
{
    const double rhs = A1 * E;
    int k = k_hi;
    while (k >= k_lo && !(Ap * pow2i(k * q) <= rhs)) --k;
    return k;
}

/* ------------------------------------------------------------------------ *
 * c-8 + c-9  New block time step of one particle.
 *   A1 = A^(1) = sqrt(|a||a2| + |j|^2),  Ap = A^(p-2) = sqrt(|a^(p-3)||a^(p-1)| + |a^(p-2)|^2)
 *   dt_crit = eta (A1/Ap)^(1/(p-3))
 *   1. dt_q = 2^floor(log2 dt_crit)
 *   2. dt_new = min(dt_q, 2 dt_old)
 *   3. dt_new == 2 dt_old and fmod(t1, dt_new) != 0  =>  dt_new = dt_old
 *   4. dt_new = min(dt_new, dt_max) ; dt_new < dt_min => dt_min
 * d[k] = pointer to the 3-vector a^(k)(t1), k = 0 .. p-1.
 * ------------------------------------------------------------------------ */
double oracle_new_dt(int order, const double *const *d, double t1, double dt_old,
                     double eta, double dt_min, double dt_max)
{
    const int p = order, q = p - 3;
    int ok;
    const int k_min = log2_exact(dt_min, &ok);
    const int k_max = log2_exact(dt_max, &ok);
    const double n0 = nrm3(d[0]), n1 = nrm3(d[1]), n2 = nrm3(d[2]);
    const double m3 = nrm3(d[p - 3]), m2 = nrm3(d[p - 2]), m1 = nrm3(d[p - 1]);
    const double A1 = sqrt(n0 * n2 + n1 * n1);
    const double Ap = sqrt(m3 * m1 + m2 * m2);
    double E = 1.0;
    for (int k = 0; k < q; ++k) E = E * eta;
    /* step 1 */
    const int k = floor_log2_ratio(A1, Ap, E, q, k_min - 1, k_max + 1);
    double dt_new = pow2i(k);
    /* step 2 */
    if (dt_new > 2.0 * dt_old) dt_new = 2.0 * dt_old;
    /* step 3 */
    if (dt_new == 2.0 * dt_old && fmod(t1, dt_new) != 0.0) dt_new = dt_old;
    /* step 4 */
    if (dt_new > dt_max) dt_new = dt_max;
    if (dt_new < dt_min) dt_new = dt_min;
    return dt_new;
}

/* ------------------------------------------------------------------------ *
 * c-10  Start-up step: dt = 2^floor(log2(eta_s |a|/|j|)) clamped to
 * [dt_min, dt_max]; |j| == 0 => dt_max.
 * ------------------------------------------------------------------------ */
void oracle_initial_dt(int64_t n, const double *acc, const double *jerk,
                       double eta_s, double dt_min, double dt_max, double *dt)
{
    int ok;
    const int k_min = log2_exact(dt_min, &ok);
    const int k_max = log2_exact(dt_max, &ok);
    for (int64_t i = 0; i < n; ++i) {
        const double na = nrm3(acc + 3 * i), nj = nrm3(jerk + 3 * i);
        const int k = floor_log2_ratio(na, nj, eta_s, 1, k_min - 1, k_max + 1);
        double d = pow2i(k);
        if (d > dt_max) d = dt_max;
        if (d < dt_min) d = dt_min;
        dt[i] = d;
    }
}

/* c-6 restated for one component at a chosen order m2 = 2, 4, 6, 8 (m2 = 2 is the trapezoid rule), in the operation
 * order of oracle_correct's own lines; used by the order limiter c-6b. */
static void corrector_xv(int m2, double h, double x0, double v0, double a0, double a1, double j0, double j1,
                         double s0, double s1, double c0, double c1, double *x1, double *v1)
{
    const double h2 = h * h, h3 = h2 * h, h4 = h3 * h;
    double v, x;
    if (m2 == 2) {
        v = v0 + (h / 2.0) * (a0 + a1);
        x = x0 + (h / 2.0) * (v0 + v);
    } else if (m2 == 4) {
        v = v0 + ((h / 2.0) * (a0 + a1) + (h2 / 12.0) * (j0 - j1));
        x = x0 + ((h / 2.0) * (v0 + v) + (h2 / 12.0) * (a0 - a1));
    } else if (m2 == 6) {
        v = v0 + ((h / 2.0) * (a0 + a1) + ((h2 / 10.0) * (j0 - j1) + (h3 / 120.0) * (s0 + s1)));
        x = x0 + ((h / 2.0) * (v0 + v) + ((h2 / 10.0) * (a0 - a1) + (h3 / 120.0) * (j0 + j1)));
    } else {
        v = v0 + ((h / 2.0) * (a0 + a1) + (((3.0 * h2) / 28.0) * (j0 - j1) + ((h3 / 84.0) * (s0 + s1) + (h4 / 1680.0) * (c0 - c1))));
        x = x0 + ((h / 2.0) * (v0 + v) + (((3.0 * h2) / 28.0) * (a0 - a1) + ((h3 / 84.0) * (j0 + j1) + (h4 / 1680.0) * (s0 - s1))));
    }
    *x1 = x;
    *v1 = v;
}

/* ------------------------------------------------------------------------ *
 * c-6 + c-7 + c-8 + c-9  Corrector and new time step for the active particles.
 * h = dt_i ; 0 = stored values at t0 = t_i ; 1 = force-call values at t1 = t_now.
 *
 * c-6 (compact two-point Hermite, P(EC)^1; `variant` 0).  variant 1 selects the
 * older 4th-order double-integral form x1 = x0 + h v0 + h^2/2 a0 + h^3/6 j0 +
 * h^4/24 a2(t0) + h^5/120 a3 (order 4 only; used by the tests to tell the two
 * readings apart, SURVEY.md c-6 "Ambiguity").
 *   p=4: v1 = v0 + h/2 (a0+a1) + h^2/12 (j0-j1)
 *        x1 = x0 + h/2 (v0+v1) + h^2/12 (a0-a1)
 *   p=6: v1 = v0 + h/2 (a0+a1) + h^2/10 (j0-j1) + h^3/120 (s0+s1)
 *        x1 = x0 + h/2 (v0+v1) + h^2/10 (a0-a1) + h^3/120 (j0+j1)
 *   p=8: v1 = v0 + h/2 (a0+a1) + 3h^2/28 (j0-j1) + h^3/84 (s0+s1) + h^4/1680 (c0-c1)
 *        x1 = x0 + h/2 (v0+v1) + 3h^2/28 (a0-a1) + h^3/84 (j0+j1) + h^4/1680 (s0-s1)
 * c-7 interpolated a^(K..2K-1)(t1), Delta = a0 - a1 (formulas below).
 *
 * c-8b: `crit_order` selects the criterion order pc.  0 = automatic, the same meaning as the CUDA library's
 * "dt_criterion_order" option value 0 (include/nbody.h): pc = p for p = 4, pc = 4 for p >= 6.  4 | 6 | 8 = pc =
 * min(p, value), so value = p is the order-p criterion of c-8.  The order-pc criterion is evaluated on
 * a^(0..pc-1)(t1).  For p = 6, pc = 4 the fourth entry is the mean crackle of the step (s1 - s0)/h instead of the
 * interpolated a3 (whose force-noise amplification is 60/h^3), so that, like p = 8, pc = 4, only derivatives the force
 * call computes directly enter the step decision.  Added after the CUDA path showed that with fp32 pair arithmetic (c-12) the interpolated
 * a^(K..2K-1) of p >= 6 are rounding-noise dominated at small h and the order-p criterion collapses dt.
 *
 * c-9b (R14, a reading added in round 2; the paper is silent, PAPER.md:15 says only "individual
 * hierarchically block time-steps"): a-posteriori step rejection.  reject_ratio R = 0 switches it off (the textbook
 * scheme); R = 2^r >= 2: if the criterion evaluated at the END of the step asks for dt_new <= h/R (the step was at
 * least R times longer than the scheme now thinks it should have been: an encounter the start-of-step criterion
 * could not see) and h/R >= dt_min, the step is NOT taken: x, v, D, pot_state and t of the particle keep their
 * values at t0 and only dt := h/R is written.  The particle is then due at t0 + h/R, which lies BEFORE the current
 * block time: the scheduler (c-11, min over t + dt) picks it next and the other particles are predicted back to
 * that time with their own polynomials.  *n_rejected (may be NULL) is incremented per rejection.
 *
 * c-6b (R15, a reading added in round 2; the paper is silent): corrector order limiter, `limit_order` != 0.
 * The velocity line of c-6 is a sum of K = p/2 quadrature terms T_1 = h/2 (a0+a1), T_2 = w2 (j0-j1), T_3 = w3 (s0+s1),
 * T_4 = w4 (c0-c1) (w_k = the order-p coefficients above).  On a smooth step their norms fall off like (h/tau)^k; when
 * an encounter sits on an end point they GROW (the end-point derivatives m v^k / r^(k+2) times h^(k+1)), and summing
 * them is summing a divergent series.  Rule: M = the number of leading terms whose norms are non-increasing
 * (|T_2| <= |T_1|, |T_3| <= |T_2|, ...; 1 <= M <= K); if M < K, x1 and v1 of this particle are taken from the
 * corrector of order 2M instead (M = 1: trapezoid).  One level below: if already the first end-point correction
 * U_1 = h/2 (a1 - a0) is larger than U_0 = h a0 (the end-point acceleration is a spike: |a1 - a0| > 2 |a0|), M = 0 and
 * x1, v1 are the particle's own Taylor prediction (c-5 in fp64): the end point is not used at all.  Everything else of
 * the step -- stored derivatives, criterion, new dt -- is unchanged.  *n_limited (may be NULL) counts the limited steps.
 *
 * State arrays (in/out, [n][3] unless noted): t[n], dt[n], x, v, D[k] = a^(k)
 * for k = 0..p-1, pot_state[n].  Force arrays in active-list order [n_act][3].
 * ------------------------------------------------------------------------ */
void oracle_correct(const int32_t *active_idx, int64_t n_act, int order,
                    double t_now, double eta, double dt_min, double dt_max,
                    double *t, double *dt, double *x, double *v, double *const *D,
                    double *pot_state,
                    const double *acc, const double *jerk, const double *snap,
                    const double *crackle, const double *pot, int variant, int crit_order,
                    int reject_ratio, int64_t *n_rejected, int limit_order, int64_t *n_limited)
{
    const int p = order;
    /* c-8b (R8b): the criterion may be evaluated on the lowest pc <= p derivatives only.
     * crit_order 0 = automatic (pc = 4 for p >= 6, else p); 4 | 6 | 8 = min(p, value); value = p is c-8.
     * pc = 4 is Aarseth's formula on a, j, a2, a3. */
    const int pc = (crit_order == 4 || crit_order == 6 || crit_order == 8)
                       ? (crit_order < p ? crit_order : p)
                       : (p >= 6 ? 4 : p);
    int64_t rejected = 0, limited = 0;
#pragma omp parallel for schedule(static) reduction(+ : rejected, limited)
    for (int64_t ia = 0; ia < n_act; ++ia) {
        const int64_t i = active_idx[ia];
        const double h = dt[i];
        const double h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h, h6 = h5 * h, h7 = h6 * h;
        double dnew[8][3], xnew[3], vnew[3];
        double cbar[3] = {0.0, 0.0, 0.0}; /* c-8b, p = 6: mean crackle over the step, (s1 - s0)/h */
        for (int c = 0; c < 3; ++c) {
            const int64_t q = 3 * i + c, qa = 3 * ia + c;
            const double x0 = x[q], v0 = v[q];
            const double a0 = D[0][q], j0 = D[1][q];
            const double a1 = acc[qa], j1 = jerk[qa];
            const double dl = a0 - a1;
            double v1, x1;
            if (p == 4) {
                v1 = v0 + ((h / 2.0) * (a0 + a1) + (h2 / 12.0) * (j0 - j1));
                const double A2 = (2.0 * ((3.0 * dl + h * j0) + (2.0 * h) * j1)) / h2;
                const double A3 = (6.0 * ((2.0 * dl + h * j0) + h * j1)) / h3;
                if (variant == 0) {
                    x1 = x0 + ((h / 2.0) * (v0 + v1) + (h2 / 12.0) * (a0 - a1));
                } else {
                    const double A2_0 = A2 - h * A3; /* a2 at t0 */
                    x1 = x0 + h * v0 + (h2 / 2.0) * a0 + (h3 / 6.0) * j0 + (h4 / 24.0) * A2_0 + (h5 / 120.0) * A3;
                }
                dnew[0][c] = a1; dnew[1][c] = j1; dnew[2][c] = A2; dnew[3][c] = A3;
            } else if (p == 6) {
                const double s0 = D[2][q], s1 = snap[qa];
                v1 = v0 + ((h / 2.0) * (a0 + a1) + ((h2 / 10.0) * (j0 - j1) + (h3 / 120.0) * (s0 + s1)));
                x1 = x0 + ((h / 2.0) * (v0 + v1) + ((h2 / 10.0) * (a0 - a1) + (h3 / 120.0) * (j0 + j1)));
                /* a3 = -3 (20D + 8h j0 + 12h j1 + h^2 s0 - 3h^2 s1)/h^3 */
                const double A3 = (-3.0 * ((((20.0 * dl + (8.0 * h) * j0) + (12.0 * h) * j1) + h2 * s0) - (3.0 * h2) * s1)) / h3;
                /* a4 = -12 (30D + 14h j0 + 16h j1 + 2h^2 s0 - 3h^2 s1)/h^4 */
                const double A4 = (-12.0 * ((((30.0 * dl + (14.0 * h) * j0) + (16.0 * h) * j1) + (2.0 * h2) * s0) - (3.0 * h2) * s1)) / h4;
                /* a5 = -60 (12D + 6h j0 + 6h j1 + h^2 s0 - h^2 s1)/h^5 */
                const double A5 = (-60.0 * ((((12.0 * dl + (6.0 * h) * j0) + (6.0 * h) * j1) + h2 * s0) - h2 * s1)) / h5;
                dnew[0][c] = a1; dnew[1][c] = j1; dnew[2][c] = s1;
                dnew[3][c] = A3; dnew[4][c] = A4; dnew[5][c] = A5;
                cbar[c] = (s1 - s0) / h;
            } else {
                const double s0 = D[2][q], s1 = snap[qa];
                const double c0 = D[3][q], c1 = crackle[qa];
                v1 = v0 + ((h / 2.0) * (a0 + a1) + (((3.0 * h2) / 28.0) * (j0 - j1) + ((h3 / 84.0) * (s0 + s1) + (h4 / 1680.0) * (c0 - c1))));
                x1 = x0 + ((h / 2.0) * (v0 + v1) + (((3.0 * h2) / 28.0) * (a0 - a1) + ((h3 / 84.0) * (j0 + j1) + (h4 / 1680.0) * (s0 - s1))));
                /* a4 =   4 (210D +  90h j0 + 120h j1 + 15h^2 s0 - 30h^2 s1 +  h^3 c0 + 4h^3 c1)/h^4 */
                const double A4 = (4.0 * ((((((210.0 * dl + (90.0 * h) * j0) + (120.0 * h) * j1) + (15.0 * h2) * s0) - (30.0 * h2) * s1) + h3 * c0) + (4.0 * h3) * c1)) / h4;
                /* a5 =  60 (168D +  78h j0 +  90h j1 + 14h^2 s0 - 20h^2 s1 +  h^3 c0 + 2h^3 c1)/h^5 */
                const double A5 = (60.0 * ((((((168.0 * dl + (78.0 * h) * j0) + (90.0 * h) * j1) + (14.0 * h2) * s0) - (20.0 * h2) * s1) + h3 * c0) + (2.0 * h3) * c1)) / h5;
                /* a6 = 120 (420D + 204h j0 + 216h j1 + 39h^2 s0 - 45h^2 s1 + 3h^3 c0 + 4h^3 c1)/h^6 */
                const double A6 = (120.0 * ((((((420.0 * dl + (204.0 * h) * j0) + (216.0 * h) * j1) + (39.0 * h2) * s0) - (45.0 * h2) * s1) + (3.0 * h3) * c0) + (4.0 * h3) * c1)) / h6;
                /* a7 = 840 (120D +  60h j0 +  60h j1 + 12h^2 s0 - 12h^2 s1 +  h^3 c0 +  h^3 c1)/h^7 */
                const double A7 = (840.0 * ((((((120.0 * dl + (60.0 * h) * j0) + (60.0 * h) * j1) + (12.0 * h2) * s0) - (12.0 * h2) * s1) + h3 * c0) + h3 * c1)) / h7;
                dnew[0][c] = a1; dnew[1][c] = j1; dnew[2][c] = s1; dnew[3][c] = c1;
                dnew[4][c] = A4; dnew[5][c] = A5; dnew[6][c] = A6; dnew[7][c] = A7;
            }
            xnew[c] = x1;
            vnew[c] = v1;
        }
        if (limit_order && variant == 0) { /* c-6b */
            const int K = p / 2;
            const double w[4] = {h / 2.0, p == 4 ? h2 / 12.0 : p == 6 ? h2 / 10.0 : (3.0 * h2) / 28.0,
                                 p == 6 ? h3 / 120.0 : h3 / 84.0, h4 / 1680.0};
            double T[4][3];
            for (int c = 0; c < 3; ++c) {
                const int64_t q = 3 * i + c, qa = 3 * ia + c;
                T[0][c] = w[0] * (D[0][q] + acc[qa]);
                T[1][c] = w[1] * (D[1][q] - jerk[qa]);
                T[2][c] = K >= 3 ? w[2] * (D[2][q] + snap[qa]) : 0.0;
                T[3][c] = K >= 4 ? w[3] * (D[3][q] - crackle[qa]) : 0.0;
            }
            /* level 0: the first end-point correction U_1 = h/2 (a1 - a0) against U_0 = h a0 */
            double U0[3], U1[3];
            for (int c = 0; c < 3; ++c) {
                U0[c] = h * D[0][3 * i + c];
                U1[c] = w[0] * (acc[3 * ia + c] - D[0][3 * i + c]);
            }
            int M = nrm3(U1) <= nrm3(U0) ? 1 : 0;
            while (M >= 1 && M < K && nrm3(T[M]) <= nrm3(T[M - 1])) ++M;
            if (M == 0) { /* the end point is not to be trusted at all: the particle's own Taylor prediction (c-5, fp64) */
                const int nd = p - 2;
                double ck[9];
                for (int k = 1; k <= 8; ++k) ck[k] = h / (double)k;
                for (int c = 0; c < 3; ++c) {
                    const int64_t q = 3 * i + c;
                    double sx = D[nd - 1][q], sv = D[nd - 1][q];
                    for (int k = nd - 1; k >= 1; --k) sx = D[k - 1][q] + ck[k + 2] * sx;
                    for (int k = nd - 1; k >= 1; --k) sv = D[k - 1][q] + ck[k + 1] * sv;
                    xnew[c] = x[q] + h * (v[q] + ck[2] * sx);
                    vnew[c] = v[q] + h * sv;
                }
                limited += 1;
            } else if (M < K) {
                for (int c = 0; c < 3; ++c) {
                    const int64_t q = 3 * i + c, qa = 3 * ia + c;
                    corrector_xv(2 * M, h, x[q], v[q], D[0][q], acc[qa], D[1][q], jerk[qa],
                                 K >= 3 ? D[2][q] : 0.0, K >= 3 ? snap[qa] : 0.0,
                                 K >= 4 ? D[3][q] : 0.0, K >= 4 ? crackle[qa] : 0.0, &xnew[c], &vnew[c]);
                }
                limited += 1;
            }
        }
        const double *dp[8];
        for (int k = 0; k < p; ++k) dp[k] = dnew[k];
        if (p == 6 && pc == 4) dp[3] = cbar; /* only directly computed derivatives enter the criterion */
        const double dt_new = oracle_new_dt(pc, dp, t_now, h, eta, dt_min, dt_max);
        if (reject_ratio >= 2 && dt_new * (double)reject_ratio <= h && h / (double)reject_ratio >= dt_min) {
            dt[i] = h / (double)reject_ratio; /* c-9b: the step is not taken; everything else stays at t0 */
            rejected += 1;
            continue;
        }
        for (int c = 0; c < 3; ++c) {
            x[3 * i + c] = xnew[c];
            v[3 * i + c] = vnew[c];
        }
        for (int k = 0; k < p; ++k)
            for (int c = 0; c < 3; ++c) D[k][3 * i + c] = dnew[k][c];
        pot_state[i] = pot[ia];
        t[i] = t_now;
        dt[i] = dt_new;
    }
    if (n_rejected) *n_rejected += rejected;
    if (n_limited) *n_limited += limited;
}

/* ------------------------------------------------------------------------ *
 * c-11 / a-1  Block selection: t_next = min_i (t_i + dt_i) (exact for dyadic
 * values); active = { i : t_i + dt_i == t_next }, ascending.  Returns n_act.
 * ------------------------------------------------------------------------ */
int64_t oracle_next_block(int64_t n, const double *t, const double *dt,
                          double *t_next_out, int32_t *active_idx)
{
    double t_next = INFINITY;
    for (int64_t i = 0; i < n; ++i) {
        const double s = t[i] + dt[i];
        if (s < t_next) t_next = s;
    }
    int64_t n_act = 0;
    for (int64_t i = 0; i < n; ++i)
        if (t[i] + dt[i] == t_next) active_idx[n_act++] = (int32_t)i;
    *t_next_out = t_next;
    return n_act;
}

/* c-11  Energy: E = Sum 1/2 m |v|^2 + 1/2 Sum m pot. */
void oracle_energy(int64_t n, const double *m, const double *v, const double *pot,
                   double *kin_out, double *pot_out)
{
    double K = 0.0, W = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        K += 0.5 * m[i] * ((v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1]) + v[3 * i + 2] * v[3 * i + 2]);
        W += 0.5 * m[i] * pot[i];
    }
    *kin_out = K;
    *pot_out = W;
}
