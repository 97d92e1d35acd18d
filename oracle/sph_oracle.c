/*
 * oracle/sph_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, per-point restatement of what the hot path computes: the real
 * spherical harmonics of "Fast evaluation of spherical harmonics with
 * sphericart" (arXiv 2302.08381; cited below as P:<line of PAPER.md>), written
 * in the paper's order and notation so it can be checked against the paper by
 * eye.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code with the CUDA path.
 *
 * The file is compiled twice (oracle/__init__.py does it):
 *   -DORACLE_LONG_DOUBLE : real = 80-bit long double -> the parity reference
 *   (default)            : real = double             -> the timed CPU baseline
 *
 * Steps (DESIGN.md "Oracle" lists the readings of the paper taken here):
 *   O1  F_l^m            Eq. C1
 *   O2  u = x/r          P:108   (normalised variant only)
 *   O3  r^2
 *   O4  c_m, s_m         Eq. 9
 *   O5  Q_l^m            Eq. 7, full triangle
 *   O6  values           Eq. 5, k = l(l+1)+m
 *   O7  d/dx, d2/dxdx    Eq. 10, product rule, once and twice
 *   O8  chain rule       P:108   (plain form with the projector I - u u^T)
 *   O9  VJP              P:112   grad_xyz[a] = sum_k dsph[a,k] grad_sph[k]
 *
 * Pins: tests/test_oracle_pins.py (none of them re-types these formulas).
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real;
#define R_SQRT sqrtl
#define NAME(f) f##_ld
#else
typedef double real;
#define R_SQRT sqrt
#define NAME(f) f##_f64
#endif

#define TRI(l, m) ((l) * ((l) + 1) / 2 + (m)) /* index into an (l,m) triangle, 0<=m<=l */

/* O1. Eq. C1: F_l^0 = sqrt((2l+1)/(2 pi)), F_l^m = -F_l^{m-1}/sqrt((l+m)(l+1-m)). */
void NAME(oracle_F_table)(int l_max, real *F) {
    const real pi = (real)3.14159265358979323846264338327950288419716939937510L;
    for (int l = 0; l <= l_max; ++l) {
        F[TRI(l, 0)] = R_SQRT((real)(2 * l + 1) / (2 * pi));
        for (int m = 1; m <= l; ++m)
            F[TRI(l, m)] = -F[TRI(l, m - 1)] / R_SQRT((real)((l + m) * (l + 1 - m)));
    }
}

/* O4. Eq. 9: s_0 = 0, c_0 = 1, s_m = x s_{m-1} + y c_{m-1}, c_m = -y s_{m-1} + x c_{m-1}. */
void NAME(oracle_cs)(real x, real y, int l_max, real *c, real *s) {
    s[0] = 0;
    c[0] = 1;
    for (int m = 1; m <= l_max; ++m) {
        s[m] = x * s[m - 1] + y * c[m - 1];
        c[m] = -y * s[m - 1] + x * c[m - 1];
    }
}

/* O5. Eq. 7:
 *   Q_0^0 = 1,  Q_l^l = -(2l-1) Q_{l-1}^{l-1},  Q_l^{l-1} = (2l-1) z Q_{l-1}^{l-1},
 *   Q_l^m = [(2l-1) z Q_{l-1}^m - (l+m-1) r^2 Q_{l-2}^m] / (l-m).                          */
void NAME(oracle_Q)(real z, real r2, int l_max, real *Q) {
    Q[TRI(0, 0)] = 1;
    for (int l = 1; l <= l_max; ++l) {
        Q[TRI(l, l)] = -(real)(2 * l - 1) * Q[TRI(l - 1, l - 1)];
        Q[TRI(l, l - 1)] = (real)(2 * l - 1) * z * Q[TRI(l - 1, l - 1)];
        for (int m = 0; m <= l - 2; ++m)
            Q[TRI(l, m)] = ((real)(2 * l - 1) * z * Q[TRI(l - 1, m)] -
                            (real)(l + m - 1) * r2 * Q[TRI(l - 2, m)]) /
                           (real)(l - m);
    }
}

/* Q_l^m with the convention Q := 0 for m > l or l < 0 (used by the derivative rules). */
static real Qget(const real *Q, int l, int m) {
    if (l < 0 || m > l) return 0;
    return Q[TRI(l, m)];
}
/* c_m, s_m with negative subscripts := 0 (they only occur multiplied by m or m(m-1) = 0). */
static real get(const real *a, int m) { return m < 0 ? 0 : a[m]; }

/*
 * O3-O7 for one point: solid harmonics Ytilde = r^l Y and their Cartesian first and
 * second derivatives at (x,y,z).  sph[L], g[3][L], H[3][3][L], L = (l_max+1)^2;
 * g and H may be NULL.
 */
static void solid_point(real x, real y, real z, int l_max, const real *F, real *c, real *s, real *Q,
                        real *sph, real *g, real *H) {
    const int L = (l_max + 1) * (l_max + 1);
    const real r2 = x * x + y * y + z * z; /* O3 */
    const real inv_sqrt2 = 1 / R_SQRT((real)2);
    NAME(oracle_cs)(x, y, l_max, c, s); /* O4 */
    NAME(oracle_Q)(z, r2, l_max, Q);    /* O5 */

    for (int l = 0; l <= l_max; ++l) {
        for (int mm = -l; mm <= l; ++mm) {
            const int m = mm < 0 ? -mm : mm; /* |m| */
            const int k = l * (l + 1) + mm;  /* S1: position inside a row */
            const real Fm = F[TRI(l, m)];
            const real Qlm = Q[TRI(l, m)];
            /* A and its x,y derivatives (Eq. 10), applied once and twice */
            real A, Ax, Ay, Axx, Axy, Ayy;
            if (mm > 0) { /* cos branch, A = c_m */
                A = c[m];
                Ax = m * get(c, m - 1);
                Ay = -m * get(s, m - 1);
                Axx = m * (m - 1) * get(c, m - 2);
                Axy = -m * (m - 1) * get(s, m - 2);
                Ayy = -Axx;
            } else if (mm < 0) { /* sin branch, A = s_|m| */
                A = s[m];
                Ax = m * get(s, m - 1);
                Ay = m * get(c, m - 1);
                Axx = m * (m - 1) * get(s, m - 2);
                Axy = m * (m - 1) * get(c, m - 2);
                Ayy = -Axx;
            } else {
                A = inv_sqrt2;
                Ax = Ay = Axx = Axy = Ayy = 0;
            }
            /* O6. Eq. 5 */
            sph[k] = Fm * Qlm * A;
            if (!g) continue;

            /* O7. Eq. 10: dQ/dx = x Q_{l-1}^{m+1}, dQ/dy = y Q_{l-1}^{m+1}, dQ/dz = (l+m) Q_{l-1}^m */
            const real Q1 = Qget(Q, l - 1, m + 1);
            const real Qz = Qget(Q, l - 1, m);
            g[0 * L + k] = Fm * (x * Q1 * A + Qlm * Ax);
            g[1 * L + k] = Fm * (y * Q1 * A + Qlm * Ay);
            g[2 * L + k] = Fm * (real)(l + m) * Qz * A;
            if (!H) continue;

            /* Eq. 10 applied twice:
             *   d2Q/dx2 = Q_{l-1}^{m+1} + x^2 Q_{l-2}^{m+2},   d2Q/dxdy = x y Q_{l-2}^{m+2},
             *   d2Q/dxdz = (l+m) x Q_{l-2}^{m+1},              d2Q/dz2 = (l+m)(l+m-1) Q_{l-2}^m  */
            const real Q2 = Qget(Q, l - 2, m + 2);
            const real Qxz = Qget(Q, l - 2, m + 1);
            const real Qzz = Qget(Q, l - 2, m);
            const real lm = (real)(l + m);
            const real Hxx = Fm * ((Q1 + x * x * Q2) * A + 2 * x * Q1 * Ax + Qlm * Axx);
            const real Hyy = Fm * ((Q1 + y * y * Q2) * A + 2 * y * Q1 * Ay + Qlm * Ayy);
            const real Hxy = Fm * (x * y * Q2 * A + x * Q1 * Ay + y * Q1 * Ax + Qlm * Axy);
            const real Hxz = Fm * lm * (x * Qxz * A + Qz * Ax);
            const real Hyz = Fm * lm * (y * Qxz * A + Qz * Ay);
            const real Hzz = Fm * lm * (lm - 1) * Qzz * A;
            H[(0 * 3 + 0) * L + k] = Hxx;
            H[(1 * 3 + 1) * L + k] = Hyy;
            H[(2 * 3 + 2) * L + k] = Hzz;
            H[(0 * 3 + 1) * L + k] = H[(1 * 3 + 0) * L + k] = Hxy;
            H[(0 * 3 + 2) * L + k] = H[(2 * 3 + 0) * L + k] = Hxz;
            H[(1 * 3 + 2) * L + k] = H[(2 * 3 + 1) * L + k] = Hyz;
        }
    }
}

/*
 * The whole path for n points (SURVEY 8(b) layouts):
 *   xyz [n,3] (double; f32 inputs are widened exactly by the caller),
 *   sph [n,L], dsph [n,3,L] or NULL, ddsph [n,3,3,L] or NULL (needs dsph).
 * normalized = 0: solid harmonics r^l Y.  normalized = 1: Y on the unit
 * sphere = Ytilde(x/r) with the chain rule applied to the derivatives.
 * Returns 0, or 1 on bad arguments / allocation failure.
 */
int NAME(oracle_compute)(const double *xyz, int64_t n, int l_max, int normalized, real *sph,
                         real *dsph, real *ddsph) {
    if (n < 0 || l_max < 0 || (ddsph && !dsph) || (n > 0 && (!xyz || !sph))) return 1;
    const int L = (l_max + 1) * (l_max + 1);
    const int T = (l_max + 1) * (l_max + 2) / 2;
    real *F = (real *)malloc(sizeof(real) * T);
    if (!F) return 1;
    NAME(oracle_F_table)(l_max, F); /* O1 */
    int failed = 0;

#pragma omp parallel
    {
        real *c = (real *)malloc(sizeof(real) * (l_max + 1));
        real *s = (real *)malloc(sizeof(real) * (l_max + 1));
        real *Q = (real *)malloc(sizeof(real) * T);
        real *gt = (real *)malloc(sizeof(real) * 3 * L);
        real *Ht = (real *)malloc(sizeof(real) * 9 * L);
        if (!c || !s || !Q || !gt || !Ht) {
#pragma omp atomic write
            failed = 1;
        } else {
#pragma omp for schedule(static)
            for (int64_t i = 0; i < n; ++i) {
                real x = xyz[3 * i + 0], y = xyz[3 * i + 1], z = xyz[3 * i + 2];
                real *Yi = sph + i * L;
                real *gi = dsph ? dsph + i * 3 * L : NULL;
                real *Hi = ddsph ? ddsph + i * 9 * L : NULL;
                if (!normalized) {
                    solid_point(x, y, z, l_max, F, c, s, Q, Yi, gi, Hi);
                    continue;
                }
                /* O2. P:108: evaluate Ytilde at u = (x/r, y/r, z/r) ... */
                const real r = R_SQRT(x * x + y * y + z * z);
                const real u[3] = {x / r, y / r, z / r};
                solid_point(u[0], u[1], u[2], l_max, F, c, s, Q, Yi, dsph ? gt : NULL,
                            ddsph ? Ht : NULL);
                if (!dsph) continue;
                /* O8. ... and apply the chain rule.  du_b/dx_a = P_ab / r with P = I - u u^T, so
                 *   dY/dx_a       = sum_b P_ab gt_b / r
                 *   d2Y/dx_a dx_c = [ sum_bd P_ab P_cd Ht_bd
                 *                     - sum_b gt_b (P_ab u_c + P_ac u_b + P_bc u_a) ] / r^2          */
                real P[3][3];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) P[a][b] = (a == b ? 1 : 0) - u[a] * u[b];
                for (int k = 0; k < L; ++k) {
                    for (int a = 0; a < 3; ++a) {
                        real acc = 0;
                        for (int b = 0; b < 3; ++b) acc += P[a][b] * gt[b * L + k];
                        gi[a * L + k] = acc / r;
                    }
                    if (!ddsph) continue;
                    for (int a = 0; a < 3; ++a)
                        for (int cc = 0; cc < 3; ++cc) {
                            real acc = 0;
                            for (int b = 0; b < 3; ++b)
                                for (int d = 0; d < 3; ++d)
                                    acc += P[a][b] * P[cc][d] * Ht[(b * 3 + d) * L + k];
                            for (int b = 0; b < 3; ++b)
                                acc -= gt[b * L + k] *
                                       (P[a][b] * u[cc] + P[a][cc] * u[b] + P[b][cc] * u[a]);
                            Hi[(a * 3 + cc) * L + k] = acc / (r * r);
                        }
                }
            }
        }
        free(c);
        free(s);
        free(Q);
        free(gt);
        free(Ht);
    }
    free(F);
    return failed;
}

/* O9. P:112: the backward pass contracts the stored derivatives with the upstream gradient:
 *   grad_xyz[i,a] = sum_k dsph[i,a,k] * grad_sph[i,k].                                            */
int NAME(oracle_vjp)(const real *dsph, const real *grad_sph, int64_t n, int l_max, real *grad_xyz) {
    if (n < 0 || l_max < 0 || (n > 0 && (!dsph || !grad_sph || !grad_xyz))) return 1;
    const int L = (l_max + 1) * (l_max + 1);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            real acc = 0;
            for (int k = 0; k < L; ++k) acc += dsph[(i * 3 + a) * L + k] * grad_sph[i * L + k];
            grad_xyz[i * 3 + a] = acc;
        }
    return 0;
}

/* Pointer-argument entry points for the pins (ctypes cannot pass an 80-bit value exactly). */
void NAME(oracle_Q_p)(const real *z, const real *r2, int l_max, real *Q) {
    NAME(oracle_Q)(*z, *r2, l_max, Q);
}
void NAME(oracle_cs_p)(const real *x, const real *y, int l_max, real *c, real *s) {
    NAME(oracle_cs)(*x, *y, l_max, c, s);
}

/* Number of OpenMP threads the loops above use (1 when built without -fopenmp). */
#ifdef _OPENMP
#include <omp.h>
int NAME(oracle_num_threads)(void) { return omp_get_max_threads(); }
#else
int NAME(oracle_num_threads)(void) { return 1; }
#endif
