// Arithmetic core of the CUDA path: the paper's Cartesian scheme with folded prefactors.
// (P:n = line n of PAPER.md, arXiv 2302.08381.)  __host__ __device__ so that a CPU harness can
// exercise exactly this code; it shares nothing with oracle/.
//
//   Ytilde_l^m = Qt_l^|m| * { s_|m| | 1/sqrt2 | c_m }                 Eq. 5, F folded
//   c_m + i s_m = (x + i y)^m                                         Eq. 9, B2
//   Qt_l^m = A z Qt_{l-1}^m - B r^2 Qt_{l-2}^m                        Eq. 7, F folded
//   d/dx, d/dy, d/dz and second derivatives                           Eq. 10, once / twice
//   normalised: evaluate at u = x/r, then
//       grad Y   = (g - l Y u) / r
//       hess Y   = (H - l (u g^T + g u^T) + l(l+2) Y u u^T - l Y I) / r^2
//     (the chain rule through x/|x| simplified with Euler's theorem for the degree-l homogeneous
//      Ytilde: u.g = l Y, H u = (l-1) g.  The oracle uses the plain projector form instead.)
#pragma once
#include "dd.cuh"
#include "tables.h"

namespace sphb200 {

#define SPH_INV_SQRT2 0.70710678118654752440

// ------------------------------------------------------------------------------------------
// Thread-per-point evaluator, column-wise: for each m the l-recurrence of column m runs with O(1)
// state (Qt_l^m, Qt_{l-1}^m) and, when gradients are wanted, column m+1 runs one row behind it
// (Eq. 10 needs Qt_{l-1}^{m+1}).  Values and gradients only (DERIV 0 or 1).
//   emit.val(k, v)        Y[k]
//   emit.grad(a, k, v)    dY/dx_a [k]
// R = double (f32 I/O) or dd (f64 I/O): the type the recurrences run in.
// ------------------------------------------------------------------------------------------
template <typename R, int DERIV, bool NORM, typename Emit>
SPH_HD void eval_point_columns(double x, double y, double z, int l_max, const SphTables& T,
                               Emit& emit) {
    using RT = rec<R>;
    R X, Y, Z, r2;
    double rinv = 1.0;
    if (NORM) {
        RT::normalize(x, y, z, X, Y, Z, rinv);
        r2 = RT::make(1.0, 0.0);
    } else {
        X = RT::make(x, 0.0);
        Y = RT::make(y, 0.0);
        Z = RT::make(z, 0.0);
        r2 = RT::r2_of(X, Y, Z);
    }
    const double xd = to_double(X), yd = to_double(Y), zd = to_double(Z);

    R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
    double c1 = 0.0, s1 = 0.0;  // c_{m-1}, s_{m-1}
    for (int m = 0; m <= l_max; ++m) {
        const double cd = to_double(c), sd = to_double(s);
        const double Ac = (m == 0) ? SPH_INV_SQRT2 : cd;  // Eq. 5: 1/sqrt2 for m = 0
        const double dm = (double)m;
        // Eq. 10: dc_m/dx = m c_{m-1}, dc_m/dy = -m s_{m-1}, ds_m/dx = m s_{m-1}, ds_m/dy = m c_{m-1}
        const double Acx = dm * c1, Acy = -dm * s1, Asx = dm * s1, Asy = dm * c1;
        const double xAc = xd * Ac, yAc = yd * Ac, xAs = xd * sd, yAs = yd * sd;

        R q = RT::make(T.D_hi[m], T.D_lo[m]);   // Qt_m^m
        R qp = RT::make(0.0, 0.0);              // Qt_{l-1}^m
        R p = RT::make(0.0, 0.0);               // Qt_{l-1}^{m+1}
        R pp = RT::make(0.0, 0.0);              // Qt_{l-2}^{m+1}
        int k0 = m * (m + 1);                   // l(l+1)
        for (int l = m; l <= l_max; ++l) {
            const double Q = to_double(q);
            const int kc = k0 + m, ks = k0 - m;
            const double Yc = Q * Ac, Ys = Q * sd;
            emit.val(kc, Yc);
            if (m > 0) emit.val(ks, Ys);
            if (DERIV >= 1) {
                const int t = SPH_TRI(l, m);
                const double q1 = T.G1[t] * to_double(p);    // F_l^m Q_{l-1}^{m+1}
                const double qz = T.Gz[t] * to_double(qp);   // F_l^m (l+m) Q_{l-1}^m
                double gxc = SPH_FMA(q1, xAc, Q * Acx), gyc = SPH_FMA(q1, yAc, Q * Acy), gzc = qz * Ac;
                double gxs = SPH_FMA(q1, xAs, Q * Asx), gys = SPH_FMA(q1, yAs, Q * Asy), gzs = qz * sd;
                if (NORM) {
                    const double lYc = (double)l * Yc, lYs = (double)l * Ys;
                    gxc = SPH_FMA(-lYc, xd, gxc) * rinv;
                    gyc = SPH_FMA(-lYc, yd, gyc) * rinv;
                    gzc = SPH_FMA(-lYc, zd, gzc) * rinv;
                    gxs = SPH_FMA(-lYs, xd, gxs) * rinv;
                    gys = SPH_FMA(-lYs, yd, gys) * rinv;
                    gzs = SPH_FMA(-lYs, zd, gzs) * rinv;
                }
                emit.grad(0, kc, gxc);
                emit.grad(1, kc, gyc);
                emit.grad(2, kc, gzc);
                if (m > 0) {
                    emit.grad(0, ks, gxs);
                    emit.grad(1, ks, gys);
                    emit.grad(2, ks, gzs);
                }
            }
            if (l < l_max) {
                const int t1 = SPH_TRI(l + 1, m);
                const R a = RT::make(T.A_hi[t1], T.A_lo[t1]);
                const R b = RT::make(T.B_hi[t1], T.B_lo[t1]);
                const R w = NORM ? qp : r2 * qp;
                const R qn = a * (Z * q) - b * w;
                qp = q;
                q = qn;
                if (DERIV >= 1) {  // column m+1 reaches row l
                    R pn;
                    if (l == m) {
                        pn = RT::make(0.0, 0.0);
                    } else if (l == m + 1) {
                        pn = RT::make(T.D_hi[m + 1], T.D_lo[m + 1]);
                    } else {
                        const int t2 = SPH_TRI(l, m + 1);
                        const R a2 = RT::make(T.A_hi[t2], T.A_lo[t2]);
                        const R b2 = RT::make(T.B_hi[t2], T.B_lo[t2]);
                        const R w2 = NORM ? pp : r2 * pp;
                        pn = a2 * (Z * p) - b2 * w2;
                    }
                    pp = p;
                    p = pn;
                }
            }
            k0 += 2 * (l + 1);
        }
        // Eq. 9: s_{m+1} = x s_m + y c_m,  c_{m+1} = -y s_m + x c_m
        c1 = cd;
        s1 = sd;
        const R cn = X * c - Y * s;
        const R sn = X * s + Y * c;
        c = cn;
        s = sn;
    }
}

// ------------------------------------------------------------------------------------------
// Pieces of the warp-per-point kernel (lane = m for the recurrences, lane = output index k for
// the assembly).
// ------------------------------------------------------------------------------------------

// c_m + i s_m = (X + iY)^m by square-and-multiply (B2); nbits = bits needed for l_max.
template <typename R>
SPH_HD void cs_power(int m, R X, R Y, int nbits, R& c, R& s) {
    using RT = rec<R>;
    c = RT::make(1.0, 0.0);
    s = RT::make(0.0, 0.0);
    R pr = X, pi = Y;
    for (int b = 0; b < nbits; ++b) {
        if ((m >> b) & 1) {
            const R cn = c * pr - s * pi;
            const R sn = c * pi + s * pr;
            c = cn;
            s = sn;
        }
        if (b + 1 < nbits) {
            const R prn = pr * pr - pi * pi;
            const R pin = (pr * pi) * 2.0;
            pr = prn;
            pi = pin;
        }
    }
}

// One step of column m of the folded Eq. 7: on entry (q, qp) = (Qt_{l-1}^m, Qt_{l-2}^m) for l > m;
// returns Qt_l^m.  For l == m returns D_m; for l < m returns 0.
template <typename R, bool NORM>
SPH_HD R column_step(int l, int m, R Z, R r2, R q, R qp, const SphTables& T) {
    using RT = rec<R>;
    if (l < m) return RT::make(0.0, 0.0);
    if (l == m) return RT::make(T.D_hi[m], T.D_lo[m]);
    const int t = SPH_TRI(l, m);
    const R a = RT::make(T.A_hi[t], T.A_lo[t]);
    const R b = RT::make(T.B_hi[t], T.B_lo[t]);
    const R w = NORM ? qp : r2 * qp;
    return rec_step(T.A_hi[t], T.A_lo[t], T.B_hi[t], T.B_lo[t], Z, q, w);   // (dd.cuh)
}

// The same column in the integer-coefficient scaling used by the warp kernel (tables.h):
//   W_l^m = (2l-1) z W_{l-1}^m - (l+m-1)(l-m-1) r^2 W_{l-2}^m,  W_m^m = 1,  Qt_l^m = Np_l^m W_l^m.
// On entry (w, wp) = (W_{l-1}^m, W_{l-2}^m); returns W_l^m (0 for l < m).
template <typename R, bool NORM>
SPH_HD R column_step_int(int l, int m, R Z, R r2, R w, R wp) {
    using RT = rec<R>;
    if (l < m) return RT::make(0.0, 0.0);
    if (l == m) return RT::make(1.0, 0.0);
    const double a = (double)(2 * l - 1);
    const double b = (double)((l + m - 1) * (l - m - 1));
    const R t = NORM ? wp : r2 * wp;
    return (Z * w) * a - t * b;
}

// Assembly of every requested output of ONE harmonic (l, mm), mm = -l..l, from the per-point
// scratch: Qt[] (triangle, doubles), cs[] = {c_0, s_0, c_1, s_1, ...} (doubles).
//   out[0]      Y
//   out[1..3]   dY/dx, dY/dy, dY/dz
//   out[4..9]   Hxx, Hxy, Hxz, Hyy, Hyz, Hzz
// (x,y,z) = the point the solid harmonics are evaluated at (u for NORM), rinv = 1/r (NORM).
// Tab: anything with members G1, Gz, H2, Hxz, Hzz indexable by SPH_TRI(l,m) (SphTables, or a
// view of copies in shared memory).
template <int DERIV, bool NORM, typename Tab>
SPH_HD void assemble_element(int l, int mm, const double* Qt, const double* cs, double x, double y,
                             double z, double rinv, const Tab& T, double* out) {
    const int m = mm < 0 ? -mm : mm;
    const int t = SPH_TRI(l, m);
    const double Q = Qt[t];
    const bool sinb = mm < 0;
    // A = c_m (cos branch), s_m (sin branch), 1/sqrt2 (m = 0)
    const double A = (mm == 0) ? SPH_INV_SQRT2 : cs[2 * m + (sinb ? 1 : 0)];
    out[0] = Q * A;
    if (DERIV < 1) return;

    const double dm = (double)m;
    const int m1 = m >= 1 ? m - 1 : 0;  // c_{m-1}, s_{m-1}; multiplied by m = 0 when absent
    const double c1 = cs[2 * m1], s1 = cs[2 * m1 + 1];
    // Eq. 10: cos branch A_x = m c_{m-1}, A_y = -m s_{m-1}; sin branch A_x = m s_{m-1}, A_y = m c_{m-1}
    const double Ax = dm * (sinb ? s1 : c1);
    const double Ay = dm * (sinb ? c1 : -s1);
    // neighbours in the triangle; the table entry is 0 whenever the neighbour does not exist,
    // so any in-range address will do for those
    const int t_l1 = l >= 1 ? SPH_TRI(l - 1, 0) : 0;
    const int i_q1 = (m + 1 <= l - 1) ? t_l1 + m + 1 : 0;
    const int i_qz = (m <= l - 1) ? t_l1 + m : 0;
    const double q1 = T.G1[t] * Qt[i_q1];
    const double qz = T.Gz[t] * Qt[i_qz];
    const double q1A = q1 * A;
    const double gx = SPH_FMA(x, q1A, Q * Ax);
    const double gy = SPH_FMA(y, q1A, Q * Ay);
    const double gz = qz * A;
    const double dl = (double)l;
    const double lY = dl * out[0];
    if (NORM) {
        out[1] = SPH_FMA(-lY, x, gx) * rinv;
        out[2] = SPH_FMA(-lY, y, gy) * rinv;
        out[3] = SPH_FMA(-lY, z, gz) * rinv;
    } else {
        out[1] = gx;
        out[2] = gy;
        out[3] = gz;
    }
    if (DERIV < 2) return;

    const double dmm = dm * (dm - 1.0);
    const int m2 = m >= 2 ? m - 2 : 0;
    const double c2 = cs[2 * m2], s2 = cs[2 * m2 + 1];
    // Eq. 10 twice: cos: A_xx = m(m-1) c_{m-2}, A_xy = -m(m-1) s_{m-2}; sin: m(m-1) s_{m-2}, m(m-1) c_{m-2}
    const double Axx = dmm * (sinb ? s2 : c2);
    const double Axy = dmm * (sinb ? c2 : -s2);
    const int t_l2 = l >= 2 ? SPH_TRI(l - 2, 0) : 0;
    const int i_q2 = (m + 2 <= l - 2) ? t_l2 + m + 2 : 0;
    const int i_qxz = (m + 1 <= l - 2) ? t_l2 + m + 1 : 0;
    const int i_qzz = (m <= l - 2) ? t_l2 + m : 0;
    const double q2A = T.H2[t] * Qt[i_q2] * A;
    const double qxz = T.Hxz[t] * Qt[i_qxz];
    const double qzz = T.Hzz[t] * Qt[i_qzz];
    const double q1Ax = q1 * Ax, q1Ay = q1 * Ay, QAxx = Q * Axx;
    // d2Q/dx2 = Q1 + x^2 Q2, d2Q/dxdy = xy Q2, d2Q/dxdz = (l+m) x Qxz, d2Q/dz2 = (l+m)(l+m-1) Qzz
    double Hxx = SPH_FMA(x * x, q2A, q1A) + SPH_FMA(2.0 * x, q1Ax, QAxx);
    double Hyy = SPH_FMA(y * y, q2A, q1A) + SPH_FMA(2.0 * y, q1Ay, -QAxx);
    double Hxy = SPH_FMA(x * y, q2A, Q * Axy) + SPH_FMA(x, q1Ay, y * q1Ax);
    const double qxzA = qxz * A;
    double Hxz = SPH_FMA(x, qxzA, qz * Ax);
    double Hyz = SPH_FMA(y, qxzA, qz * Ay);
    double Hzz = qzz * A;
    if (NORM) {
        // hess Y = (H - l(u g^T + g u^T) + l(l+2) Y u u^T - l Y I) / r^2   with g, H, Y at u
        const double r2inv = rinv * rinv;
        const double lgx = dl * gx, lgy = dl * gy, lgz = dl * gz;
        const double w = (dl + 2.0) * lY;
        const double wx = w * x, wy = w * y, wz = w * z;
        Hxx = (SPH_FMA(x, SPH_FMA(-2.0, lgx, wx), Hxx) - lY) * r2inv;
        Hyy = (SPH_FMA(y, SPH_FMA(-2.0, lgy, wy), Hyy) - lY) * r2inv;
        Hzz = (SPH_FMA(z, SPH_FMA(-2.0, lgz, wz), Hzz) - lY) * r2inv;
        Hxy = SPH_FMA(x, wy - lgy, SPH_FMA(-y, lgx, Hxy)) * r2inv;
        Hxz = SPH_FMA(x, wz - lgz, SPH_FMA(-z, lgx, Hxz)) * r2inv;
        Hyz = SPH_FMA(y, wz - lgz, SPH_FMA(-z, lgy, Hyz)) * r2inv;
    }
    out[4] = Hxx;
    out[5] = Hxy;
    out[6] = Hxz;
    out[7] = Hyy;
    out[8] = Hyz;
    out[9] = Hzz;
}

// Assembly of every requested output of the PAIR of harmonics (l, +m) and (l, -m), m >= 0, from
// the per-point scratch.  Both share Qt_l^m and every Legendre-side factor of Eq. 10 (the five
// neighbours in the triangle, the coefficient tables, the second-derivative tensor of Q); only the
// azimuthal factor A = c_m | s_m and its derivatives differ, so a pair costs little more than one
// element.  t = SPH_TRI(l, m).  oc[] = outputs of (l, +m), os[] = outputs of (l, -m) (meaningless
// for m == 0), both in the order of assemble_element.
// The neighbours' indices need no clamping: with t1 = t - l (= TRI(l-1, m)) and
// t2 = t - 2l + 1 (= TRI(l-2, m)) every index below lies in [0, t + 1] and the table entry is 0
// whenever the neighbour does not exist, so what is read there only has to be finite.
template <int DERIV, bool NORM, typename Tab>
SPH_HD void assemble_pair(int l, int m, int t, const double* Qt, const double* cs, double x, double y,
                          double z, double rinv, const Tab& T, double* oc, double* os) {
    const double Q = Qt[t];
    const double c0 = (m == 0) ? SPH_INV_SQRT2 : cs[2 * m];
    const double s0 = cs[2 * m + 1];
    oc[0] = Q * c0;
    os[0] = Q * s0;
    if (DERIV < 1) return;

    const double dm = (double)m, dl = (double)l;
    const int m1 = m >= 1 ? m - 1 : 0;  // c_{m-1}, s_{m-1}; multiplied by m = 0 when absent
    const double c1 = cs[2 * m1], s1 = cs[2 * m1 + 1];
    const int t1 = t - l;
    const double q1 = T.G1[t] * Qt[t1 + 1];   // F_l^m Q_{l-1}^{m+1}
    const double qz = T.Gz[t] * Qt[t1];       // F_l^m (l+m) Q_{l-1}^m
    const double a1 = x * q1, a2 = y * q1;
    // Eq. 10: cos branch A_x = m c_{m-1}, A_y = -m s_{m-1}; sin branch A_x = m s_{m-1}, A_y = m c_{m-1}
    const double Acx = dm * c1, Acy = -dm * s1, Asx = dm * s1, Asy = dm * c1;
    const double gcx = SPH_FMA(a1, c0, Q * Acx), gcy = SPH_FMA(a2, c0, Q * Acy), gcz = qz * c0;
    const double gsx = SPH_FMA(a1, s0, Q * Asx), gsy = SPH_FMA(a2, s0, Q * Asy), gsz = qz * s0;
    const double lYc = dl * oc[0], lYs = dl * os[0];
    if (NORM) {
        oc[1] = SPH_FMA(-lYc, x, gcx) * rinv;
        oc[2] = SPH_FMA(-lYc, y, gcy) * rinv;
        oc[3] = SPH_FMA(-lYc, z, gcz) * rinv;
        os[1] = SPH_FMA(-lYs, x, gsx) * rinv;
        os[2] = SPH_FMA(-lYs, y, gsy) * rinv;
        os[3] = SPH_FMA(-lYs, z, gsz) * rinv;
    } else {
        oc[1] = gcx, oc[2] = gcy, oc[3] = gcz;
        os[1] = gsx, os[2] = gsy, os[3] = gsz;
    }
    if (DERIV < 2) return;

    const double dmm = dm * (dm - 1.0);
    const int m2 = m >= 2 ? m - 2 : 0;
    const double c2 = cs[2 * m2], s2 = cs[2 * m2 + 1];
    const int t2 = t1 - l + 1;
    const double q2 = T.H2[t] * Qt[t2 + 2];
    const double qxz = T.Hxz[t] * Qt[t2 + 1];
    const double qzz = T.Hzz[t] * Qt[t2];
    // second derivatives of Q (Eq. 10 twice): Q1 + x^2 Q2, xy Q2, (l+m) x Qxz, (l+m)(l+m-1) Qzz
    const double Qxx = SPH_FMA(x * x, q2, q1), Qyy = SPH_FMA(y * y, q2, q1), Qxy = (x * y) * q2;
    const double Qxz = x * qxz, Qyz = y * qxz;
    const double b1 = 2.0 * a1, b2 = 2.0 * a2;
    const double r2inv = rinv * rinv;
    const double w2 = dl + 2.0;
    // one branch: A, its first derivatives (Ax, Ay), second derivatives Axx (= -Ayy), Axy
    auto branch = [&](double A, double Ax, double Ay, double Axx, double Axy, double gx, double gy, double gz,
                      double lY, double* o) {
        const double QAxx = Q * Axx;
        double Hxx = SPH_FMA(Qxx, A, SPH_FMA(b1, Ax, QAxx));
        double Hyy = SPH_FMA(Qyy, A, SPH_FMA(b2, Ay, -QAxx));
        double Hxy = SPH_FMA(Qxy, A, SPH_FMA(a1, Ay, SPH_FMA(a2, Ax, Q * Axy)));
        double Hxz = SPH_FMA(Qxz, A, qz * Ax);
        double Hyz = SPH_FMA(Qyz, A, qz * Ay);
        double Hzz = qzz * A;
        if (NORM) {
            // hess Y = (H - l(u g^T + g u^T) + l(l+2) Y u u^T - l Y I) / r^2   with g, H, Y at u
            const double lgx = dl * gx, lgy = dl * gy, lgz = dl * gz;
            const double w = w2 * lY;
            const double wx = w * x, wy = w * y, wz = w * z;
            Hxx = (SPH_FMA(x, SPH_FMA(-2.0, lgx, wx), Hxx) - lY) * r2inv;
            Hyy = (SPH_FMA(y, SPH_FMA(-2.0, lgy, wy), Hyy) - lY) * r2inv;
            Hzz = (SPH_FMA(z, SPH_FMA(-2.0, lgz, wz), Hzz) - lY) * r2inv;
            Hxy = SPH_FMA(x, wy - lgy, SPH_FMA(-y, lgx, Hxy)) * r2inv;
            Hxz = SPH_FMA(x, wz - lgz, SPH_FMA(-z, lgx, Hxz)) * r2inv;
            Hyz = SPH_FMA(y, wz - lgz, SPH_FMA(-z, lgy, Hyz)) * r2inv;
        }
        o[4] = Hxx, o[5] = Hxy, o[6] = Hxz, o[7] = Hyy, o[8] = Hyz, o[9] = Hzz;
    };
    // Eq. 10 twice: cos: A_xx = m(m-1) c_{m-2}, A_xy = -m(m-1) s_{m-2}; sin: m(m-1) s_{m-2}, m(m-1) c_{m-2}
    branch(c0, Acx, Acy, dmm * c2, -dmm * s2, gcx, gcy, gcz, lYc, oc);
    branch(s0, Asx, Asy, dmm * s2, dmm * c2, gsx, gsy, gsz, lYs, os);
}


// All outputs of ONE harmonic from scalars: Q = Qt_l^m, the five Legendre-side neighbours already
// multiplied by their table ratios (q1 = F Q_{l-1}^{m+1}, qz = F (l+m) Q_{l-1}^m, q2 = F Q_{l-2}^{m+2},
// qxz = F (l+m) Q_{l-2}^{m+1}, qzz = F (l+m)(l+m-1) Q_{l-2}^m; 0 where the neighbour does not exist),
// the azimuthal factor A and its derivatives (A_yy = -A_xx).  Same formulas and output order as
// assemble_element; used by the unrolled Hessian kernels, whose columns live in registers.
template <bool NORM>
SPH_HD void assemble_scalars(int l, double Q, double q1, double qz, double q2, double qxz, double qzz, double A,
                             double Ax, double Ay, double Axx, double Axy, double x, double y, double z,
                             double rinv, double* out) {
    out[0] = Q * A;
    const double q1A = q1 * A;
    const double gx = SPH_FMA(x, q1A, Q * Ax);
    const double gy = SPH_FMA(y, q1A, Q * Ay);
    const double gz = qz * A;
    const double dl = (double)l;
    const double lY = dl * out[0];
    if (NORM) {
        out[1] = SPH_FMA(-lY, x, gx) * rinv;
        out[2] = SPH_FMA(-lY, y, gy) * rinv;
        out[3] = SPH_FMA(-lY, z, gz) * rinv;
    } else {
        out[1] = gx;
        out[2] = gy;
        out[3] = gz;
    }
    const double q2A = q2 * A;
    const double q1Ax = q1 * Ax, q1Ay = q1 * Ay, QAxx = Q * Axx;
    // d2Q/dx2 = Q1 + x^2 Q2, d2Q/dxdy = xy Q2, d2Q/dxdz = (l+m) x Qxz, d2Q/dz2 = (l+m)(l+m-1) Qzz
    double Hxx = SPH_FMA(x * x, q2A, q1A) + SPH_FMA(2.0 * x, q1Ax, QAxx);
    double Hyy = SPH_FMA(y * y, q2A, q1A) + SPH_FMA(2.0 * y, q1Ay, -QAxx);
    double Hxy = SPH_FMA(x * y, q2A, Q * Axy) + SPH_FMA(x, q1Ay, y * q1Ax);
    const double qxzA = qxz * A;
    double Hxz = SPH_FMA(x, qxzA, qz * Ax);
    double Hyz = SPH_FMA(y, qxzA, qz * Ay);
    double Hzz = qzz * A;
    if (NORM) {
        // hess Y = (H - l(u g^T + g u^T) + l(l+2) Y u u^T - l Y I) / r^2   with g, H, Y at u
        const double r2inv = rinv * rinv;
        const double lgx = dl * gx, lgy = dl * gy, lgz = dl * gz;
        const double w = (dl + 2.0) * lY;
        const double wx = w * x, wy = w * y, wz = w * z;
        Hxx = (SPH_FMA(x, SPH_FMA(-2.0, lgx, wx), Hxx) - lY) * r2inv;
        Hyy = (SPH_FMA(y, SPH_FMA(-2.0, lgy, wy), Hyy) - lY) * r2inv;
        Hzz = (SPH_FMA(z, SPH_FMA(-2.0, lgz, wz), Hzz) - lY) * r2inv;
        Hxy = SPH_FMA(x, wy - lgy, SPH_FMA(-y, lgx, Hxy)) * r2inv;
        Hxz = SPH_FMA(x, wz - lgz, SPH_FMA(-z, lgx, Hxz)) * r2inv;
        Hyz = SPH_FMA(y, wz - lgz, SPH_FMA(-z, lgy, Hyz)) * r2inv;
    }
    out[4] = Hxx, out[5] = Hxy, out[6] = Hxz, out[7] = Hyy, out[8] = Hyz, out[9] = Hzz;
}

}  // namespace sphb200
