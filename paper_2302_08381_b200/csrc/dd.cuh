// Recurrence arithmetic at twice the I/O precision.
//
// The tolerance of the path is relative to max(|Y|, 1e-3 * row scale).
// An element near a zero of Y_l^m inherits the absolute rounding error of the recurrences
// (~l * eps * row scale), so recurrences carried in the I/O precision cannot meet it: f32 I/O
// runs them in f64, f64 I/O runs them in double-double ("dd", ~106 bits) built from FMA-based
// error-free transformations.  Assembly of the outputs then happens in f64.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

// The arithmetic core is __host__ __device__ so that a CPU harness can run the very same code
// (host build: compile with -ffp-contract=off so the error-free transformations stay exact).
#define SPH_HD __host__ __device__ __forceinline__
#ifdef __CUDA_ARCH__
#define SPH_ADD(a, b) __dadd_rn((a), (b))
#define SPH_SUB(a, b) __dsub_rn((a), (b))
#define SPH_MUL(a, b) __dmul_rn((a), (b))
#define SPH_FMA(a, b, c) __fma_rn((a), (b), (c))
#define SPH_RSQRT(a) rsqrt(a)
#else
#define SPH_ADD(a, b) ((a) + (b))
#define SPH_SUB(a, b) ((a) - (b))
#define SPH_MUL(a, b) ((a) * (b))
#define SPH_FMA(a, b, c) fma((a), (b), (c))
#define SPH_RSQRT(a) (1.0 / sqrt(a))
#endif

namespace sphb200 {

struct dd {
    double hi, lo;
};

SPH_HD dd dd_make(double hi, double lo = 0.0) { return dd{hi, lo}; }

// a + b = s + e exactly, |a| >= |b| (or a == 0)
SPH_HD dd quick_two_sum(double a, double b) {
    double s = SPH_ADD(a, b);
    double e = SPH_SUB(b, SPH_SUB(s, a));
    return dd{s, e};
}
// a + b = s + e exactly
SPH_HD dd two_sum(double a, double b) {
    double s = SPH_ADD(a, b);
    double bb = SPH_SUB(s, a);
    double e = SPH_ADD(SPH_SUB(a, SPH_SUB(s, bb)), SPH_SUB(b, bb));
    return dd{s, e};
}
// a * b = p + e exactly
SPH_HD dd two_prod(double a, double b) {
    double p = SPH_MUL(a, b);
    double e = SPH_FMA(a, b, -p);
    return dd{p, e};
}

SPH_HD dd operator+(dd a, dd b) {  // "sloppy" add: error ~2^-104 (|a|+|b|)
    dd s = two_sum(a.hi, b.hi);
    s.lo = SPH_ADD(s.lo, SPH_ADD(a.lo, b.lo));
    return quick_two_sum(s.hi, s.lo);
}
SPH_HD dd operator-(dd a) { return dd{-a.hi, -a.lo}; }
SPH_HD dd operator-(dd a, dd b) { return a + (-b); }
SPH_HD dd operator*(dd a, dd b) {
    dd p = two_prod(a.hi, b.hi);
    p.lo = SPH_FMA(a.hi, b.lo, p.lo);
    p.lo = SPH_FMA(a.lo, b.hi, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
SPH_HD dd operator*(dd a, double b) {
    dd p = two_prod(a.hi, b);
    p.lo = SPH_FMA(a.lo, b, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
SPH_HD dd operator*(double a, dd b) { return b * a; }

// The two recurrence types share this small vocabulary so the kernels are written once.
template <typename R> struct rec;

template <> struct rec<double> {
    using type = double;
    SPH_HD static double make(double hi, double) { return hi; }
    SPH_HD static double to_double(double a) { return a; }
    // (x,y,z) -> unit vector u and 1/r (as double)
    SPH_HD static void normalize(double x, double y, double z, double& ux,
                                                     double& uy, double& uz, double& rinv) {
        double r2 = SPH_FMA(x, x, SPH_FMA(y, y, z * z));
        rinv = SPH_RSQRT(r2);
        // one Newton step: rsqrt() is good to ~1 ulp, this makes the unit vector's norm 1 to eps
        rinv = SPH_FMA(rinv * 0.5, SPH_FMA(-r2 * rinv, rinv, 1.0), rinv);
        ux = x * rinv;
        uy = y * rinv;
        uz = z * rinv;
    }
    SPH_HD static double r2_of(double x, double y, double z) {
        return SPH_FMA(x, x, SPH_FMA(y, y, z * z));
    }
};

template <> struct rec<dd> {
    using type = dd;
    SPH_HD static dd make(double hi, double lo) { return dd{hi, lo}; }
    SPH_HD static double to_double(dd a) { return a.hi; }
    SPH_HD static void normalize(double x, double y, double z, dd& ux, dd& uy,
                                                     dd& uz, double& rinv) {
        dd r2 = two_prod(x, x) + two_prod(y, y) + two_prod(z, z);
        double y0 = SPH_RSQRT(r2.hi);
        // Newton in dd: y1 = y0 + y0 (1 - r2 y0^2) / 2, the bracket evaluated in dd
        dd t = (r2 * y0) * y0;                       // ~1
        double delta = SPH_SUB(SPH_SUB(1.0, t.hi), t.lo);
        dd ri = quick_two_sum(y0, y0 * delta * 0.5);
        rinv = ri.hi;
        ux = ri * x;
        uy = ri * y;
        uz = ri * z;
    }
    SPH_HD static dd r2_of(dd x, dd y, dd z) { return x * x + y * y + z * z; }
};

// One step of the folded Eq. 7 (tables.h): a (Z q) - b w.
// Double-double form: the three products keep their error terms unnormalised ((hi, e) with
// |e| ~ 2^-53 |hi|: first-order terms only, the dropped ones are ~2^-106), the difference of the
// high parts is an exact two_sum, and the result is normalised once: 23 operations instead of the
// 32 of  a * (Z * q) - b * w  with normalised intermediates, same ~2^-100 relative accuracy.
SPH_HD double rec_step(double a_hi, double, double b_hi, double, double Z, double q, double w) {
    return SPH_FMA(a_hi * Z, q, -(b_hi * w));
}
SPH_HD dd rec_step(double a_hi, double a_lo, double b_hi, double b_lo, dd Z, dd q, dd w) {
    const double p = SPH_MUL(Z.hi, q.hi);
    double e = SPH_FMA(Z.hi, q.hi, -p);
    e = SPH_FMA(Z.hi, q.lo, e);
    e = SPH_FMA(Z.lo, q.hi, e);
    const double th = SPH_MUL(a_hi, p);
    double te = SPH_FMA(a_hi, p, -th);
    te = SPH_FMA(a_hi, e, te);
    te = SPH_FMA(a_lo, p, te);
    const double uh = SPH_MUL(b_hi, w.hi);
    double ue = SPH_FMA(b_hi, w.hi, -uh);
    ue = SPH_FMA(b_hi, w.lo, ue);
    ue = SPH_FMA(b_lo, w.hi, ue);
    const dd s = two_sum(th, -uh);
    return quick_two_sum(s.hi, SPH_ADD(s.lo, SPH_SUB(te, ue)));
}

// The same step WITHOUT the final normalisation: the result is the unevaluated pair (hi, lo) with
// hi = fl(fl(a_hi fl(Z_hi q_hi)) - fl(b_hi w_hi)) -- the plain f64 recurrence on the high parts -- and
// lo = the first-order correction (every rounding error of those operations, exact by FMA / two_sum,
// plus the low parts of a, b, Z, q, w).  |lo| stays ~ l 2^-53 |hi| over a whole column, so the
// second-order terms dropped are ~2^-94; the value is hi + lo (pair_value).  What this buys is the
// DEPENDENCY DEPTH from one step to the next: 3 operations for hi, 4 for lo, against 8-10 through the
// normalisation -- the columns of Eq. 7 are latency-bound chains.  q and w may be such pairs themselves.
SPH_HD double rec_step_u(double a_hi, double, double b_hi, double, double Z, double q, double w) {
    return SPH_FMA(a_hi * Z, q, -(b_hi * w));
}
SPH_HD dd rec_step_u(double a_hi, double a_lo, double b_hi, double b_lo, dd Z, dd q, dd w) {
    const double p = SPH_MUL(Z.hi, q.hi);
    double e = SPH_FMA(Z.hi, q.hi, -p);
    e = SPH_FMA(Z.lo, q.hi, e);
    e = SPH_FMA(Z.hi, q.lo, e);              // (the carried low part enters last)
    const double th = SPH_MUL(a_hi, p);
    double te = SPH_FMA(a_hi, p, -th);
    te = SPH_FMA(a_lo, p, te);
    te = SPH_FMA(a_hi, e, te);
    const double uh = SPH_MUL(b_hi, w.hi);
    double ue = SPH_FMA(b_hi, w.hi, -uh);
    ue = SPH_FMA(b_lo, w.hi, ue);
    ue = SPH_FMA(b_hi, w.lo, ue);
    const dd s = two_sum(th, -uh);
    dd r;
    r.hi = s.hi;
    r.lo = SPH_ADD(s.lo, SPH_SUB(te, ue));
    return r;
}
SPH_HD double pair_value(double a) { return a; }
SPH_HD double pair_value(dd a) { return SPH_ADD(a.hi, a.lo); }

SPH_HD double rec_step2(double a, double b, double Z, double q, double w) { return rec_step(a, 0.0, b, 0.0, Z, q, w); }
SPH_HD dd rec_step2(dd a, dd b, dd Z, dd q, dd w) { return rec_step(a.hi, a.lo, b.hi, b.lo, Z, q, w); }

SPH_HD double to_double(double a) { return a; }
SPH_HD double to_double(dd a) { return a.hi; }

}  // namespace sphb200
