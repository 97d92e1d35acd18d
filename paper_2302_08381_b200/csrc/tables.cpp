// Host-side construction of SphTables (see tables.h for the formulas and their derivation
// from Eq. 3, Eq. 7, Eq. 10 and App. C of the paper).  Square roots are taken in IEEE quad
// precision so that the double-double constants are good to ~1e-32.
#include "tables.h"

#include <quadmath.h>

typedef __float128 quad;

static void split(quad v, double* hi, double* lo) {
    *hi = (double)v;
    *lo = (double)(v - (quad)*hi);
}

extern "C" void sph_build_tables(SphTables* t) {
    const quad pi = 4 * atanq((quad)1);
    for (int i = 0; i < SPH_TRI_SIZE; ++i) {
        t->A_hi[i] = t->A_lo[i] = t->B_hi[i] = t->B_lo[i] = 0.0;
        t->G1[i] = t->Gz[i] = t->H2[i] = t->Hxz[i] = t->Hzz[i] = 0.0;
    }
    quad D = 1 / sqrtq(2 * pi);
    for (int m = 0; m <= SPH_MAX_L; ++m) {
        if (m > 0) D *= sqrtq((quad)(2 * m + 1) / (quad)(2 * m));
        split(D, &t->D_hi[m], &t->D_lo[m]);
    }
    // Np_l^m = sqrt((2l+1)/(2 pi) (l-m)!/(l+m)!) (2m-1)!! / (l-m)!
    quad fact[2 * SPH_MAX_L + 1];
    fact[0] = 1;
    for (int i = 1; i <= 2 * SPH_MAX_L; ++i) fact[i] = fact[i - 1] * i;
    quad dfact = 1;  // (2m-1)!!
    for (int m = 0; m <= SPH_MAX_L; ++m) {
        if (m > 0) dfact *= (2 * m - 1);
        for (int l = m; l <= SPH_MAX_L; ++l)
            t->Np[SPH_TRI(l, m)] = (double)(sqrtq((quad)(2 * l + 1) / (2 * pi) * fact[l - m] / fact[l + m]) *
                                            dfact / fact[l - m]);
    }
    for (int l = 1; l <= SPH_MAX_L; ++l) {
        for (int m = 0; m <= l; ++m) {
            const int i = SPH_TRI(l, m);
            const quad ql = l, qm = m;
            if (m < l) {
                quad A = sqrtq((4 * ql * ql - 1) / (ql * ql - qm * qm));
                split(A, &t->A_hi[i], &t->A_lo[i]);
                if (m <= l - 2) {
                    quad B = A * sqrtq(((ql - 1) * (ql - 1) - qm * qm) / (4 * (ql - 1) * (ql - 1) - 1));
                    split(B, &t->B_hi[i], &t->B_lo[i]);
                }
                t->Gz[i] = (double)sqrtq((2 * ql + 1) / (2 * ql - 1) * (ql - qm) * (ql + qm));
            }
            if (m <= l - 2) {
                t->G1[i] = (double)-sqrtq((2 * ql + 1) / (2 * ql - 1) * (ql - qm) * (ql - qm - 1));
                t->Hzz[i] = (double)sqrtq((2 * ql + 1) / (2 * ql - 3) * (ql - qm) * (ql - qm - 1) *
                                          (ql + qm) * (ql + qm - 1));
            }
            if (m <= l - 3)
                t->Hxz[i] = (double)-sqrtq((2 * ql + 1) / (2 * ql - 3) * (ql + qm) * (ql - qm) *
                                           (ql - qm - 1) * (ql - qm - 2));
            if (m <= l - 4)
                t->H2[i] = (double)sqrtq((2 * ql + 1) / (2 * ql - 3) * (ql - qm) * (ql - qm - 1) *
                                         (ql - qm - 2) * (ql - qm - 3));
        }
    }
}
