// Coefficient tables of the CUDA path (host-built once, uploaded per device).
//
// The kernels run the paper's recurrences with the prefactor folded into the Legendre part,
// Qt_l^m = F_l^m Q_l^m (App. C: "incorporate the prefactors in the definition of the
// modified associated Legendre polynomials ... avoids possible instabilities connected with the
// fact that F_l^m become very small for large m ~ l").  Folding Eq. 3 into Eq. 7
// gives, for fixed m and l >= m+1,
//     Qt_l^m = A_l^m z Qt_{l-1}^m - B_l^m r^2 Qt_{l-2}^m,       Qt_m^m = D_m,  Qt_{m-1}^m = 0,
//     A_l^m = sqrt((4l^2-1)/(l^2-m^2)),   B_l^m = A_l^m sqrt(((l-1)^2-m^2)/(4(l-1)^2-1)),
//     D_0 = 1/sqrt(2 pi),  D_m = D_{m-1} sqrt((2m+1)/(2m))      (= F_m^m (-1)^m (2m-1)!!, Eq. 7 line 1)
// and the derivative rules of Eq. 10 pick up ratios of prefactors:
//     F_l^m Q_{l-1}^{m+1}          = G1_l^m  Qt_{l-1}^{m+1},  G1  = -sqrt((2l+1)/(2l-1) (l-m)(l-m-1))
//     F_l^m (l+m) Q_{l-1}^m        = Gz_l^m  Qt_{l-1}^m,      Gz  =  sqrt((2l+1)/(2l-1) (l-m)(l+m))
//     F_l^m Q_{l-2}^{m+2}          = H2_l^m  Qt_{l-2}^{m+2},  H2  =  sqrt((2l+1)/(2l-3) (l-m)(l-m-1)(l-m-2)(l-m-3))
//     F_l^m (l+m) Q_{l-2}^{m+1}    = Hxz_l^m Qt_{l-2}^{m+1},  Hxz = -sqrt((2l+1)/(2l-3) (l+m)(l-m)(l-m-1)(l-m-2))
//     F_l^m (l+m)(l+m-1) Q_{l-2}^m = Hzz_l^m Qt_{l-2}^m,      Hzz =  sqrt((2l+1)/(2l-3) (l-m)(l-m-1)(l+m)(l+m-1))
// (Gz is App. C's Eq. C2 with the factor sqrt((2l+1)/(2l-1)) the print omits, reading E4.)
// A, B, D are stored as double-double (hi + lo) because the f64 path runs its recurrences in dd.
//
// The warp-per-point kernel runs the UNfolded Eq. 7 scaled to integer coefficients instead
// (its lanes sit on different (l,m), so a dd coefficient table would cost four loads per step):
//     W_l^m := (l-m)! Q_l^m / Q_m^m,   W_m^m = 1,
//     W_l^m = (2l-1) z W_{l-1}^m - (l+m-1)(l-m-1) r^2 W_{l-2}^m          (Eq. 7 times (l-m-1)!/Q_m^m)
//     Qt_l^m = Np_l^m W_l^m,   Np_l^m = F_l^m Q_m^m / (l-m)! = sqrt((2l+1)/(2 pi) (l-m)!/(l+m)!) (2m-1)!!/(l-m)!
#pragma once

#define SPH_MAX_L 32
#define SPH_TRI_SIZE ((SPH_MAX_L + 1) * (SPH_MAX_L + 2) / 2) /* 561 */

struct SphTables {
    double A_hi[SPH_TRI_SIZE], A_lo[SPH_TRI_SIZE];
    double B_hi[SPH_TRI_SIZE], B_lo[SPH_TRI_SIZE];
    double G1[SPH_TRI_SIZE], Gz[SPH_TRI_SIZE];
    double H2[SPH_TRI_SIZE], Hxz[SPH_TRI_SIZE], Hzz[SPH_TRI_SIZE];
    double D_hi[SPH_MAX_L + 1], D_lo[SPH_MAX_L + 1];
    double Np[SPH_TRI_SIZE];
};

// index of (l,m), 0 <= m <= l, in the triangle arrays
#define SPH_TRI(l, m) ((l) * ((l) + 1) / 2 + (m))

#ifdef __cplusplus
extern "C"
#endif
    void
    sph_build_tables(struct SphTables* t); /* tables.cpp; quad-precision square roots */
