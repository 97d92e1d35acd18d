// Recompute-in-backward VJP: grad_xyz[i,a] = sum_k (d sph[i,k] / d xyz[i,a]) grad_sph[i,k]
// evaluated from xyz and grad_sph alone -- the backward pass of P:112 without the [n,3,L] array of
// stored derivatives.  Per point it reads 3 + L values and writes 3, against 4 L + 3 for the stored
// form (C5: 220 B instead of 796 B), and the forward pass no longer has to write dsph at all.
//
// Mapping: ONE lane per point doing both branches of Eq. 5 (the Legendre recurrences, half of the
// work, run once for the two; with two lanes per point as in kernel_tpb.cuh C5 took 216 us), 32
// points per warp, l_max a compile-time constant, one tile per single-warp CTA, non-persistent grid.  The
// tile's grad_sph rows are one contiguous range: a 1-D TMA bulk load brings them to shared memory.
//
// The gradient of one harmonic (Eq. 10 with the prefactors folded, normalised form as in
// kernel_tpb.cuh) is linear in three Legendre-side terms whose coefficients depend on the column m
// only,
//     dY/dx = [(q1 - l Q) x A + Q A_x] / r,  dY/dy likewise,  dY/dz = (qz - l Q z) A / r,
// so inside a column only five sums over l are accumulated,
//     S1 = sum q1 w,  Sz = sum qz w,  SQ = sum Q w,  Sl = sum l Q w      (w = grad_sph[i, k(l, +-m)]),
// and the column contributes  x A (S1 - Sl) + A_x SQ,  y A (S1 - Sl) + A_y SQ,  A (Sz - z Sl)
// (solid harmonics: the same without the Sl terms and without 1/r).
#pragma once
#include "kernel_tpb.cuh"

namespace sphb200 {

struct VjprParams {
    const void* xyz;
    const void* grad_sph;
    void* grad_xyz;
    int64_t n;
    int pdl;   // launched as a programmatic dependent launch (see kernel_tpb.cuh)
};

template <typename T, typename R, bool NORM, int LMAX>
__global__ void __launch_bounds__(32, 16) sph_vjpr_kernel(const VjprParams prm) {
    using RT = rec<R>;
    constexpr int L = (LMAX + 1) * (LMAX + 1);
    constexpr int PTS = 32;   // points per tile
    constexpr uint32_t W_BYTES = PTS * L * sizeof(T);
    const SphTables& TB = c_tables_tpb;
    extern __shared__ __align__(128) unsigned char smem[];
    T* Wt = reinterpret_cast<T*>(smem);                          // [32][L] upstream gradients of the tile
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + W_BYTES);
    const int lane = threadIdx.x;
    const int pl = lane;                   // point inside the tile
    const int64_t n = prm.n;
    const int64_t tile = blockIdx.x;
    const int64_t p0 = tile * PTS;
    const int64_t p = p0 + pl;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    const T* __restrict__ gsph = static_cast<const T*>(prm.grad_sph);
    T* __restrict__ gxyz = static_cast<T*>(prm.grad_xyz);

    // programmatic dependent launch: see kernel_tpb.cuh
    if (prm.pdl) {
        grid_launch_dependents();
        grid_dependency_wait();
    }

    const bool full = n - p0 >= PTS;
    if (full) {
        if (lane == 0) {
            mbar_init(bar, 1);
            fence_mbar_init();
            mbar_arrive_expect_tx(bar, W_BYTES);
            bulk_load(Wt, gsph + p0 * L, W_BYTES, bar);
        }
    } else {   // ragged last tile: byte count need not be a multiple of 16 -> plain loads
        const int np = (int)(n - p0);
        for (int i = lane; i < PTS * L; i += 32) Wt[i] = i < np * L ? gsph[p0 * L + i] : T(0);
    }
    __syncwarp();

    // lanes past the end compute a harmless point
    double x = 0.0, y = 0.0, z = 1.0;
    if (p < n) {
        x = static_cast<double>(__ldg(xyz + 3 * p + 0));
        y = static_cast<double>(__ldg(xyz + 3 * p + 1));
        z = static_cast<double>(__ldg(xyz + 3 * p + 2));
    }
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

    double Qc[LMAX + 1];   // column m:   Qc[l] = Qt_l^m     (0 for l < m)
    double Qn[LMAX + 1];   // column m+1: Qn[l] = Qt_l^{m+1} (0 for l < m+1)
    auto column = [&](auto Mc, double* dst) {   // column M of the folded Eq. 7 (kernel_tpb.cuh)
        constexpr int M = decltype(Mc)::value;
        R q = RT::make(TB.D_hi[M], TB.D_lo[M]), qp = RT::make(0.0, 0.0);
        static_for<M, LMAX + 1>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            dst[l] = to_double(q);
            if constexpr (l < LMAX) {
                constexpr int t1 = SPH_TRI(l + 1, M);
                const R a = RT::make(TB.A_hi[t1], TB.A_lo[t1]);
                R qn;
                if constexpr (l == M) {
                    qn = a * (Z * q);
                } else {
                    const R w = NORM ? qp : r2 * qp;
                    qn = rec_step(TB.A_hi[t1], TB.A_lo[t1], TB.B_hi[t1], TB.B_lo[t1], Z, q, w);   // (dd.cuh)
                }
                qp = q;
                q = qn;
            }
        });
    };
    column(std::integral_constant<int, 0>{}, Qc);

    if (full) mbar_wait(bar, 0);
    const T* W = Wt + pl * L;

    R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
    double c1 = 0.0, s1 = 0.0;  // c_{m-1}, s_{m-1}
    double ax = 0.0, ay = 0.0, az = 0.0;
    static_for<0, LMAX + 1>([&](auto mc) {
        constexpr int m = decltype(mc)::value;
        if constexpr (m < LMAX) column(std::integral_constant<int, m + 1>{}, Qn);
        const double cd = to_double(c), sd = to_double(s);
        const double dm = (double)m;
        // azimuthal factors of the two branches and their x/y derivatives (Eq. 9, Eq. 10); the sin
        // branch has no m = 0 harmonic
        const double Ac = (m == 0) ? SPH_INV_SQRT2 : cd, As = sd;
        const double Acx = dm * c1, Acy = -dm * s1, Asx = dm * s1, Asy = dm * c1;
        double S1c = 0.0, Szc = 0.0, SQc = 0.0, Slc = 0.0;   // the four sums of the cos branch
        double S1s = 0.0, Szs = 0.0, SQs = 0.0, Sls = 0.0;   // ... of the sin branch
        static_for<m, LMAX + 1>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            constexpr int kc = l * (l + 1) + m, ks = l * (l + 1) - m;
            constexpr int t = SPH_TRI(l, m);
            const double wc = static_cast<double>(W[kc]);
            const double ws = (m > 0) ? static_cast<double>(W[ks]) : 0.0;
            const double Q = Qc[l];
            SQc = SPH_FMA(Q, wc, SQc);
            SQs = SPH_FMA(Q, ws, SQs);
            if (NORM) {
                const double lQ = (double)l * Q;
                Slc = SPH_FMA(lQ, wc, Slc);
                Sls = SPH_FMA(lQ, ws, Sls);
            }
            if constexpr (l >= m + 2) {   // F_l^m Q_{l-1}^{m+1}
                const double q1 = TB.G1[t] * Qn[l - 1];
                S1c = SPH_FMA(q1, wc, S1c);
                S1s = SPH_FMA(q1, ws, S1s);
            }
            if constexpr (l >= m + 1) {   // F_l^m (l+m) Q_{l-1}^m
                const double qz = TB.Gz[t] * Qc[l - 1];
                Szc = SPH_FMA(qz, wc, Szc);
                Szs = SPH_FMA(qz, ws, Szs);
            }
        });
        const double T1c = NORM ? S1c - Slc : S1c, T1s = NORM ? S1s - Sls : S1s;
        const double Tzc = NORM ? SPH_FMA(-zd, Slc, Szc) : Szc, Tzs = NORM ? SPH_FMA(-zd, Sls, Szs) : Szs;
        ax += SPH_FMA(xd * Ac, T1c, Acx * SQc) + SPH_FMA(xd * As, T1s, Asx * SQs);
        ay += SPH_FMA(yd * Ac, T1c, Acy * SQc) + SPH_FMA(yd * As, T1s, Asy * SQs);
        az = SPH_FMA(Ac, Tzc, SPH_FMA(As, Tzs, az));
        if constexpr (m < LMAX) {   // next column, next power of (x + i y): Eq. 9
            static_for<m + 1, LMAX + 1>([&](auto lc) { Qc[decltype(lc)::value] = Qn[decltype(lc)::value]; });
            c1 = cd;
            s1 = sd;
            const R cn = X * c - Y * s;
            const R sn = X * s + Y * c;
            c = cn;
            s = sn;
        }
    });
    if (NORM) {
        ax *= rinv;
        ay *= rinv;
        az *= rinv;
    }
    if (p < n) {
        gxyz[3 * p + 0] = static_cast<T>(ax);
        gxyz[3 * p + 1] = static_cast<T>(ay);
        gxyz[3 * p + 2] = static_cast<T>(az);
    }
}

}  // namespace sphb200
