// Fused density expansion (Eq. 1):
//     c[s, n, lm] = sum over the points k of segment s of  R[k, n, l] * Y_l^m(r_k / |r_k|)
// with the radial values R_nl(r_k) supplied by the caller (the paper leaves the radial basis to the
// application) and segments given by ascending offsets (e.g. the neighbour list of centre s).
// The harmonics never reach HBM: per point the kernel reads 3 + n_rad (l_max+1) values, and it
// writes n_rad L values per SEGMENT -- against L values written and read back per POINT when
// sphericart_cuda_compute is followed by a separate contraction.
//
// One warp per segment.  Per tile of 16 points of the segment
//   1. two lanes per point (cos | sin branch of Eq. 5, as in kernel_tpb.cuh, l_max compile-time)
//      evaluate the normalised harmonics into a [16][L] image in shared memory (f64 / double-double
//      recurrences, stored in the I/O type), while the tile's radial values ([16][n_rad][l_max+1],
//      one contiguous range) are copied next to it, widened to double ONCE here: the contraction
//      runs in f64 and reads every radial value 2l+1 times (ncu on the first version, which widened
//      each operand where it was used: the XU pipe of the f32->f64 conversions 63 % busy, the top
//      pipe of the kernel);
//   2. lane = harmonic index lm (ceil(L/32) passes): acc[pass][n] += R[p][n][l(lm)] * Y[p][lm] over
//      the tile's points, in f64 registers;
// and at the end of the segment the accumulators go out, coalesced along lm.
#pragma once
#include "kernel_tpb.cuh"

namespace sphb200 {

struct ExpandParams {
    const void* xyz;        // [n, 3]
    const void* radial;     // [n, n_rad, l_max+1]
    const int64_t* seg_ptr; // [n_seg + 1]
    void* coeff;            // [n_seg, n_rad, L]
    int64_t n_seg;
    int n_rad;
    int warps_per_cta;
};

constexpr int EXP_MAX_RAD = 16;   // accumulators per pass held in registers

template <int ESIZE, int LMAX> struct ExpandShape {
    static constexpr int L = (LMAX + 1) * (LMAX + 1);
    static constexpr int passes = (L + 31) / 32;
    // per warp: Y image [16][L] in the I/O type + radial image [16][n_rad][LMAX+1] in double, the
    // latter followed by nrad_max rows of padding (the unrolled contraction reads nrad_max rows per
    // point whatever n_rad is; what it reads past n_rad only feeds accumulators that are dropped)
    static constexpr int y_bytes = (TPB_PTS * L * ESIZE + 15) & ~15;
    __host__ __device__ static constexpr int r_bytes(int n_rad, int nrad_max) {
        return (TPB_PTS * n_rad + nrad_max) * (LMAX + 1) * 8;
    }
    __host__ __device__ static constexpr int warp_bytes(int n_rad, int nrad_max) { return y_bytes + r_bytes(n_rad, nrad_max); }
};

template <typename T, typename R, int LMAX, int NRAD_MAX>
__global__ void __launch_bounds__(128) sph_expand_kernel(const ExpandParams prm) {
    using RT = rec<R>;
    using Shape = ExpandShape<sizeof(T), LMAX>;
    constexpr int L = Shape::L;
    constexpr int PASSES = Shape::passes;
    const SphTables& TB = c_tables_tpb;
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int n_rad = prm.n_rad;
    const int64_t seg = (int64_t)blockIdx.x * prm.warps_per_cta + warp;
    if (seg >= prm.n_seg) return;
    unsigned char* my = smem + (size_t)warp * Shape::warp_bytes(n_rad, NRAD_MAX);
    T* Ys = reinterpret_cast<T*>(my);
    double* Rs = reinterpret_cast<double*>(my + Shape::y_bytes);
    const int pl = lane & (TPB_PTS - 1);   // point inside the tile
    const bool sinb = lane >= TPB_PTS;     // branch
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    const T* __restrict__ radial = static_cast<const T*>(prm.radial);
    T* __restrict__ coeff = static_cast<T*>(prm.coeff);
    const int64_t k_begin = prm.seg_ptr[seg], k_end = prm.seg_ptr[seg + 1];
    const int rstride = n_rad * (LMAX + 1);   // radial values per point

    // this lane's harmonics in the accumulation: lm = lane + 32 pass, and their degree l
    int l_of[PASSES];
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
        const int lm = lane + 32 * ps;
        int l = (int)sqrtf((float)lm);
        l += ((l + 1) * (l + 1) <= lm);
        l -= (l * l > lm);
        l_of[ps] = lm < L ? l : 0;
    }
    double acc[PASSES][NRAD_MAX];
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
        for (int nr = 0; nr < NRAD_MAX; ++nr) acc[ps][nr] = 0.0;

    for (int64_t k0 = k_begin; k0 < k_end; k0 += TPB_PTS) {
        const int np = (int)((k_end - k0 < TPB_PTS) ? k_end - k0 : TPB_PTS);
        __syncwarp();   // the previous tile's accumulation is done with both images
        // ---- radial values of the tile: one contiguous range -----------------------------------
        for (int i = lane; i < np * rstride; i += 32) Rs[i] = static_cast<double>(__ldg(radial + k0 * rstride + i));
        // ---- harmonics of the tile: two lanes per point ----------------------------------------
        double x = 0.0, y = 0.0, z = 1.0;  // lanes past the end compute a harmless point
        if (pl < np) {
            x = static_cast<double>(__ldg(xyz + 3 * (k0 + pl) + 0));
            y = static_cast<double>(__ldg(xyz + 3 * (k0 + pl) + 1));
            z = static_cast<double>(__ldg(xyz + 3 * (k0 + pl) + 2));
        }
        R X, Y, Z;
        double rinv;
        RT::normalize(x, y, z, X, Y, Z, rinv);
        T* S = Ys + pl * L;
        double Qc[LMAX + 1];
        R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
        static_for<0, LMAX + 1>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            // column m of the folded Eq. 7 (r^2 = 1 on the unit sphere), as in kernel_tpb.cuh
            {
                R q = RT::make(TB.D_hi[m], TB.D_lo[m]), qp = RT::make(0.0, 0.0);
                static_for<m, LMAX + 1>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    Qc[l] = to_double(q);
                    if constexpr (l < LMAX) {
                        constexpr int t1 = SPH_TRI(l + 1, m);
                        const R a = RT::make(TB.A_hi[t1], TB.A_lo[t1]);
                        R qn;
                        if constexpr (l == m) qn = a * (Z * q);
                        else qn = a * (Z * q) - RT::make(TB.B_hi[t1], TB.B_lo[t1]) * qp;
                        qp = q;
                        q = qn;
                    }
                });
            }
            const double A = sinb ? to_double(s) : (m == 0 ? SPH_INV_SQRT2 : to_double(c));
            const bool emit = (m > 0) || !sinb;   // the sin branch has no m = 0 output
            static_for<m, LMAX + 1>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                constexpr int kc = l * (l + 1) + m, ks = l * (l + 1) - m;
                if (emit) S[sinb ? ks : kc] = static_cast<T>(Qc[l] * A);   // Eq. 5
            });
            if constexpr (m < LMAX) {   // Eq. 9
                const R cn = X * c - Y * s;
                const R sn = X * s + Y * c;
                c = cn;
                s = sn;
            }
        });
        __syncwarp();
        // ---- accumulate: lane = harmonic, over the tile's points --------------------------------
        for (int p = 0; p < np; ++p) {
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps) {
                const int lm = lane + 32 * ps;
                if (lm < L) {
                    const double yv = static_cast<double>(Ys[p * L + lm]);
                    const double* rp = Rs + p * rstride + l_of[ps];
#pragma unroll
                    for (int nr = 0; nr < NRAD_MAX; ++nr) acc[ps][nr] = fma(rp[nr * (LMAX + 1)], yv, acc[ps][nr]);
                }
            }
        }
    }
    // ---- c[seg, n, lm], coalesced along lm ----------------------------------------------------------
#pragma unroll
    for (int nr = 0; nr < NRAD_MAX; ++nr) {
        if (nr < n_rad) {
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps) {
                const int lm = lane + 32 * ps;
                if (lm < L) coeff[(seg * n_rad + nr) * L + lm] = static_cast<T>(acc[ps][nr]);
            }
        }
    }
}

}  // namespace sphb200
