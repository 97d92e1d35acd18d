// Fused density expansion (Eq. 1) for every l_max and n_rad the compile-time
// kernel of kernel_expand.cuh has no instantiation for (l_max > 8 or n_rad > 16), and for
// l_max <= 3, where that kernel's f32 image of the harmonics is too coarse for the tolerance:
//     c[s, n, lm] = sum over the points k of segment s of  R[k, n, l] * Y_l^m(r_k / |r_k|).
// One CTA per (segment, slice of the radial rows).  Per tile of PT points of the segment
//   1. thread = (point, column class): c_m, s_m by square-and-multiply (B2) and column m of
//      the folded Eq. 7 -- double for f32 I/O, double-double for f64 I/O -- for the columns
//      m = class, class + NCLS, ...; the harmonics go to a [PT][L] image in shared memory as f64;
//   2. thread = up to EXG_ACC output elements (n, lm) of the slice, accumulated in f64 registers
//      for the whole segment: one shared-memory read of Y and one cached read of R per term.
// The harmonics never reach HBM.  Run-time l_max and n_rad; slices re-evaluate the harmonics, so
// the kernel is at its best while n_rad * L <= 256 * EXG_ACC (one slice).
#pragma once
#include "ptx.cuh"
#include "sph_core.cuh"

namespace sphb200 {

constexpr int EXG_THREADS = 256;
constexpr int EXG_ACC = 24;   // output elements per thread

struct ExpandGenParams {
    const void* xyz;         // [n, 3]
    const void* radial;      // [n, n_rad, l_max+1]
    const int64_t* seg_ptr;  // [n_seg + 1]
    void* coeff;             // [n_seg, n_rad, L]
    int n_rad, l_max;
    int pts_tile;            // PT: points per tile (a power of two <= 32)
    int rows_per_slice;      // radial rows one CTA accumulates
};

template <typename T, typename R>
__global__ void __launch_bounds__(EXG_THREADS) sph_expand_generic_kernel(const ExpandGenParams prm, const SphTables* __restrict__ tab) {
    using RT = rec<R>;
    extern __shared__ __align__(16) unsigned char smem[];
    double* Ys = reinterpret_cast<double*>(smem);   // [PT][L]
    const int l_max = prm.l_max, L = (l_max + 1) * (l_max + 1), n_rad = prm.n_rad, PT = prm.pts_tile;
    const int64_t seg = blockIdx.x;
    const int n0 = blockIdx.y * prm.rows_per_slice;
    const int rows = min(prm.rows_per_slice, n_rad - n0);
    const int n_elem = rows * L;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    const T* __restrict__ radial = static_cast<const T*>(prm.radial);
    T* __restrict__ coeff = static_cast<T*>(prm.coeff);
    const int rstride = n_rad * (l_max + 1);
    const int64_t k_begin = prm.seg_ptr[seg], k_end = prm.seg_ptr[seg + 1];

    // this thread's output elements e = tid + j * THREADS of the slice: (n, lm) -> offsets into a point's
    // radial values and into a row of the Y image
    int roff[EXG_ACC], yoff[EXG_ACC];
    double acc[EXG_ACC];
#pragma unroll
    for (int j = 0; j < EXG_ACC; ++j) {
        const int e = threadIdx.x + j * EXG_THREADS;
        acc[j] = 0.0;
        roff[j] = -1;
        yoff[j] = 0;
        if (e < n_elem) {
            const int nl = e / L, lm = e - nl * L;
            int l = (int)sqrtf((float)lm);
            l += ((l + 1) * (l + 1) <= lm);
            l -= (l * l > lm);
            roff[j] = (n0 + nl) * (l_max + 1) + l;
            yoff[j] = lm;
        }
    }
    int nbits = 0;
    while ((1 << nbits) <= (l_max < 31 ? l_max : 31)) ++nbits;
    if (l_max == 32) nbits = 6;
    const int pt = threadIdx.x & (PT - 1), cls = threadIdx.x / PT, NCLS = EXG_THREADS / PT;

    for (int64_t k0 = k_begin; k0 < k_end; k0 += PT) {
        const int np = (int)min((int64_t)PT, k_end - k0);
        __syncthreads();   // the previous tile's contraction is done with the image
        if (pt < np) {
            const int64_t k = k0 + pt;
            R X, Y, Z;
            double rinv;
            RT::normalize(static_cast<double>(__ldg(xyz + 3 * k)), static_cast<double>(__ldg(xyz + 3 * k + 1)),
                          static_cast<double>(__ldg(xyz + 3 * k + 2)), X, Y, Z, rinv);
            const R one = RT::make(1.0, 0.0);
            double* Yp = Ys + pt * L;
            for (int m = cls; m <= l_max; m += NCLS) {
                R c, s;
                cs_power<R>(m, X, Y, nbits, c, s);
                const double cd = (m == 0) ? SPH_INV_SQRT2 : to_double(c), sd = to_double(s);
                R q = RT::make(tab->D_hi[m], tab->D_lo[m]), qp = RT::make(0.0, 0.0);
                for (int l = m;; ++l) {
                    const double Q = to_double(q);
                    Yp[l * (l + 1) + m] = Q * cd;            // Eq. 5, F folded into Q
                    if (m > 0) Yp[l * (l + 1) - m] = Q * sd;
                    if (l == l_max) break;
                    const R qn = column_step<R, true>(l + 1, m, Z, one, q, qp, *tab);
                    qp = q;
                    q = qn;
                }
            }
        }
        __syncthreads();
        for (int p = 0; p < np; ++p) {
            const T* __restrict__ Rp = radial + (k0 + p) * rstride;
            const double* __restrict__ Yp = Ys + p * L;
#pragma unroll
            for (int j = 0; j < EXG_ACC; ++j)
                if (roff[j] >= 0) acc[j] = fma(static_cast<double>(__ldg(Rp + roff[j])), Yp[yoff[j]], acc[j]);
        }
    }
#pragma unroll
    for (int j = 0; j < EXG_ACC; ++j) {
        const int e = threadIdx.x + j * EXG_THREADS;
        if (e < n_elem) coeff[(seg * n_rad + n0) * L + e] = static_cast<T>(acc[j]);
    }
}

}  // namespace sphb200
