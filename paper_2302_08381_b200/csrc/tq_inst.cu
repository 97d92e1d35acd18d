// One translation unit per element type of the tq kernels (kernel_tq.cuh), compiled twice by
// build.py with -DTQ_F64=0|1.  Exports (C++ linkage, declared in tpb_api.h):
//   sph_tq_upload_<f32|f64>(tables)   copy the coefficient tables into this unit's constant bank
//   sph_tq_launch_<f32|f64>(args)     pick a launch shape and launch; 1 if no shape fits, -1 CUDA error
#include "kernel_tv.cuh"
#include "tpb_api.h"

#ifndef TQ_F64
#error "compile with -DTQ_F64=0|1"
#endif

namespace sphb200 {

#if TQ_F64
typedef double tq_T;
typedef dd tq_R;
#define TQ_NAME(f) f##_f64
#else
typedef float tq_T;
typedef double tq_R;
#define TQ_NAME(f) f##_f32
#endif

typedef void (*TqKernel)(const TqParams);

template <int MODE, bool CONV> static TqKernel pick(int deriv, int norm) {
    if constexpr (MODE == 1) return norm ? sph_tq_kernel<tq_T, tq_R, 2, true, 1, false> : sph_tq_kernel<tq_T, tq_R, 2, false, 1, false>;
    else if constexpr (MODE == 2) return norm ? sph_tq_kernel<tq_T, tq_R, 1, true, 2, false> : sph_tq_kernel<tq_T, tq_R, 1, false, 2, false>;
    else {
        if (deriv == 0) return norm ? sph_tq_kernel<tq_T, tq_R, 0, true, 0, CONV> : sph_tq_kernel<tq_T, tq_R, 0, false, 0, CONV>;
        if (deriv == 1) return norm ? sph_tq_kernel<tq_T, tq_R, 1, true, 0, CONV> : sph_tq_kernel<tq_T, tq_R, 1, false, 0, CONV>;
        return norm ? sph_tq_kernel<tq_T, tq_R, 2, true, 0, CONV> : sph_tq_kernel<tq_T, tq_R, 2, false, 0, CONV>;
    }
}

template <bool CONV, int NPL> static TqKernel pick_direct(int deriv, int norm) {
    if (deriv == 0) return norm ? sph_tq_kernel<tq_T, tq_R, 0, true, 0, CONV, NPL> : sph_tq_kernel<tq_T, tq_R, 0, false, 0, CONV, NPL>;
    if (deriv == 1) return norm ? sph_tq_kernel<tq_T, tq_R, 1, true, 0, CONV, NPL> : sph_tq_kernel<tq_T, tq_R, 1, false, 0, CONV, NPL>;
    return norm ? sph_tq_kernel<tq_T, tq_R, 2, true, 0, CONV, NPL> : sph_tq_kernel<tq_T, tq_R, 2, false, 0, CONV, NPL>;
}

// Launch shape: points per phase-A batch B (32, 16, 8), points per tile P, warps per CTA W, images
// per CTA N.  The measured table (tq_table.h) first; the rules behind it serve the cells the table
// leaves to other kernels when tq is asked for anyway (forced, another convention, the contracting
// modes); the tq_* options override both.  The shape shrinks (N, then B, then P) until it fits.
// values-only kernel (kernel_tv.cuh): the largest batch that leaves room for two CTAs per SM (or fits at all)
static int tv_launch(const TqArgs& a) {
    const int esize = (int)sizeof(tq_T);
    const int budget = a.smem_optin - 1024;
    const unsigned char* shape = TV_SHAPE[TQ_F64][a.l_max];   // the measured table first (tq_table.h)
    int bB = g_opt.tq_batch > 0 ? g_opt.tq_batch : (shape[0] ? shape[0] : 32);
    if (g_opt.tq_batch <= 0 && !shape[0])
        while (bB > 8 && (int64_t)TvSmem(a.l_max, esize, bB).total > 100 * 1024) bB >>= 1;
    while (bB > 8 && (int64_t)TvSmem(a.l_max, esize, bB).total > budget) bB >>= 1;
    if ((bB != 32 && bB != 16 && bB != 8) || (int64_t)TvSmem(a.l_max, esize, bB).total > budget) return 1;
    const TvSmem lay(a.l_max, esize, bB);
    const int bW = g_opt.tq_warps > 0 && g_opt.tq_warps <= TQ_MAX_WARPS ? g_opt.tq_warps : (shape[0] ? shape[1] : 8);
    auto kern = a.normalized ? sph_tv_kernel<tq_T, tq_R, true> : sph_tv_kernel<tq_T, tq_R, false>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, a.smem_optin) != cudaSuccess) return -1;
    TvParams prm{};
    prm.xyz = a.xyz;
    prm.sph = a.sph;
    prm.ab_hi = a.d_ab;
    prm.ab_lo = a.d_ab + SPH_TRI_SIZE;
    prm.n = a.n;
    prm.l_max = a.l_max;
    prm.batch = bB;
    {   // f64 I/O: warps for Eq. 9 alone, balanced against the column warps (as for the two-phase kernel)
        const int NC = 32 / bB, T = (a.l_max + 1) * (a.l_max + 2) / 2;
        int best = 1;
        double best_t = 1e30;
        for (int wc = 1; wc <= 2 && wc < bW; ++wc) {
            const int nseg = wc * NC;
            int h = 1, sq = 0;
            while (2 * h * nseg <= a.l_max + nseg) h <<= 1, ++sq;
            const int last = a.l_max + 1 - (nseg - 1) * h;   // the last segment's length
            const double t_cs = 50.0 * (last > h ? last : h) + (nseg > 1 ? 40.0 * sq + 50.0 * (nseg - 2) : 0.0);
            const double t_col = 25.0 * T / ((bW - wc) * NC);
            const double t = t_cs > t_col ? t_cs : t_col;
            if (t < best_t) best_t = t, best = wc;
        }
        prm.cs_warps = g_opt.tq_cs_warps > 0 && g_opt.tq_cs_warps < bW ? g_opt.tq_cs_warps : (shape[0] ? shape[2] : best);
    }
    const int64_t n_batches = (a.n + bB - 1) / bB;
    int64_t bpc = n_batches / ((int64_t)a.sm_count * 16);   // several batches per CTA: the powers run one batch ahead
    if (bpc > 8) bpc = 8;
    if (bpc < 1) bpc = 1;
    prm.batches_per_cta = (int)bpc;
    const int64_t grid = (n_batches + bpc - 1) / bpc;
    if (grid > 0x7fffffff) return 1;
    kern<<<(unsigned)grid, bW * 32, lay.total, a.stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int TQ_NAME(sph_tq_launch)(const TqArgs& a) {
    if (a.mode == 3) return tv_launch(a);
    const int esize = (int)sizeof(tq_T);
    const int deriv = a.mode == 1 ? 2 : (a.mode == 2 ? 1 : a.deriv);
    const int rows = tq_img_rows(a.mode, deriv), ptb = tq_pt_bytes(a.mode);
    const int64_t L = (int64_t)(a.l_max + 1) * (a.l_max + 1);
    const int budget = a.smem_optin - 1024;
    const unsigned char* shape = TQ_SHAPE[TQ_F64][deriv][a.l_max];
    const bool tab = a.mode == 0 && shape[0] != 0;
    int bB = tab ? shape[0] : 32;
    int bP = tab ? shape[1] : ((int64_t)4 * rows * L * esize <= 24 * 1024 ? 4 : 2);
    int bW = tab ? shape[2] : 8;
    if (!tab && (a.l_max + 1) * (a.l_max + 2) / 2 <= 64) bP = 8, bW = 4;   // short triangles: fewer, fuller warps
    int bN = tab ? shape[3] : 1;
    // direct stores (no staging image): table entries {B, 0, W, 0 | 4} (two or four points per lane in phase B), or
    // the tq_direct option (1: on with two points per lane, 4: on with four, 2: off)
    bool direct = a.mode == 0 && ((tab && shape[1] == 0 && g_opt.tq_direct != 2) || g_opt.tq_direct == 1 || g_opt.tq_direct == 4);
    int npl = g_opt.tq_direct == 4 ? 4 : (g_opt.tq_direct == 0 && tab && shape[1] == 0 && shape[3] == 4 ? 4 : 2);
    if (tab && shape[1] == 0) bP = 2, bN = 1;   // (used only when tq_direct = 2 turns the entry's direct stores off)
    // Cells the table leaves to the unrolled kernels reach this one through sphericart_cuda_compute_ex (another
    // convention) or when forced.  Measured there (e3nn axes, l_max 1-11): direct stores from 32-point batches
    // with 2 warps (4 from l_max = 9) run 1.3-2.5x faster than the staged shapes above (f32 gradients
    // l_max 4 / 10: 1.7 / 1.9 -> 2.7 / 3.9 TB/s); f64 with derivatives prefers 16-point staged tiles.
    if (!tab && a.mode == 0 && g_opt.tq_direct == 0 && g_opt.tq_points == 0 && g_opt.tq_images == 0) {
        const int T = (a.l_max + 1) * (a.l_max + 2) / 2;
        bB = 32, bW = T <= 45 ? 2 : 4;
        if (TQ_F64 && deriv >= 1) bP = 16, bN = 1, bW = a.l_max <= 5 ? 2 : 4;
        else direct = true;
    }
    // contracting modes: little or nothing staged: tiles of 16 points (8 pairs x chunks divide evenly among 8 warps)
    if (a.mode != 0) bP = 16, bN = a.mode == 1 ? 2 : 1, bW = 8, bB = 32;
    if (g_opt.tq_batch > 0) bB = g_opt.tq_batch;
    if (g_opt.tq_points > 0) bP = g_opt.tq_points;
    if (g_opt.tq_warps > 0) bW = g_opt.tq_warps;
    if (g_opt.tq_images > 0 && a.mode != 2) bN = g_opt.tq_images;
    if (bW < 1 || bW > TQ_MAX_WARPS || (a.mode != 0 && bW > TQ_RED_WARPS) || bN < 1 || bN > 2) return 1;
    if (direct) bP = bB, bN = 1;
    if ((bB != 32 && bB != 16 && bB != 8) || bP > bB || bP < 1 || bB % bP != 0) return 1;
    auto bytes = [&](int B, int P, int N) { return (int64_t)TqSmem(a.l_max, deriv, rows, ptb, esize, B, P, N, direct).total; };
    const bool fixed = tab || g_opt.tq_batch > 0 || g_opt.tq_points > 0 || g_opt.tq_images > 0;
    if (!fixed)
        while (bB > 8 && bB / 2 >= bP && bytes(bB, bP, bN) > 110 * 1024) bB >>= 1;
    while (bytes(bB, bP, bN) > budget) {   // shrink until it fits: images, then the batch, then the tile
        if (bN == 2) bN = 1;
        else if (direct && bB > 8) bB >>= 1, bP = bB;
        else if (direct) return 1;
        else if (bB > 8 && bB / 2 >= bP) bB >>= 1;
        else if (bP > 1) bP >>= 1;
        else return 1;
    }
    const TqSmem lay(a.l_max, deriv, rows, ptb, esize, bB, bP, bN, direct);

    TqKernel kern = a.mode == 1 ? pick<1, false>(deriv, a.normalized)
                  : a.mode == 2 ? pick<2, false>(deriv, a.normalized)
                  : a.conv ? (direct ? (npl == 4 ? pick_direct<true, 4>(deriv, a.normalized) : pick_direct<true, 2>(deriv, a.normalized))
                                     : pick<0, true>(deriv, a.normalized))
                  : direct ? (npl == 4 ? pick_direct<false, 4>(deriv, a.normalized) : pick_direct<false, 2>(deriv, a.normalized))
                           : pick<0, false>(deriv, a.normalized);
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, a.smem_optin) != cudaSuccess) return -1;

    TqParams prm{};
    prm.xyz = a.xyz;
    prm.sph = a.sph;
    prm.dsph = a.dsph;
    prm.ddsph = a.ddsph;
    prm.gsph = a.gsph;
    prm.vvec = a.vvec;
    prm.gxyz = a.gxyz;
    prm.tab = a.d_tab;
    prm.lm = a.d_lm;
    prm.ab_hi = a.d_ab;
    prm.ab_lo = a.d_ab + SPH_TRI_SIZE;
    prm.n = a.n;
    prm.l_max = a.l_max;
    prm.batch = bB;
    prm.pts_tile = bP;
    prm.n_images = bN;
    {   // f64 I/O: one or two warps for Eq. 9 alone, whichever balances them against the column warps
        // (per lane: ~50 operations per power + ~40 per squaring against ~23 per Legendre entry)
        const int NC = 32 / bB, T = (a.l_max + 1) * (a.l_max + 2) / 2;
        int best = 1;
        double best_t = 1e30;
        for (int wc = 1; wc <= 2 && wc < bW; ++wc) {
            const int nseg = wc * NC;
            int h = 1, sq = 0;
            while (2 * h * nseg <= a.l_max + nseg) h <<= 1, ++sq;
            const int last = a.l_max + 1 - (nseg - 1) * h;   // the last segment's length
            const double t_cs = 50.0 * (last > h ? last : h) + (nseg > 1 ? 40.0 * sq + 50.0 * (nseg - 2) : 0.0);
            const double t_col = 23.0 * T / ((bW - wc) * NC);
            const double t = t_cs > t_col ? t_cs : t_col;
            if (t < best_t) best_t = t, best = wc;
        }
        prm.cs_warps = g_opt.tq_cs_warps > 0 && g_opt.tq_cs_warps < bW ? g_opt.tq_cs_warps : best;
    }
    for (int i = 0; i < 3; ++i) prm.src[i] = a.src[i], prm.row[i] = a.row[i];
    for (int l = 0; l <= SPH_MAX_L; ++l) prm.lscale[l] = a.lscale ? a.lscale[l] : 1.0;
    const int64_t n_batches = (a.n + bB - 1) / bB;
    // a few batches per CTA amortise the table copy; keep >= ~16 CTAs per SM for the block scheduler
    int64_t bpc = n_batches / ((int64_t)a.sm_count * 16);
    if (bpc > 4) bpc = 4;
    if (bpc < 1) bpc = 1;
    prm.batches_per_cta = (int)bpc;
    const int64_t grid = (n_batches + bpc - 1) / bpc;
    if (grid > 0x7fffffff) return 1;
    kern<<<(unsigned)grid, bW * 32, lay.total, a.stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int TQ_NAME(sph_tq_upload)(const SphTables* host_tables) {
    return cudaMemcpyToSymbol(c_tables_tq, host_tables, sizeof(SphTables)) == cudaSuccess ? 0 : -1;
}

}  // namespace sphb200
