// One translation unit per (element type, DERIV) of the tpb kernels -- compiled four times by
// build.py with -DTPB_F64=0|1 -DTPB_DERIV=0|1|2 so that the instantiations build in parallel.
// Exports (C++ linkage, declared in tpb_api.h):
//   sph_tpb_upload_<f32|f64>_<v|g>(tables)   copy the coefficient tables into this unit's constant bank
//   sph_tpb_launch_<f32|f64>_<v|g>(...)      launch if l_max has an instantiation (returns 1 if not)
#include "kernel_tpb.cuh"
#include "options.h"
#include "tpb_api.h"

#ifndef TPB_F64
#error "compile with -DTPB_F64=0|1 -DTPB_DERIV=0|1"
#endif


namespace sphb200 {

#if TPB_F64
typedef double tpb_T;
typedef dd tpb_R;
#else
typedef float tpb_T;
typedef double tpb_R;
#endif

#if TPB_F64 && TPB_DERIV == 2
#define TPB_NAME(f) f##_f64_h
#elif TPB_DERIV == 2
#define TPB_NAME(f) f##_f32_h
#elif TPB_F64 && TPB_DERIV
#define TPB_NAME(f) f##_f64_g
#elif TPB_F64
#define TPB_NAME(f) f##_f64_v
#elif TPB_DERIV
#define TPB_NAME(f) f##_f32_g
#else
#define TPB_NAME(f) f##_f32_v
#endif


template <int LMAX, bool NORM, int SPLIT, bool BB = false>
static int launch_split(int sm_count, TpbParams prm, cudaStream_t stream) {
    using Shape = TpbShape<sizeof(tpb_T), TPB_DERIV, LMAX, SPLIT, BB>;
    static_assert(Shape::fit >= 1, "tile does not fit in shared memory");
    auto kern = sph_tpb_kernel<tpb_T, tpb_R, TPB_DERIV, NORM, LMAX, SPLIT, BB>;
    static bool attr_done[64] = {false};   // per device; benign race (idempotent call)
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (dev >= 0 && dev < 64 && !attr_done[dev]) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Shape::tile_bytes) != cudaSuccess)
            return -1;
        attr_done[dev] = true;
    }
    // One tile per CTA where a tile is >= ~12 KB (C3: 166 us against 172 us with four tiles, C5 with
    // gradients: 476 against 508): the CTA launch is cheap next to such a tile.  Small tiles (values
    // only, low l_max) take up to four per CTA, or the launch rate of the block scheduler shows
    // (C5 values only, 3.1 KB tiles: 170 us with one, 147 with two, 136 with four or eight).
    const int64_t n_tiles = (prm.n + Shape::pts - 1) / Shape::pts;
    const int k_env = g_opt.tpb_tiles;
    int64_t k = k_env > 0 ? k_env : 12288 / Shape::tile_bytes;
    if (k < 1) k = 1;
    if (k_env <= 0 && k > 4) k = 4;
    prm.tiles_per_cta = (int)k;
    const int64_t ctas = (n_tiles + k - 1) / k;
    if (ctas > 0x7fffffff) return 1;
    // Programmatic dependent launch: the CTAs of this grid may become resident while the previous
    // kernel in the stream drains; each waits (griddepcontrol.wait, first thing in the kernel) until
    // that kernel has completed and its memory is visible, so stream order is kept for ANY
    // predecessor.  It hides the launch ramp between back-to-back calls (C2: 22.8 -> 20.8 us).  Only
    // for grids of a few waves: the two griddepcontrol instructions cost every CTA a fixed latency,
    // which a grid of 250 000 one-tile CTAs cannot hide (C5 values only: 169 -> 261 us with them).
    const int pdl = g_opt.pdl && ctas <= (int64_t)sm_count * 64;
    prm.pdl = pdl;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ctas);
    cfg.blockDim = dim3(SPLIT * 32);
    cfg.dynamicSmemBytes = Shape::tile_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, prm) == cudaSuccess ? 0 : -1;
}

// Two warps per tile where shared memory, not registers, limits the tiles in flight (<= 12 per
// SM): the second warp then fills issue slots that would idle and halves a tile's latency.
// Measured: C2 24.7 -> 22.8 us, C3 166 -> 164 us; C5 (17 tiles fit) 476 -> 562 us, so not there.
template <int LMAX, bool NORM>
static int launch_one(int sm_count, const TpbParams& prm, cudaStream_t stream) {
    const int split_env = g_opt.tpb_split;
    // One lane per point doing both branches of Eq. 5 (32-point tiles) where the Legendre recurrences
    // dominate, i.e. values only: f64 (double-double recurrences) up to l_max = 13, f32 up to 10, and
    // f64 gradients up to l_max = 4.  Measured: f64 values l_max 4/6/8: 2.9/3.2/3.4 -> 5.2/6.1/5.3
    // TB/s, f32 values l_max 2/4/6: 2.8/4.8/5.1 -> 4.2/5.3/5.9; with Hessians it loses (f64
    // l_max = 4: 7.0 -> 4.7), so not there.
    constexpr bool bb = TPB_DERIV == 0 ? (TPB_F64 ? LMAX <= 13 : LMAX <= 10) : (TPB_DERIV == 1 && TPB_F64 && LMAX <= 4);
    if constexpr (bb) {
        // f64 values, l_max 8-12: ONE warp per tile although few tiles fit (its ~250 registers hold every
        // column's running pair; two warps at 128 registers each re-load them).  Measured, one / two warps:
        // l_max 8: 6.2 / 5.9 TB/s, 10: 5.6-6.0 / 4.5-4.9, 12: 3.9-4.3 / 3.5-3.8; l_max 13: 3.3-3.6 either way.
        constexpr bool one = TPB_F64 && TPB_DERIV == 0 && LMAX >= 8 && LMAX <= 12;
        constexpr bool s2 = LMAX >= 4 && !one && TpbShape<sizeof(tpb_T), TPB_DERIV, LMAX, 1, true>::fit <= 12;
        if constexpr (s2) {
            if (split_env != 1) return launch_split<LMAX, NORM, 2, true>(sm_count, prm, stream);
        } else if constexpr (LMAX >= 4) {
            if (split_env == 2) return launch_split<LMAX, NORM, 2, true>(sm_count, prm, stream);
        }
        return launch_split<LMAX, NORM, 1, true>(sm_count, prm, stream);
    } else {
        constexpr bool can_split = LMAX >= 4;
        if constexpr (can_split) {
            // (long value-only rows: one warp per tile would need > 128 registers at 13+ tiles per SM and spills)
            // Two cells measured faster with one warp: f32 values l_max 19 (3.8 against 3.4 TB/s), f32 Hessians
            // l_max 4 (7.1 against 6.6).
            constexpr bool one = !TPB_F64 && ((TPB_DERIV == 0 && LMAX == 19) || (TPB_DERIV == 2 && LMAX == 4));
            constexpr bool dflt = !one && (TpbShape<sizeof(tpb_T), TPB_DERIV, LMAX, 1>::fit <= 12 || (TPB_DERIV == 0 && LMAX >= 13));
            const bool want = split_env ? split_env == 2 : dflt;
            if (want) return launch_split<LMAX, NORM, 2>(sm_count, prm, stream);
        }
        return launch_split<LMAX, NORM, 1>(sm_count, prm, stream);
    }
}

#define TPB_CASE(LM) \
    case LM:         \
        return normalized ? launch_one<LM, true>(sm_count, prm, stream) : launch_one<LM, false>(sm_count, prm, stream);

int TPB_NAME(sph_tpb_launch)(int sm_count, const void* xyz, int64_t n, int l_max, int normalized, void* sph,
                             void* dsph, void* ddsph, cudaStream_t stream) {
    TpbParams prm{xyz, sph, dsph, ddsph, n, 1, 0};
    switch (l_max) {
        TPB_CASE(1)
        TPB_CASE(2)
        TPB_CASE(3)
        TPB_CASE(4)
        TPB_CASE(5)
        TPB_CASE(6)
#if TPB_DERIV < 2 || !TPB_F64   // Hessians: f32 up to l_max = 8, f64 up to 6 (a 16-point tile must fit)
        TPB_CASE(7)
        TPB_CASE(8)
#endif
#if TPB_DERIV < 2
#if !TPB_F64 || !TPB_DERIV    // f32 (C3 is l_max = 16 values) and f64 values: up to l_max = 16 / 12
        TPB_CASE(9)
        TPB_CASE(10)
        TPB_CASE(11)
        TPB_CASE(12)
#endif
#if !TPB_F64 || !TPB_DERIV   // (f64 values: up to l_max = 13)
        TPB_CASE(13)
#endif
#if !TPB_F64
        TPB_CASE(14)
        TPB_CASE(15)
        TPB_CASE(16)
#endif
#if !TPB_F64 && !TPB_DERIV     // f32 values: up to l_max = 23 (from 24 on the run-time kernel is as fast)
        TPB_CASE(17)
        TPB_CASE(18)
        TPB_CASE(19)
        TPB_CASE(20)
        TPB_CASE(21)
        TPB_CASE(22)
        TPB_CASE(23)
#endif
#endif
        default:
            return 1;
    }
}

int TPB_NAME(sph_tpb_upload)(const SphTables* host_tables) {
    return cudaMemcpyToSymbol(c_tables_tpb, host_tables, sizeof(SphTables)) == cudaSuccess ? 0 : -1;
}

}  // namespace sphb200
