// Launch options of the library: compiled-in defaults, changed only through
// sphericart_cuda_set_option (include/sphericart_cuda.h) by test harnesses and experiments.
// Nothing on the call path reads the environment.
#pragma once
#include <cstdint>

namespace sphb200 {

enum ForceKernel {
    FORCE_NONE = 0,   // default dispatch
    FORCE_TPB,        // compile-time-l_max kernels only where they exist (same as default)
    FORCE_TPG,        // several lanes per point, run-time l_max
    FORCE_W,          // warp-per-point family (wc where it applies by default)
    FORCE_W1,         // one-warp-per-point kernel even for the longest rows
    FORCE_WC,         // CTA-cooperative kernel wherever it can run (l_max >= 19)
    FORCE_TQ,         // two-phase kernel (kernel_tq.cuh) wherever it can run
    FORCE_TV,         // values-only kernel (kernel_tv.cuh) wherever it can run
    FORCE_GENERIC,    // recompute VJP / expansion: the run-time-l_max kernels
};

struct SphOptions {
    int force_kernel = FORCE_NONE;
    int tpg_lp = 0;          // lanes per point of the tpg kernel (0: chosen from the row length)
    int w_nbuf = 1;          // staging images per warp of the w kernel
    int w_warps = 0;         // warps per CTA of the w kernel (0: as many as fit)
    int w_ppw = 0;           // points per warp and CTA of the w kernel (0: from n)
    int wc_min_l = 0;        // smallest l_max the wc kernel takes (0: the dispatch's own rule)
    int vjp_warps = 0;       // warps per CTA of the stored-derivative VJP kernel (0: as many as fit)
    int tpb_tiles = 0;       // tiles per CTA of the tpb kernels (0: from the tile size)
    int tpb_split = 0;       // warps per tile of the tpb kernels (0: the dispatch's own rule)
    int pdl = 1;             // programmatic dependent launch for small grids
    int tq_points = 0;       // points per tile of the tq kernel (0: the planner's choice)
    int tq_warps = 0;        // warps per CTA of the tq kernel (0: the planner's choice)
    int tq_images = 0;       // staging images per CTA of the tq kernel (0: two unless only one fits)
    int tq_cs_warps = 0;     // f64 I/O: warps of the tq kernel's recurrence phase that run Eq. 9 only (0: balanced by the planner)
    int tq_direct = 0;       // tq forward: 1 / 4 = store straight to global memory (no staging image), two / four points per lane; 2 = never; 0 = the table's choice
    int tq_batch = 0;        // points per phase-A batch of the tq kernel (0: the planner's choice)
    int64_t host_chunk_bytes = (int64_t)256 << 20;   // _host entry points: bytes per chunk and stream
};

extern SphOptions g_opt;     // api.cu

}  // namespace sphb200
