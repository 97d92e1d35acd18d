// One translation unit per element type of the recompute-in-backward VJP kernels (kernel_vjpr.cuh),
// compiled twice by build.py with -DVJPR_F64=0|1.  Exports (C++ linkage, declared in tpb_api.h):
//   sph_vjpr_upload_<f32|f64>(tables)   copy the coefficient tables into this unit's constant bank
//   sph_vjpr_launch_<f32|f64>(...)      launch if l_max has an instantiation (returns 1 if not)
#include "kernel_vjpr.cuh"
#include "options.h"
#include "tpb_api.h"

#ifndef VJPR_F64
#error "compile with -DVJPR_F64=0|1"
#endif

namespace sphb200 {

#if VJPR_F64
typedef double vjpr_T;
typedef dd vjpr_R;
#define VJPR_NAME(f) f##_f64
#else
typedef float vjpr_T;
typedef double vjpr_R;
#define VJPR_NAME(f) f##_f32
#endif

template <int LMAX, bool NORM> static int launch_one(int sm_count, VjprParams prm, cudaStream_t stream) {
    constexpr int L = (LMAX + 1) * (LMAX + 1);
    constexpr int smem = 32 * L * (int)sizeof(vjpr_T) + 16;   // 32 points per tile
    auto kern = sph_vjpr_kernel<vjpr_T, vjpr_R, NORM, LMAX>;
    static bool attr_done[64] = {false};   // per device; benign race (idempotent call)
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (dev >= 0 && dev < 64 && !attr_done[dev]) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
        attr_done[dev] = true;
    }
    const int64_t n_tiles = (prm.n + 31) / 32;
    if (n_tiles > 0x7fffffff) return 1;
    // programmatic dependent launch, as for the forward kernels (tpb_inst.cu)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_tiles);
    cfg.blockDim = dim3(32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    prm.pdl = g_opt.pdl && n_tiles <= (int64_t)sm_count * 64;   // small grids only (tpb_inst.cu)
    cfg.numAttrs = prm.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, prm) == cudaSuccess ? 0 : -1;
}

#define VJPR_CASE(LM) \
    case LM:          \
        return normalized ? launch_one<LM, true>(sm_count, prm, stream) : launch_one<LM, false>(sm_count, prm, stream);

int VJPR_NAME(sph_vjpr_launch)(int sm_count, const void* xyz, const void* grad_sph, void* grad_xyz, int64_t n, int l_max,
                               int normalized, cudaStream_t stream) {
    VjprParams prm{xyz, grad_sph, grad_xyz, n, 0};
    switch (l_max) {
        VJPR_CASE(1)
        VJPR_CASE(2)
        VJPR_CASE(3)
        VJPR_CASE(4)
        VJPR_CASE(5)
        VJPR_CASE(6)
        VJPR_CASE(7)
        VJPR_CASE(8)
#if !VJPR_F64
        VJPR_CASE(9)
        VJPR_CASE(10)
        VJPR_CASE(11)
        VJPR_CASE(12)
#endif
        default:
            return 1;
    }
}

int VJPR_NAME(sph_vjpr_upload)(const SphTables* host_tables) {
    return cudaMemcpyToSymbol(c_tables_tpb, host_tables, sizeof(SphTables)) == cudaSuccess ? 0 : -1;
}

}  // namespace sphb200
