// One translation unit per (element type, DERIV) of the tpb kernels -- compiled four times by
// build.py with -DTPB_F64=0|1 -DTPB_DERIV=0|1 so that the instantiations build in parallel.
// Exports (C++ linkage, declared in tpb_api.h):
//   sph_tpb_upload_<f32|f64>_<v|g>(tables)   copy the coefficient tables into this unit's constant bank
//   sph_tpb_launch_<f32|f64>_<v|g>(...)      launch if l_max has an instantiation (returns 1 if not)
#include "kernel_tpb.cuh"
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

#if TPB_F64 && TPB_DERIV
#define TPB_NAME(f) f##_f64_g
#elif TPB_F64
#define TPB_NAME(f) f##_f64_v
#elif TPB_DERIV
#define TPB_NAME(f) f##_f32_g
#else
#define TPB_NAME(f) f##_f32_v
#endif

template <int LMAX, bool NORM>
static int launch_one(int sm_count, const TpbParams& prm, cudaStream_t stream) {
    using Shape = TpbShape<sizeof(tpb_T), TPB_DERIV, LMAX>;
    static_assert(Shape::warps >= 1, "tile does not fit in shared memory");
    auto kern = sph_tpb_kernel<tpb_T, tpb_R, TPB_DERIV, NORM, LMAX>;
    static bool attr_done[64] = {false};   // per device; benign race (idempotent call)
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (dev >= 0 && dev < 64 && !attr_done[dev]) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Shape::smem) != cudaSuccess)
            return -1;
        attr_done[dev] = true;
    }
    const int64_t n_tiles = (prm.n + TPB_PTS - 1) / TPB_PTS;
    int64_t ctas = (n_tiles + Shape::warps - 1) / Shape::warps;
    if (ctas > sm_count) ctas = sm_count;
    kern<<<(int)ctas, Shape::warps * 32, Shape::smem, stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

#define TPB_CASE(LM) \
    case LM:         \
        return normalized ? launch_one<LM, true>(sm_count, prm, stream) : launch_one<LM, false>(sm_count, prm, stream);

int TPB_NAME(sph_tpb_launch)(int sm_count, const void* xyz, int64_t n, int l_max, int normalized, void* sph,
                             void* dsph, cudaStream_t stream) {
    TpbParams prm{xyz, sph, dsph, n};
    switch (l_max) {
        TPB_CASE(1)
        TPB_CASE(2)
        TPB_CASE(3)
        TPB_CASE(4)
        TPB_CASE(5)
        TPB_CASE(6)
        TPB_CASE(7)
        TPB_CASE(8)
#if !TPB_DERIV && !TPB_F64   // long value-only rows: f32 only (C3 is l_max = 16)
        TPB_CASE(9)
        TPB_CASE(10)
        TPB_CASE(11)
        TPB_CASE(12)
        TPB_CASE(13)
        TPB_CASE(14)
        TPB_CASE(15)
        TPB_CASE(16)
#endif
        default:
            return 1;
    }
}

int TPB_NAME(sph_tpb_upload)(const SphTables* host_tables) {
    return cudaMemcpyToSymbol(c_tables_tpb, host_tables, sizeof(SphTables)) == cudaSuccess ? 0 : -1;
}

}  // namespace sphb200
