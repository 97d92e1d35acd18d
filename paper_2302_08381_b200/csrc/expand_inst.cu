// One translation unit per element type of the fused density-expansion kernels (kernel_expand.cuh),
// compiled twice by build.py with -DEXPAND_F64=0|1.  Exports (C++ linkage, declared in tpb_api.h):
//   sph_expand_upload_<f32|f64>(tables)   copy the coefficient tables into this unit's constant bank
//   sph_expand_launch_<f32|f64>(...)      launch if (l_max, n_rad) has an instantiation (returns 1 if not)
#include "kernel_expand.cuh"
#include "tpb_api.h"

#ifndef EXPAND_F64
#error "compile with -DEXPAND_F64=0|1"
#endif

namespace sphb200 {

#if EXPAND_F64
typedef double exp_T;
typedef dd exp_R;
#define EXP_NAME(f) f##_f64
#else
typedef float exp_T;
typedef double exp_R;
#define EXP_NAME(f) f##_f32
#endif

template <int LMAX, int NRAD_MAX> static int launch_nr(int smem_optin, ExpandParams prm, cudaStream_t stream) {
    using Shape = ExpandShape<sizeof(exp_T), LMAX>;
    auto kern = sph_expand_kernel<exp_T, exp_R, LMAX, NRAD_MAX>;
    int warps = 2;   // small CTAs: more of them fit beside each other in shared memory
    while (warps > 1 && warps * Shape::warp_bytes(prm.n_rad, NRAD_MAX) > smem_optin - 1024) warps >>= 1;
    const int smem = warps * Shape::warp_bytes(prm.n_rad, NRAD_MAX);
    if (smem > smem_optin - 1024) return 1;
    static int attr_bytes[64] = {0};   // per device: largest size granted so far (benign race, idempotent call)
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (dev < 0 || dev >= 64 || attr_bytes[dev] < smem) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
        if (dev >= 0 && dev < 64) attr_bytes[dev] = smem;
    }
    prm.warps_per_cta = warps;
    // persistent grid: as many CTAs as are resident at once (the kernel shares the segments among them by
    // point count), fewer when there are fewer segments than warps
    static int resident[64] = {0}, resident_smem[64] = {0};     // per device, for the last shared-memory size (benign race, idempotent)
    if (dev < 0 || dev >= 64) return -1;
    if (resident[dev] == 0 || resident_smem[dev] != smem) {
        int sms = 0, per_sm = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, warps * 32, smem) != cudaSuccess) return -1;
        if (per_sm < 1) per_sm = 1;
        resident[dev] = sms * per_sm;
        resident_smem[dev] = smem;
    }
    int64_t ctas = (prm.n_seg + warps - 1) / warps;
    if (ctas > resident[dev]) ctas = resident[dev];
    kern<<<(unsigned)ctas, warps * 32, smem, stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

template <int LMAX> static int launch_one(int smem_optin, const ExpandParams& prm, cudaStream_t stream) {
    if (prm.n_rad <= 8) return launch_nr<LMAX, 8>(smem_optin, prm, stream);
    if (prm.n_rad <= EXP_MAX_RAD) return launch_nr<LMAX, EXP_MAX_RAD>(smem_optin, prm, stream);
    return 1;
}

#define EXP_CASE(LM) \
    case LM:         \
        return launch_one<LM>(smem_optin, prm, stream);

int EXP_NAME(sph_expand_launch)(int smem_optin, const void* xyz, const void* radial, const int64_t* seg_ptr,
                                int64_t n_seg, int l_max, int n_rad, void* coeff, cudaStream_t stream) {
    ExpandParams prm{xyz, radial, seg_ptr, coeff, n_seg, n_rad, 4};
    switch (l_max) {
        EXP_CASE(0)
        EXP_CASE(1)
        EXP_CASE(2)
        EXP_CASE(3)
        EXP_CASE(4)
        EXP_CASE(5)
        EXP_CASE(6)
        EXP_CASE(7)
        EXP_CASE(8)
        default:
            return 1;
    }
}

int EXP_NAME(sph_expand_upload)(const SphTables* host_tables) {
    return cudaMemcpyToSymbol(c_tables_tpb, host_tables, sizeof(SphTables)) == cudaSuccess ? 0 : -1;
}

}  // namespace sphb200
