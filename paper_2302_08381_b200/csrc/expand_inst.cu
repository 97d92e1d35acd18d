// One translation unit per element type of the fused density-expansion kernels (kernel_expand.cuh),
// compiled twice by build.py with -DEXPAND_F64=0|1.  Exports (C++ linkage, declared in tpb_api.h):
//   sph_expand_upload_<f32|f64>(tables)   copy the coefficient tables into this unit's constant bank
//   sph_expand_launch_<f32|f64>(...)      launch if (l_max, n_rad) has an instantiation (returns 1 if not)
//   sph_expand_rt_launch_<f32|f64>(...)   the run-time-l_max kernel: any l_max <= 32, n_rad <= 16 (returns 1 if not)
#include "kernel_expand_rt.cuh"
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

// Run-time l_max (kernel_expand_rt.cuh): the degrees are packed greedily into bands of at most NTB N-tiles
// (a degree l has ceil((2l+1)/8) of them), one CTA row per band.
template <int MT, int NTB> static int launch_rt(int smem_optin, ExpandRtParams prm, cudaStream_t stream) {
    using Shape = ExpandRtShape<sizeof(exp_T), NTB>;
    auto kern = sph_expand_rt_kernel<exp_T, exp_R, MT, NTB>;
    static_assert(NTB <= EXRT_MAX_NTB, "tile descriptors");
    int nb = 0, tiles = 0, col = 0;
    for (int l = 0; l <= prm.l_max; ++l) {
        const int tl = (2 * l + 1 + 7) / 8;
        if (nb == 0 || tiles + tl > NTB) {
            if (nb == EXRT_MAX_BANDS) return 1;
            prm.band_l0[nb++] = (unsigned char)l;
            tiles = 0;
            col = 0;
        }
        for (int sub = 0; sub < tl; ++sub)
            prm.tile_desc[nb - 1][tiles + sub] = (uint32_t)l | ((uint32_t)sub << 6) | ((uint32_t)(col + 8 * sub) << 10);
        tiles += tl;
        col += 2 * l + 1;
        prm.band_l1[nb - 1] = (unsigned char)l;
        prm.band_tiles[nb - 1] = (unsigned char)tiles;
    }
    prm.n_bands = nb;
    int warps = 2;
    while (warps > 1 && warps * Shape::warp_bytes(prm.n_rad, prm.l_max, 8 * MT) > smem_optin - 1024) warps >>= 1;
    const int smem = warps * Shape::warp_bytes(prm.n_rad, prm.l_max, 8 * MT);
    if (smem > smem_optin - 1024) return 1;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return -1;
    static int attr_bytes[64] = {0}, resident[64] = {0}, resident_smem[64] = {0};   // per device (benign races, idempotent)
    if (attr_bytes[dev] < smem) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
        attr_bytes[dev] = smem;
    }
    if (resident[dev] == 0 || resident_smem[dev] != smem) {
        int sms = 0, per_sm = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, warps * 32, smem) != cudaSuccess) return -1;
        resident[dev] = sms * (per_sm < 1 ? 1 : per_sm);
        resident_smem[dev] = smem;
    }
    prm.warps_per_cta = warps;
    // a few CTAs per resident slot and band: the bands cost differently (a higher band runs longer
    // recurrences), the block scheduler evens them out
    int64_t ctas = ((int64_t)4 * resident[dev] + nb - 1) / nb;
    const int64_t most = (prm.n_seg + warps - 1) / warps;
    if (ctas > most) ctas = most;
    if (ctas < 1) ctas = 1;
    kern<<<dim3((unsigned)ctas, (unsigned)nb), warps * 32, smem, stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int EXP_NAME(sph_expand_rt_launch)(int smem_optin, const void* xyz, const void* radial, const int64_t* seg_ptr,
                                   int64_t n_seg, int l_max, int n_rad, void* coeff, cudaStream_t stream) {
    ExpandRtParams prm{};
    prm.xyz = xyz;
    prm.radial = radial;
    prm.seg_ptr = seg_ptr;
    prm.coeff = coeff;
    prm.n_seg = n_seg;
    prm.n_rad = n_rad;
    prm.l_max = l_max;
    if (n_rad <= 8) return launch_rt<1, 16>(smem_optin, prm, stream);
    if (n_rad <= 16) return launch_rt<2, 9>(smem_optin, prm, stream);   // (l = 32 alone has 9 N-tiles)
    return 1;
}

int EXP_NAME(sph_expand_upload)(const SphTables* host_tables) {
    return cudaMemcpyToSymbol(c_tables_tpb, host_tables, sizeof(SphTables)) == cudaSuccess ? 0 : -1;
}

}  // namespace sphb200
