// Host entry points of the tpb translation units (tpb_inst.cu, compiled once per element type
// and derivative order).  Return: 0 launched, 1 no instantiation for this l_max, -1 CUDA error.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tables.h"

namespace sphb200 {
#define SPH_TPB_DECL(sfx)                                                                                   \
    int sph_tpb_launch_##sfx(int sm_count, const void* xyz, int64_t n, int l_max, int normalized, void* sph, \
                             void* dsph, void* ddsph, cudaStream_t stream);                                              \
    int sph_tpb_upload_##sfx(const SphTables* host_tables);
SPH_TPB_DECL(f32_v)
SPH_TPB_DECL(f32_g)
SPH_TPB_DECL(f64_v)
SPH_TPB_DECL(f64_g)
SPH_TPB_DECL(f32_h)
SPH_TPB_DECL(f64_h)
#undef SPH_TPB_DECL
// recompute-in-backward VJP (vjpr_inst.cu, compiled once per element type); same return codes
#define SPH_VJPR_DECL(sfx)                                                                              \
    int sph_vjpr_launch_##sfx(int sm_count, const void* xyz, const void* grad_sph, void* grad_xyz, int64_t n, int l_max, \
                              int normalized, cudaStream_t stream);                                      \
    int sph_vjpr_upload_##sfx(const SphTables* host_tables);
SPH_VJPR_DECL(f32)
SPH_VJPR_DECL(f64)
#undef SPH_VJPR_DECL
// fused density expansion of Eq. 1 (expand_inst.cu, compiled once per element type); same return codes
#define SPH_EXPAND_DECL(sfx)                                                                                   \
    int sph_expand_launch_##sfx(int smem_optin, const void* xyz, const void* radial, const int64_t* seg_ptr,  \
                                int64_t n_seg, int l_max, int n_rad, void* coeff, cudaStream_t stream);       \
    int sph_expand_upload_##sfx(const SphTables* host_tables);                                                \
    /* run-time l_max <= 32, n_rad <= 16 (kernel_expand_rt.cuh): 1 if n_rad is larger, -1 CUDA error */      \
    int sph_expand_rt_launch_##sfx(int smem_optin, const void* xyz, const void* radial, const int64_t* seg_ptr, \
                                   int64_t n_seg, int l_max, int n_rad, void* coeff, cudaStream_t stream);
SPH_EXPAND_DECL(f32)
SPH_EXPAND_DECL(f64)
#undef SPH_EXPAND_DECL
// two-phase kernel (tq_inst.cu, compiled once per element type); same return codes
struct TqArgs {
    int sm_count, smem_optin;
    int mode;          // 0 forward, 1 second-order VJP, 2 recompute VJP, 3 forward values only (kernel_tv.cuh)
    int deriv;         // mode 0: 0 values, 1 + gradients, 2 + Hessians
    int normalized;
    int conv;          // mode 0: another axis / scale convention (src, row, lscale)
    const void* xyz;
    void* sph;         // mode 0: sph; mode 1: grad_grad_sph (may be NULL)
    void* dsph;
    void* ddsph;
    const void* gsph;  // modes 1, 2
    const void* vvec;  // mode 1
    void* gxyz;        // modes 1, 2
    int64_t n;
    int l_max;
    const SphTables* d_tab;
    const unsigned short* d_lm;
    const double2* d_ab;
    int src[3], row[3];
    const double* lscale;   // [SPH_MAX_L + 1] or NULL
    cudaStream_t stream;
};
int sph_tq_launch_f32(const TqArgs& a);
int sph_tq_launch_f64(const TqArgs& a);
int sph_tq_upload_f32(const SphTables* host_tables);
int sph_tq_upload_f64(const SphTables* host_tables);
}  // namespace sphb200
