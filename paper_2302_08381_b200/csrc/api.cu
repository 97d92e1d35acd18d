// C ABI of the library (include/sphericart_cuda.h): argument checks, one-time per-device setup,
// kernel selection and launch.  No torch types, no exceptions across the boundary.
#include "../../include/sphericart_cuda.h"

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include <cuda_runtime.h>

#include "options.h"
#include "ptx.cuh"
#include "sph_core.cuh"
#include "tables.h"
namespace sphb200 {
// constant-bank copy of the coefficient tables for the kernels of this translation unit
__constant__ SphTables c_tables;
}  // namespace sphb200

#include "kernel_vjp.cuh"
#include "kernel_expand_generic.cuh"
#include "kernel_tpg.cuh"
#include "tq_table.h"
#include "kernel_w.cuh"
#include "kernel_wc.cuh"
#include "tpb_api.h"

namespace sphb200 {

SphOptions g_opt;   // options.h

static thread_local char g_err[512] = "";
static thread_local const char* g_last_kernel = "";
static std::atomic<int64_t> g_launches{0};

static void launched(const char* family) {
    g_last_kernel = family;
    g_launches.fetch_add(1, std::memory_order_relaxed);
}

static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(call)                                                                      \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(SPHERICART_CUDA_ECUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

// ---------------------------------------------------------------------------------------------
// per-device state
// ---------------------------------------------------------------------------------------------
constexpr int MAX_DEVICES = 64;
struct DeviceState {
    bool ready = false;
    std::atomic<bool> ready_flag{false};
    int sm_count = 0;
    int smem_optin = 0;          // max dynamic shared memory per block
    SphTables* d_tables = nullptr;   // copy of the tables in global memory (warp kernel)
    unsigned short* d_lm = nullptr;  // (l | m << 8) of every triangle index (tq kernel)
    double2* d_ab = nullptr;         // {A_hi, B_hi}[t], then {A_lo, B_lo}[t] (tq kernel)
};
static DeviceState g_dev[MAX_DEVICES];
static std::mutex g_mutex;
static SphTables g_host_tables;
static std::once_flag g_tables_once;

static int device_state(DeviceState** out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(SPHERICART_CUDA_ECUDA, "device index %d out of range", dev);
    DeviceState& st = g_dev[dev];
    if (st.ready_flag.load(std::memory_order_acquire)) {   // the common case takes no lock
        *out = &st;
        return 0;
    }
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!st.ready) {
        std::call_once(g_tables_once, [] { sph_build_tables(&g_host_tables); });
        cudaDeviceProp prop;
        CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
        if (prop.major < 10)
            return fail(SPHERICART_CUDA_ECUDA, "device %d is sm_%d%d; this library is built for sm_100a only",
                        dev, prop.major, prop.minor);
        st.sm_count = prop.multiProcessorCount;
        st.smem_optin = (int)prop.sharedMemPerBlockOptin;
        CUDA_TRY(cudaMemcpyToSymbol(c_tables, &g_host_tables, sizeof(SphTables)));
        if (sph_tpb_upload_f32_v(&g_host_tables) || sph_tpb_upload_f32_g(&g_host_tables) ||
            sph_tpb_upload_f64_v(&g_host_tables) || sph_tpb_upload_f64_g(&g_host_tables) ||
            sph_tpb_upload_f32_h(&g_host_tables) || sph_tpb_upload_f64_h(&g_host_tables) ||
            sph_vjpr_upload_f32(&g_host_tables) || sph_vjpr_upload_f64(&g_host_tables) ||
            sph_expand_upload_f32(&g_host_tables) || sph_expand_upload_f64(&g_host_tables) ||
            sph_tq_upload_f32(&g_host_tables) || sph_tq_upload_f64(&g_host_tables))
            return fail(SPHERICART_CUDA_ECUDA, "table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        CUDA_TRY(cudaMalloc(&st.d_tables, sizeof(SphTables)));
        CUDA_TRY(cudaMemcpy(st.d_tables, &g_host_tables, sizeof(SphTables), cudaMemcpyHostToDevice));
        static unsigned short lm[SPH_TRI_SIZE];
        for (int l = 0; l <= SPH_MAX_L; ++l)
            for (int m = 0; m <= l; ++m) lm[SPH_TRI(l, m)] = (unsigned short)(l | (m << 8));
        CUDA_TRY(cudaMalloc(&st.d_lm, sizeof(lm)));
        CUDA_TRY(cudaMemcpy(st.d_lm, lm, sizeof(lm), cudaMemcpyHostToDevice));
        static double2 ab[2 * SPH_TRI_SIZE];
        for (int t = 0; t < SPH_TRI_SIZE; ++t) {
            ab[t] = make_double2(g_host_tables.A_hi[t], g_host_tables.B_hi[t]);
            ab[SPH_TRI_SIZE + t] = make_double2(g_host_tables.A_lo[t], g_host_tables.B_lo[t]);
        }
        CUDA_TRY(cudaMalloc(&st.d_ab, sizeof(ab)));
        CUDA_TRY(cudaMemcpy(st.d_ab, ab, sizeof(ab), cudaMemcpyHostToDevice));
        st.ready = true;
        st.ready_flag.store(true, std::memory_order_release);
    }
    *out = &st;
    return 0;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (device, kernel)
constexpr int MAX_OPTIN_KERNELS = 512;   // more than the instantiations api.cu can launch
static int allow_smem(const void* func, int bytes) {
    static std::mutex m;
    static const void* done[MAX_DEVICES][MAX_OPTIN_KERNELS];
    static int n_done[MAX_DEVICES];
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(m);
    for (int i = 0; i < n_done[dev]; ++i)
        if (done[dev][i] == func) return 0;
    (void)bytes;
    CUDA_TRY(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, g_dev[dev].smem_optin));
    if (n_done[dev] >= MAX_OPTIN_KERNELS)
        return fail(SPHERICART_CUDA_ECUDA, "internal: more than %d opt-in kernels", MAX_OPTIN_KERNELS);
    done[dev][n_done[dev]++] = func;
    return 0;
}

// ---------------------------------------------------------------------------------------------
// forward: warp-per-point kernel (any l_max <= 32, Hessians)
// ---------------------------------------------------------------------------------------------
static int launch_w(const DeviceState& st, const void* xyz, int64_t n, int l_max, int normalized, int dtype,
                    void* sph, void* dsph, void* ddsph, cudaStream_t stream) {
    if (g_opt.force_kernel != FORCE_W1) {
        // the longest f64 rows: the warps of a CTA share one point, chunks of a third of a row, ~3 KB
        // bulk stores (kernel_wc.cuh says where it wins); FORCE_WC takes it wherever it can run
        const bool force_wc = g_opt.force_kernel == FORCE_WC;
        // (default: f64 with Hessians from l_max = 29 -- 5.1-5.8 TB/s at 38 k points against 4.2 of the two-phase
        // kernel's one-point tiles, which win below -- and every f64 output set at l_max = 32)
        int min_l = force_wc ? 19 : (dtype == SPHERICART_CUDA_F64 ? (ddsph ? 29 : 32) : SPHERICART_CUDA_MAX_L + 1);
        if (g_opt.wc_min_l > 0) min_l = g_opt.wc_min_l;
        WcLaunch lc{};
        if (wc_plan(min_l, st.sm_count, st.smem_optin, n, l_max, normalized, dtype, sph, dsph, ddsph, xyz, st.d_tables, &lc) == 0) {
            int rc = allow_smem(lc.func, (int)lc.smem);
            if (rc) return rc;
            wc_launch(lc, stream);
            launched("wc");
            CUDA_TRY(cudaGetLastError());
            return 0;
        }
    }
    WkLaunch lw{};
    int rc = wk_plan(st.sm_count, st.smem_optin, n, l_max, normalized, dtype, sph, dsph, ddsph, xyz,
                     st.d_tables, &lw);
    if (rc) return fail(SPHERICART_CUDA_ECUDA, "warp kernel: no launch configuration fits (l_max=%d)", l_max);
    rc = allow_smem(lw.func, (int)lw.smem);
    if (rc) return rc;
    wk_launch(lw, stream);
    launched("w");
    CUDA_TRY(cudaGetLastError());
    return 0;
}

// ---------------------------------------------------------------------------------------------
// two-phase kernel (tq_inst.cu): forward (optionally in another convention), second-order VJP,
// recompute VJP.  Returns 0 launched, 1 no shape fits, -1 CUDA error.
// ---------------------------------------------------------------------------------------------
struct TqConv {
    int src[3], row[3];
    double lscale[SPH_MAX_L + 1];
};
static int launch_tq(const DeviceState& st, int mode, int normalized, int dtype, const TqConv* conv, const void* xyz,
                     void* sph, void* dsph, void* ddsph, const void* gsph, const void* vvec, void* gxyz, int64_t n,
                     int l_max, cudaStream_t stream) {
    TqArgs a{};
    a.sm_count = st.sm_count;
    a.smem_optin = st.smem_optin;
    a.mode = mode;
    a.deriv = ddsph ? 2 : (dsph ? 1 : 0);
    a.normalized = normalized;
    a.conv = conv != nullptr;
    a.xyz = xyz;
    a.sph = sph;
    a.dsph = dsph;
    a.ddsph = ddsph;
    a.gsph = gsph;
    a.vvec = vvec;
    a.gxyz = gxyz;
    a.n = n;
    a.l_max = l_max;
    a.d_tab = st.d_tables;
    a.d_lm = st.d_lm;
    a.d_ab = st.d_ab;
    for (int i = 0; i < 3; ++i) a.src[i] = conv ? conv->src[i] : i, a.row[i] = conv ? conv->row[i] : i;
    a.lscale = conv ? conv->lscale : nullptr;
    a.stream = stream;
    const int r = dtype == SPHERICART_CUDA_F32 ? sph_tq_launch_f32(a) : sph_tq_launch_f64(a);
    if (r == 0) launched(mode == 0 ? "tq" : (mode == 1 ? "tq_vjp2" : (mode == 2 ? "tq_vjpr" : "tv")));
    return r;
}

// where the values-only kernel (kernel_tv.cuh) beats the other families (measured: tq_table.h)
static bool tv_wins(int dtype, int l_max) { return TV_SHAPE[dtype != 0][l_max][0] != 0; }

static bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

static int check_common(int64_t n, int l_max, int dtype) {
    if (n < 0) return fail(SPHERICART_CUDA_EINVAL, "n = %lld is negative", (long long)n);
    if (l_max < 0 || l_max > SPHERICART_CUDA_MAX_L)
        return fail(SPHERICART_CUDA_EINVAL, "l_max = %d outside [0, %d]", l_max, SPHERICART_CUDA_MAX_L);
    if (dtype != SPHERICART_CUDA_F32 && dtype != SPHERICART_CUDA_F64)
        return fail(SPHERICART_CUDA_EINVAL, "dtype = %d is neither 0 (f32) nor 1 (f64)", dtype);
    return 0;
}

static int compute_device(const void* xyz, int64_t n, int l_max, int normalized, int dtype, void* sph,
                          void* dsph, void* ddsph, cudaStream_t stream) {
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (normalized != 0 && normalized != 1)
        return fail(SPHERICART_CUDA_EINVAL, "normalized = %d is neither 0 nor 1", normalized);
    if (ddsph && !dsph) return fail(SPHERICART_CUDA_EINVAL, "ddsph given without dsph");
    if (n == 0) return 0;
    if (!xyz || !sph) return fail(SPHERICART_CUDA_EINVAL, "xyz and sph must not be NULL when n > 0");
    if (misaligned(xyz) || misaligned(sph) || misaligned(dsph) || misaligned(ddsph))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned");
    DeviceState* st = nullptr;
    rc = device_state(&st);
    if (rc) return rc;

    const int force = g_opt.force_kernel;
    const bool force_w = force == FORCE_W || force == FORCE_W1 || force == FORCE_WC;
    if (!dsph && (force == FORCE_TV || (force == FORCE_NONE && tv_wins(dtype, l_max)))) {
        // values only: every Legendre entry straight into the image (kernel_tv.cuh)
        const int r = launch_tq(*st, 3, normalized, dtype, nullptr, xyz, sph, nullptr, nullptr, nullptr, nullptr, nullptr, n, l_max,
                                stream);
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "tv launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) return 0;
    }
    if (force == FORCE_TQ || (force == FORCE_NONE && TQ_SHAPE[dtype != 0][ddsph ? 2 : (dsph ? 1 : 0)][l_max][0])) {
        // two-phase kernel: recurrences lane = point, assembly lane = (l, m) pair, small full-row tiles
        const int r = launch_tq(*st, 0, normalized, dtype, nullptr, xyz, sph, dsph, ddsph, nullptr, nullptr, nullptr, n, l_max,
                                stream);
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "tq launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) return 0;
    }
    if (force == FORCE_NONE || force == FORCE_TPB) {
        // compile-time-l_max kernels (two threads per point): every l_max that has an instantiation
        const bool f32 = dtype == SPHERICART_CUDA_F32;
        auto launch = ddsph ? (f32 ? sph_tpb_launch_f32_h : sph_tpb_launch_f64_h)
                            : dsph ? (f32 ? sph_tpb_launch_f32_g : sph_tpb_launch_f64_g)
                                   : (f32 ? sph_tpb_launch_f32_v : sph_tpb_launch_f64_v);
        int r = launch(st->sm_count, xyz, n, l_max, normalized, sph, dsph, ddsph, stream);
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "tpb launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) {
            launched("tpb");
            return 0;
        }
    }
    if (!ddsph && !force_w) {
        // any other l_max without Hessians: several lanes per point, run-time l_max
        TpgLaunch lg{};
        if (tpg_plan(st->smem_optin, n, l_max, normalized, dtype, sph, dsph, xyz, st->d_tables, &lg) == 0) {
            rc = allow_smem(lg.func, (int)lg.smem);
            if (rc) return rc;
            tpg_launch(lg, stream);
            launched("tpg");
            CUDA_TRY(cudaGetLastError());
            return 0;
        }
    }
    return launch_w(*st, xyz, n, l_max, normalized, dtype, sph, dsph, ddsph, stream);
}

// ---------------------------------------------------------------------------------------------
// recompute-in-backward VJP, any l_max: one thread per point, runtime l_max, grad_sph read straight
// from global memory.  The compile-time-l_max kernels of kernel_vjpr.cuh cover the l_max that
// matter for speed; this one keeps the entry point total.
// ---------------------------------------------------------------------------------------------
template <typename T> struct VjprEmit {
    const T* w;
    double a[3];
    __device__ __forceinline__ void val(int, double) {}
    __device__ __forceinline__ void grad(int c, int k, double v) { a[c] = fma(v, static_cast<double>(w[k]), a[c]); }
};

template <typename T, typename R, bool NORM>
__global__ void __launch_bounds__(128) sph_vjpr_generic_kernel(const T* __restrict__ xyz, const T* __restrict__ gsph,
                                                               T* __restrict__ gxyz, int64_t n, int l_max) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int L = (l_max + 1) * (l_max + 1);
    VjprEmit<T> e{gsph + p * L, {0.0, 0.0, 0.0}};
    eval_point_columns<R, 1, NORM>(static_cast<double>(xyz[3 * p]), static_cast<double>(xyz[3 * p + 1]),
                                   static_cast<double>(xyz[3 * p + 2]), l_max, c_tables, e);
    gxyz[3 * p + 0] = static_cast<T>(e.a[0]);
    gxyz[3 * p + 1] = static_cast<T>(e.a[1]);
    gxyz[3 * p + 2] = static_cast<T>(e.a[2]);
}

static int vjp_recompute_device(const void* xyz, const void* grad_sph, void* grad_xyz, int64_t n, int l_max,
                                int normalized, int dtype, cudaStream_t stream) {
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (normalized != 0 && normalized != 1)
        return fail(SPHERICART_CUDA_EINVAL, "normalized = %d is neither 0 nor 1", normalized);
    if (n == 0) return 0;
    if (!xyz || !grad_sph || !grad_xyz)
        return fail(SPHERICART_CUDA_EINVAL, "xyz, grad_sph and grad_xyz must not be NULL when n > 0");
    if (misaligned(xyz) || misaligned(grad_sph) || misaligned(grad_xyz))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned");
    DeviceState* st = nullptr;
    rc = device_state(&st);
    if (rc) return rc;
    const bool f32 = dtype == SPHERICART_CUDA_F32;
    if (g_opt.force_kernel != FORCE_GENERIC) {
        int r = (f32 ? sph_vjpr_launch_f32 : sph_vjpr_launch_f64)(st->sm_count, xyz, grad_sph, grad_xyz, n, l_max, normalized, stream);
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "vjpr launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) {
            launched("vjpr");
            return 0;
        }
    }
    if (g_opt.force_kernel != FORCE_GENERIC) {
        // every other l_max: the two-phase kernel, gradients contracted with grad_sph as they are assembled
        const int r = launch_tq(*st, 2, normalized, dtype, nullptr, xyz, nullptr, nullptr, nullptr, grad_sph, nullptr, grad_xyz,
                                n, l_max, stream);
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "tq launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) return 0;
    }
    const int64_t blocks = (n + 127) / 128;
    if (blocks > 0x7fffffff) return fail(SPHERICART_CUDA_EINVAL, "n = %lld is too large", (long long)n);
    if (f32) {
        auto k = normalized ? sph_vjpr_generic_kernel<float, double, true> : sph_vjpr_generic_kernel<float, double, false>;
        k<<<(unsigned)blocks, 128, 0, stream>>>((const float*)xyz, (const float*)grad_sph, (float*)grad_xyz, n, l_max);
    } else {
        auto k = normalized ? sph_vjpr_generic_kernel<double, dd, true> : sph_vjpr_generic_kernel<double, dd, false>;
        k<<<(unsigned)blocks, 128, 0, stream>>>((const double*)xyz, (const double*)grad_sph, (double*)grad_xyz, n, l_max);
    }
    launched("vjpr_generic");
    CUDA_TRY(cudaGetLastError());
    return 0;
}

static int vjp_device(const void* dsph, const void* grad_sph, void* grad_xyz, int64_t n, int l_max, int dtype,
                      cudaStream_t stream) {
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (n == 0) return 0;
    if (!dsph || !grad_sph || !grad_xyz)
        return fail(SPHERICART_CUDA_EINVAL, "dsph, grad_sph and grad_xyz must not be NULL when n > 0");
    if (misaligned(dsph) || misaligned(grad_sph) || misaligned(grad_xyz))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned");
    DeviceState* st = nullptr;
    rc = device_state(&st);
    if (rc) return rc;

    const int L = (l_max + 1) * (l_max + 1);
    const int esize = dtype == SPHERICART_CUDA_F32 ? 4 : 8;
    VjpParams prm{};
    prm.dsph = dsph;
    prm.grad_sph = grad_sph;
    prm.grad_xyz = grad_xyz;
    prm.n = n;
    prm.L = L;
    prm.tile_bytes = 4u * 32u * L * esize;
    const int budget = st->smem_optin - 1024;
    int warps = (int)(budget / ((int64_t)VJP_NBUF * prm.tile_bytes + VJP_NBUF * 8));
    const int want = g_opt.vjp_warps > 0 ? g_opt.vjp_warps : VJP_MAX_THREADS / 32;
    if (warps > want) warps = want;
    const int64_t n_tiles = (n + 31) / 32;
    void (*kern)(const VjpParams);
    if (warps >= 1) {
        kern = dtype == SPHERICART_CUDA_F32 ? sph_vjp_kernel<float> : sph_vjp_kernel<double>;
    } else {
        // rows too long to stage a 32-point tile: warp-per-point streaming kernel
        if (wk_launch_vjp(st->sm_count, dsph, grad_sph, grad_xyz, n, L, dtype, stream) == 0) {
            launched("vjp_warp");
            return 0;
        }
        return fail(SPHERICART_CUDA_ECUDA, "vjp launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    int64_t per_sm = (n_tiles + st->sm_count - 1) / st->sm_count;
    if (per_sm < warps) warps = (int)(per_sm < 1 ? 1 : per_sm);
    int64_t ctas = (n_tiles + warps - 1) / warps;
    if (ctas > st->sm_count) ctas = st->sm_count;
    prm.warps_per_cta = warps;
    const size_t smem = (size_t)warps * VJP_NBUF * (prm.tile_bytes + 8);
    rc = allow_smem((const void*)kern, (int)smem);
    if (rc) return rc;
    kern<<<(int)ctas, warps * 32, smem, stream>>>(prm);
    launched("vjp");
    CUDA_TRY(cudaGetLastError());
    return 0;
}

// ---------------------------------------------------------------------------------------------
// host-buffer entry points: chunked, two streams, transfers overlap compute
// ---------------------------------------------------------------------------------------------
struct HostWs {  // grow-only device workspace, one set per stream slot
    void* buf[2][5] = {{nullptr}};
    size_t cap[2][5] = {{0}};
    cudaStream_t stream[2] = {nullptr, nullptr};
    int device = -1;
};
static HostWs g_ws;
static std::mutex g_ws_mutex;

static int ws_reserve(int slot, int which, size_t bytes) {
    if (g_ws.cap[slot][which] >= bytes) return 0;
    if (g_ws.buf[slot][which]) cudaFree(g_ws.buf[slot][which]);
    g_ws.buf[slot][which] = nullptr;
    g_ws.cap[slot][which] = 0;
    if (cudaMalloc(&g_ws.buf[slot][which], bytes) != cudaSuccess) {
        cudaGetLastError();
        return fail(SPHERICART_CUDA_ENOMEM, "cudaMalloc of %zu bytes failed", bytes);
    }
    g_ws.cap[slot][which] = bytes;
    return 0;
}

static int ws_streams() {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (g_ws.device != dev) {
        for (int s = 0; s < 2; ++s) {
            for (int w = 0; w < 5; ++w) {
                if (g_ws.buf[s][w]) cudaFree(g_ws.buf[s][w]);
                g_ws.buf[s][w] = nullptr;
                g_ws.cap[s][w] = 0;
            }
            if (g_ws.stream[s]) cudaStreamDestroy(g_ws.stream[s]);
            CUDA_TRY(cudaStreamCreateWithFlags(&g_ws.stream[s], cudaStreamNonBlocking));
        }
        g_ws.device = dev;
    }
    return 0;
}

// points per chunk so that one chunk's buffers stay near `target` bytes
static int64_t chunk_points(int64_t n, size_t bytes_per_point, size_t target) {
    int64_t c = (int64_t)(target / (bytes_per_point ? bytes_per_point : 1));
    c &= ~(int64_t)31;
    if (c < 32) c = 32;
    return c < n ? c : n;
}

// ---------------------------------------------------------------------------------------------
// sphericart_cuda_vjp_noalloc: the stored-derivative VJP for callers that must not allocate
// ---------------------------------------------------------------------------------------------
// A split-row variant of sph_vjp_warp_kernel (kernel_w.cuh): a point's row of L harmonics is cut into
// S slices, one warp per (point, slice), so that a SMALL batch with long rows still fills the machine;
// the warps' partial sums (3 doubles per point and slice) go through a scratch in global memory and a
// second kernel adds the S slices of every point in a fixed order (deterministic).  The scratch is a
// file-scope array of the library image: every GPU that loads the library holds its
// SPHERICART_CUDA_NOALLOC_SCRATCH_BYTES until the process exits, and the call allocates nothing.
// The array's name is a host-side stand-in in host code; the kernels get the address that
// cudaGetSymbolAddress returns for the current device (noalloc_state below).
constexpr int NOALLOC_MAX_SLICES = 8;
static_assert(SPHERICART_CUDA_NOALLOC_SCRATCH_BYTES ==
                  (size_t)SPHERICART_CUDA_NOALLOC_MAX_POINTS * NOALLOC_MAX_SLICES * 3 * sizeof(double),
              "scratch size = max points x max slices x 3 partial sums");
static __device__ __align__(256) unsigned char g_noalloc_scratch[SPHERICART_CUDA_NOALLOC_SCRATCH_BYTES];

// partial[(s * n + p) * 3 + a] = sum over slice s of dsph[p, a, k] * grad_sph[p, k]
template <typename T>
__global__ void __launch_bounds__(256) sph_vjp_split_kernel(const T* __restrict__ dsph, const T* __restrict__ gsph,
                                                            double* __restrict__ partial, int64_t n, int L, int S) {
    const int lane = threadIdx.x & 31;
    const int64_t unit = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);   // (point, slice)
    if (unit >= n * S) return;
    const int64_t p = unit / S;
    const int s = (int)(unit - p * S);
    const int k0 = (int)((int64_t)L * s / S), k1 = (int)((int64_t)L * (s + 1) / S);
    const T* g = gsph + p * L;
    const T* d = dsph + p * 3 * L;
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int k = k0 + lane; k < k1; k += 32) {
        const double w = static_cast<double>(__ldcs(g + k));
        ax = fma(static_cast<double>(__ldcs(d + k)), w, ax);
        ay = fma(static_cast<double>(__ldcs(d + L + k)), w, ay);
        az = fma(static_cast<double>(__ldcs(d + 2 * L + k)), w, az);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, o);
        ay += __shfl_xor_sync(0xffffffffu, ay, o);
        az += __shfl_xor_sync(0xffffffffu, az, o);
    }
    if (lane == 0) {
        double* out = partial + ((int64_t)s * n + p) * 3;
        out[0] = ax;
        out[1] = ay;
        out[2] = az;
    }
}

// grad_xyz[p, a] = sum_s partial[s][p][a], slices in ascending order
template <typename T>
__global__ void __launch_bounds__(256) sph_vjp_split_sum_kernel(const double* __restrict__ partial, T* __restrict__ gxyz,
                                                                int64_t n, int S) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // = 3 p + a
    if (i >= 3 * n) return;
    double sum = 0.0;
    for (int s = 0; s < S; ++s) sum += partial[(int64_t)s * n * 3 + i];
    gxyz[i] = static_cast<T>(sum);
}

struct NoallocState {
    std::atomic<bool> ready{false};
    int sm_count = 0;
    double* scratch = nullptr;   // DEVICE address of g_noalloc_scratch on this device
};
static NoallocState g_noalloc[MAX_DEVICES];

// once per device, with that device current; no allocation (no cudaMalloc, no stream, no event)
static int noalloc_state(NoallocState** out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(SPHERICART_CUDA_ECUDA, "device index %d out of range", dev);
    NoallocState& st = g_noalloc[dev];
    if (!st.ready.load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!st.ready.load(std::memory_order_relaxed)) {
            int major = 0;
            CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
            if (major < 10)
                return fail(SPHERICART_CUDA_ECUDA, "device %d is sm_%dx; this library is built for sm_100a only", dev, major);
            CUDA_TRY(cudaDeviceGetAttribute(&st.sm_count, cudaDevAttrMultiProcessorCount, dev));
            void* ptr = nullptr;
            CUDA_TRY(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
            if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u))
                return fail(SPHERICART_CUDA_ECUDA, "cudaGetSymbolAddress returned %p for the scratch array", ptr);
            st.scratch = static_cast<double*>(ptr);
            st.ready.store(true, std::memory_order_release);
        }
    }
    *out = &st;
    return 0;
}

static int vjp_noalloc_device(const void* dsph, const void* grad_sph, void* grad_xyz, int64_t n, int l_max, int dtype,
                              cudaStream_t stream) {
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (n > SPHERICART_CUDA_NOALLOC_MAX_POINTS)
        return fail(SPHERICART_CUDA_EINVAL,
                    "vjp_noalloc: n = %lld exceeds SPHERICART_CUDA_NOALLOC_MAX_POINTS = %d (the static scratch holds "
                    "no more); split the batch or call sphericart_cuda_vjp",
                    (long long)n, SPHERICART_CUDA_NOALLOC_MAX_POINTS);
    if (n == 0) return 0;
    if (!dsph || !grad_sph || !grad_xyz)
        return fail(SPHERICART_CUDA_EINVAL, "dsph, grad_sph and grad_xyz must not be NULL when n > 0");
    if (misaligned(dsph) || misaligned(grad_sph) || misaligned(grad_xyz))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned");
    NoallocState* st = nullptr;
    rc = noalloc_state(&st);
    if (rc) return rc;
    const int L = (l_max + 1) * (l_max + 1);
    // slices: enough (point, slice) warps for ~16 per SM, at least 32 harmonics per slice
    int S = (int)(((int64_t)st->sm_count * 16 + n - 1) / n);
    if (S > L / 32) S = L / 32;
    if (S > NOALLOC_MAX_SLICES) S = NOALLOC_MAX_SLICES;
    if (S < 1) S = 1;
    const int64_t units = n * S;
    const int warps_per_cta = 8;
    const int64_t ctas = (units + warps_per_cta - 1) / warps_per_cta;
    const int64_t sum_ctas = (3 * n + 255) / 256;
    if (dtype == SPHERICART_CUDA_F32) {
        sph_vjp_split_kernel<float><<<(unsigned)ctas, warps_per_cta * 32, 0, stream>>>(
            static_cast<const float*>(dsph), static_cast<const float*>(grad_sph), st->scratch, n, L, S);
        sph_vjp_split_sum_kernel<float><<<(unsigned)sum_ctas, 256, 0, stream>>>(st->scratch, static_cast<float*>(grad_xyz), n, S);
    } else {
        sph_vjp_split_kernel<double><<<(unsigned)ctas, warps_per_cta * 32, 0, stream>>>(
            static_cast<const double*>(dsph), static_cast<const double*>(grad_sph), st->scratch, n, L, S);
        sph_vjp_split_sum_kernel<double><<<(unsigned)sum_ctas, 256, 0, stream>>>(st->scratch, static_cast<double*>(grad_xyz), n, S);
    }
    launched("vjp_split");
    launched("vjp_split_sum");
    CUDA_TRY(cudaGetLastError());
    return 0;
}

}  // namespace sphb200

using namespace sphb200;

extern "C" {

int sphericart_cuda_compute(const void* xyz, int64_t n, int l_max, int normalized, int dtype, void* sph,
                            void* dsph, void* ddsph, void* stream) {
    return compute_device(xyz, n, l_max, normalized, dtype, sph, dsph, ddsph, static_cast<cudaStream_t>(stream));
}

int sphericart_cuda_vjp(const void* xyz, const void* dsph, const void* grad_sph, void* grad_xyz, int64_t n,
                        int l_max, int dtype, void* stream) {
    (void)xyz;  // reserved (reading B1)
    return vjp_device(dsph, grad_sph, grad_xyz, n, l_max, dtype, static_cast<cudaStream_t>(stream));
}

int sphericart_cuda_vjp_recompute(const void* xyz, const void* grad_sph, void* grad_xyz, int64_t n, int l_max,
                                  int normalized, int dtype, void* stream) {
    return vjp_recompute_device(xyz, grad_sph, grad_xyz, n, l_max, normalized, dtype,
                                static_cast<cudaStream_t>(stream));
}

int sphericart_cuda_compute_ex(const void* xyz, int64_t n, int l_max, int normalized, int dtype, int axes, int scale,
                               void* sph, void* dsph, void* ddsph, void* stream) {
    if (axes != SPHERICART_CUDA_AXES_STANDARD && axes != SPHERICART_CUDA_AXES_E3NN)
        return fail(SPHERICART_CUDA_EINVAL, "axes = %d is neither 0 (standard) nor 1 (e3nn)", axes);
    if (scale < SPHERICART_CUDA_SCALE_INTEGRAL || scale > SPHERICART_CUDA_SCALE_NORM)
        return fail(SPHERICART_CUDA_EINVAL, "scale = %d is not 0 (integral), 1 (component) or 2 (norm)", scale);
    if (axes == SPHERICART_CUDA_AXES_STANDARD && scale == SPHERICART_CUDA_SCALE_INTEGRAL)
        return compute_device(xyz, n, l_max, normalized, dtype, sph, dsph, ddsph, static_cast<cudaStream_t>(stream));
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (normalized != 0 && normalized != 1)
        return fail(SPHERICART_CUDA_EINVAL, "normalized = %d is neither 0 nor 1", normalized);
    if (ddsph && !dsph) return fail(SPHERICART_CUDA_EINVAL, "ddsph given without dsph");
    if (n == 0) return 0;
    if (!xyz || !sph) return fail(SPHERICART_CUDA_EINVAL, "xyz and sph must not be NULL when n > 0");
    if (misaligned(xyz) || misaligned(sph) || misaligned(dsph) || misaligned(ddsph))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned");
    DeviceState* st = nullptr;
    rc = device_state(&st);
    if (rc) return rc;
    TqConv conv;
    const bool e3nn = axes == SPHERICART_CUDA_AXES_E3NN;
    // e3nn axes: the evaluation frame is (x', y', z') = (z, x, y) of the caller's point, so axis a of
    // the evaluation frame is the caller's axis src[a]
    const int src[3] = {e3nn ? 2 : 0, e3nn ? 0 : 1, e3nn ? 1 : 2};
    for (int i = 0; i < 3; ++i) conv.src[i] = conv.row[i] = src[i];
    const double four_pi = 12.566370614359172953850573533118;
    for (int l = 0; l <= SPH_MAX_L; ++l)
        conv.lscale[l] = scale == SPHERICART_CUDA_SCALE_INTEGRAL ? 1.0
                       : scale == SPHERICART_CUDA_SCALE_COMPONENT ? sqrt(four_pi) : sqrt(four_pi / (2 * l + 1));
    const int r = launch_tq(*st, 0, normalized, dtype, &conv, xyz, sph, dsph, ddsph, nullptr, nullptr, nullptr, n, l_max,
                            static_cast<cudaStream_t>(stream));
    if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "tq launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    if (r > 0) return fail(SPHERICART_CUDA_ENOTSUP, "compute_ex: rows of l_max = %d with these outputs do not fit the kernel", l_max);
    return 0;
}

int sphericart_cuda_vjp2(const void* xyz, const void* grad_sph, const void* v, void* grad_grad_xyz, void* grad_grad_sph,
                         int64_t n, int l_max, int normalized, int dtype, void* stream) {
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (normalized != 0 && normalized != 1)
        return fail(SPHERICART_CUDA_EINVAL, "normalized = %d is neither 0 nor 1", normalized);
    if (n == 0) return 0;
    if (!xyz || !grad_sph || !v || !grad_grad_xyz)
        return fail(SPHERICART_CUDA_EINVAL, "xyz, grad_sph, v and grad_grad_xyz must not be NULL when n > 0");
    if (misaligned(xyz) || misaligned(grad_sph) || misaligned(v) || misaligned(grad_grad_xyz) || misaligned(grad_grad_sph))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned");
    DeviceState* st = nullptr;
    rc = device_state(&st);
    if (rc) return rc;
    const int r = launch_tq(*st, 1, normalized, dtype, nullptr, xyz, grad_grad_sph, nullptr, nullptr, grad_sph, v, grad_grad_xyz,
                            n, l_max, static_cast<cudaStream_t>(stream));
    if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "tq launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    if (r > 0) return fail(SPHERICART_CUDA_ENOTSUP, "vjp2: l_max = %d does not fit the kernel", l_max);
    return 0;
}

int sphericart_cuda_expand(const void* xyz, const void* radial, const int64_t* seg_ptr, int64_t n_seg, int l_max,
                           int n_rad, int dtype, void* coeff, void* stream) {
    int rc = check_common(n_seg, l_max, dtype);
    if (rc) return rc;
    if (n_rad < 1) return fail(SPHERICART_CUDA_EINVAL, "n_rad = %d must be at least 1", n_rad);
    if (n_seg == 0) return 0;
    if (!seg_ptr || !coeff) return fail(SPHERICART_CUDA_EINVAL, "seg_ptr and coeff must not be NULL when n_seg > 0");
    // (xyz and radial are read for the points of non-empty segments only: both may be NULL when every
    // segment is empty, i.e. seg_ptr[n_seg] = 0, which the host cannot see without a synchronisation)
    if ((xyz == nullptr) != (radial == nullptr))
        return fail(SPHERICART_CUDA_EINVAL, "xyz and radial must both be given, or both be NULL when there are no points");
    if (misaligned(xyz) || misaligned(radial) || misaligned(coeff) || (reinterpret_cast<uintptr_t>(seg_ptr) & 7u))
        return fail(SPHERICART_CUDA_EALIGN, "device pointers must be 16-byte aligned (seg_ptr: 8)");
    DeviceState* st = nullptr;
    rc = device_state(&st);
    if (rc) return rc;
    // the compile-time kernel (DMMA contraction) where it has an instantiation (l_max <= 8, n_rad <= 16)
    if (g_opt.force_kernel != FORCE_GENERIC) {
        const int r = (dtype == SPHERICART_CUDA_F32 ? sph_expand_launch_f32 : sph_expand_launch_f64)(
            st->smem_optin, xyz, radial, seg_ptr, n_seg, l_max, n_rad, coeff, static_cast<cudaStream_t>(stream));
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "expand launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) {
            launched("expand");
            return 0;
        }
    }
    // any l_max with n_rad <= 16: the run-time-l_max DMMA kernel, degrees in bands
    if (g_opt.force_kernel != FORCE_GENERIC) {
        const int r = (dtype == SPHERICART_CUDA_F32 ? sph_expand_rt_launch_f32 : sph_expand_rt_launch_f64)(
            st->smem_optin, xyz, radial, seg_ptr, n_seg, l_max, n_rad, coeff, static_cast<cudaStream_t>(stream));
        if (r < 0) return fail(SPHERICART_CUDA_ECUDA, "expand launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (r == 0) {
            launched("expand_rt");
            return 0;
        }
    }
    // every other (l_max, n_rad): run-time sizes, one CTA per (segment, slice of the radial rows)
    const int L = (l_max + 1) * (l_max + 1);
    if (n_seg > 0x7fffffff) return fail(SPHERICART_CUDA_EINVAL, "n_seg = %lld is too large", (long long)n_seg);
    ExpandGenParams gp{};
    gp.xyz = xyz;
    gp.radial = radial;
    gp.seg_ptr = seg_ptr;
    gp.coeff = coeff;
    gp.n_rad = n_rad;
    gp.l_max = l_max;
    gp.pts_tile = 32;
    while (gp.pts_tile > 1 && (size_t)gp.pts_tile * L * 8 > (size_t)48 * 1024) gp.pts_tile >>= 1;   // a few CTAs per SM
    gp.rows_per_slice = EXG_THREADS * EXG_ACC / L;
    if (gp.rows_per_slice > n_rad) gp.rows_per_slice = n_rad;
    const int slices = (n_rad + gp.rows_per_slice - 1) / gp.rows_per_slice;
    if (slices > 65535) return fail(SPHERICART_CUDA_EINVAL, "n_rad = %d is too large", n_rad);
    const size_t smem = (size_t)gp.pts_tile * L * 8;
    const dim3 grid((unsigned)n_seg, (unsigned)slices);
    if (dtype == SPHERICART_CUDA_F32) {
        auto k = sph_expand_generic_kernel<float, double>;
        rc = allow_smem((const void*)k, (int)smem);
        if (rc) return rc;
        k<<<grid, EXG_THREADS, smem, static_cast<cudaStream_t>(stream)>>>(gp, st->d_tables);
    } else {
        auto k = sph_expand_generic_kernel<double, dd>;
        rc = allow_smem((const void*)k, (int)smem);
        if (rc) return rc;
        k<<<grid, EXG_THREADS, smem, static_cast<cudaStream_t>(stream)>>>(gp, st->d_tables);
    }
    CUDA_TRY(cudaGetLastError());
    launched("expand_generic");
    return 0;
}

// Every exit of the chunk loops below passes through here: both streams are drained before the
// call returns, so no copy is still writing into (or reading from) the caller's buffers -- also
// when a later chunk failed.
static int host_finish(int rc) {
    cudaError_t e0 = cudaStreamSynchronize(g_ws.stream[0]);
    cudaError_t e1 = cudaStreamSynchronize(g_ws.stream[1]);
    if (rc) return rc;
    if (e0 != cudaSuccess || e1 != cudaSuccess)
        return fail(SPHERICART_CUDA_ECUDA, "cudaStreamSynchronize failed: %s",
                    cudaGetErrorString(e0 != cudaSuccess ? e0 : e1));
    return 0;
}
#define HOST_TRY(call)                                                                                    \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess)                                                                            \
            return host_finish(fail(SPHERICART_CUDA_ECUDA, "%s failed: %s", #call, cudaGetErrorString(e_))); \
    } while (0)

int sphericart_cuda_compute_host(const void* xyz, int64_t n, int l_max, int normalized, int dtype, void* sph,
                                 void* dsph, void* ddsph) {
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (ddsph && !dsph) return fail(SPHERICART_CUDA_EINVAL, "ddsph given without dsph");
    if (n == 0) return 0;
    if (!xyz || !sph) return fail(SPHERICART_CUDA_EINVAL, "xyz and sph must not be NULL when n > 0");
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    rc = ws_streams();
    if (rc) return rc;
    const size_t es = dtype == SPHERICART_CUDA_F32 ? 4 : 8;
    const size_t L = (size_t)(l_max + 1) * (l_max + 1);
    const size_t bpp = es * L * (1 + (dsph ? 3 : 0) + (ddsph ? 9 : 0));
    const int64_t chunk = chunk_points(n, bpp, (size_t)g_opt.host_chunk_bytes);
    int slot = 0;
    for (int64_t p0 = 0; p0 < n; p0 += chunk, slot ^= 1) {
        const int64_t np = (n - p0 < chunk) ? n - p0 : chunk;
        cudaStream_t s = g_ws.stream[slot];
        if ((rc = ws_reserve(slot, 0, (size_t)np * 3 * es))) return host_finish(rc);
        if ((rc = ws_reserve(slot, 1, (size_t)np * L * es))) return host_finish(rc);
        if (dsph && (rc = ws_reserve(slot, 2, (size_t)np * 3 * L * es))) return host_finish(rc);
        if (ddsph && (rc = ws_reserve(slot, 3, (size_t)np * 9 * L * es))) return host_finish(rc);
        void** b = g_ws.buf[slot];
        HOST_TRY(cudaMemcpyAsync(b[0], (const char*)xyz + (size_t)p0 * 3 * es, (size_t)np * 3 * es,
                                 cudaMemcpyHostToDevice, s));
        rc = compute_device(b[0], np, l_max, normalized, dtype, b[1], dsph ? b[2] : nullptr,
                            ddsph ? b[3] : nullptr, s);
        if (rc) return host_finish(rc);
        HOST_TRY(cudaMemcpyAsync((char*)sph + (size_t)p0 * L * es, b[1], (size_t)np * L * es,
                                 cudaMemcpyDeviceToHost, s));
        if (dsph)
            HOST_TRY(cudaMemcpyAsync((char*)dsph + (size_t)p0 * 3 * L * es, b[2], (size_t)np * 3 * L * es,
                                     cudaMemcpyDeviceToHost, s));
        if (ddsph)
            HOST_TRY(cudaMemcpyAsync((char*)ddsph + (size_t)p0 * 9 * L * es, b[3], (size_t)np * 9 * L * es,
                                     cudaMemcpyDeviceToHost, s));
    }
    return host_finish(0);
}

int sphericart_cuda_vjp_host(const void* xyz, const void* dsph, const void* grad_sph, void* grad_xyz, int64_t n,
                             int l_max, int dtype) {
    (void)xyz;
    int rc = check_common(n, l_max, dtype);
    if (rc) return rc;
    if (n == 0) return 0;
    if (!dsph || !grad_sph || !grad_xyz)
        return fail(SPHERICART_CUDA_EINVAL, "dsph, grad_sph and grad_xyz must not be NULL when n > 0");
    std::lock_guard<std::mutex> lock(g_ws_mutex);
    rc = ws_streams();
    if (rc) return rc;
    const size_t es = dtype == SPHERICART_CUDA_F32 ? 4 : 8;
    const size_t L = (size_t)(l_max + 1) * (l_max + 1);
    const int64_t chunk = chunk_points(n, 4 * L * es, (size_t)g_opt.host_chunk_bytes);
    int slot = 0;
    for (int64_t p0 = 0; p0 < n; p0 += chunk, slot ^= 1) {
        const int64_t np = (n - p0 < chunk) ? n - p0 : chunk;
        cudaStream_t s = g_ws.stream[slot];
        if ((rc = ws_reserve(slot, 2, (size_t)np * 3 * L * es))) return host_finish(rc);
        if ((rc = ws_reserve(slot, 1, (size_t)np * L * es))) return host_finish(rc);
        if ((rc = ws_reserve(slot, 4, (size_t)np * 3 * es))) return host_finish(rc);
        void** b = g_ws.buf[slot];
        HOST_TRY(cudaMemcpyAsync(b[2], (const char*)dsph + (size_t)p0 * 3 * L * es, (size_t)np * 3 * L * es,
                                 cudaMemcpyHostToDevice, s));
        HOST_TRY(cudaMemcpyAsync(b[1], (const char*)grad_sph + (size_t)p0 * L * es, (size_t)np * L * es,
                                 cudaMemcpyHostToDevice, s));
        rc = vjp_device(b[2], b[1], b[4], np, l_max, dtype, s);
        if (rc) return host_finish(rc);
        HOST_TRY(cudaMemcpyAsync((char*)grad_xyz + (size_t)p0 * 3 * es, b[4], (size_t)np * 3 * es,
                                 cudaMemcpyDeviceToHost, s));
    }
    return host_finish(0);
}

int sphericart_cuda_set_option(const char* name, const char* value) {
    if (!name || !value) return fail(SPHERICART_CUDA_EINVAL, "set_option: NULL name or value");
    struct IntOpt { const char* name; int* slot; };
    const IntOpt ints[] = {{"tpg_lp", &g_opt.tpg_lp}, {"w_nbuf", &g_opt.w_nbuf}, {"w_warps", &g_opt.w_warps},
                           {"w_ppw", &g_opt.w_ppw}, {"wc_min_l", &g_opt.wc_min_l}, {"vjp_warps", &g_opt.vjp_warps},
                           {"tpb_tiles", &g_opt.tpb_tiles}, {"tpb_split", &g_opt.tpb_split}, {"pdl", &g_opt.pdl},
                           {"tq_points", &g_opt.tq_points}, {"tq_warps", &g_opt.tq_warps}, {"tq_batch", &g_opt.tq_batch}, {"tq_images", &g_opt.tq_images}, {"tq_cs_warps", &g_opt.tq_cs_warps}, {"tq_direct", &g_opt.tq_direct}};
    if (!strcmp(name, "force_kernel")) {
        struct { const char* v; int code; } const kinds[] = {
            {"", FORCE_NONE}, {"auto", FORCE_NONE}, {"tpb", FORCE_TPB}, {"tpg", FORCE_TPG}, {"w", FORCE_W},
            {"w1", FORCE_W1}, {"wc", FORCE_WC}, {"tq", FORCE_TQ}, {"tv", FORCE_TV}, {"generic", FORCE_GENERIC}};
        for (const auto& k : kinds)
            if (!strcmp(value, k.v)) {
                g_opt.force_kernel = k.code;
                return 0;
            }
        return fail(SPHERICART_CUDA_EINVAL, "set_option: unknown kernel family '%s'", value);
    }
    if (!strcmp(name, "host_chunk_bytes")) {
        const long long v = atoll(value);
        if (v < 4096) return fail(SPHERICART_CUDA_EINVAL, "set_option: host_chunk_bytes = %s is below 4096", value);
        g_opt.host_chunk_bytes = v;
        return 0;
    }
    for (const auto& o : ints)
        if (!strcmp(name, o.name)) {
            *o.slot = atoi(value);
            return 0;
        }
    return fail(SPHERICART_CUDA_EINVAL, "set_option: unknown option '%s'", name);
}

int sphericart_cuda_vjp_noalloc(const void* dsph, const void* grad_sph, void* grad_xyz, int64_t n, int l_max,
                                int dtype, void* stream) {
    return vjp_noalloc_device(dsph, grad_sph, grad_xyz, n, l_max, dtype, static_cast<cudaStream_t>(stream));
}

const char* sphericart_cuda_last_kernel(void) { return g_last_kernel; }

const char* sphericart_cuda_last_error(void) { return g_err; }

int64_t sphericart_cuda_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

}  // extern "C"
