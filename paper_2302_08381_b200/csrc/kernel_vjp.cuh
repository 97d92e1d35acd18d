// Backward kernel: grad_xyz[i,a] = sum_k dsph[i,a,k] * grad_sph[i,k].
//
// A streaming READ of 4L elements per point against 3 written: bound by HBM read bandwidth.
// Mirror image of the forward kernel: a warp owns tiles of 32 consecutive points, whose dsph and
// grad_sph rows are two contiguous byte ranges; lane 0 pulls them into shared memory with 1-D TMA
// bulk loads (full lines, completion counted on an mbarrier), double-buffered so the next tile is
// in flight while the 32 lanes each contract their own point's rows (row pitch L words: conflict-
// free for odd L).  Products of two f32 are exact in f64 and the sums are accumulated in f64, so
// the result is the correctly rounded contraction up to ~L eps64.
#pragma once
#include "ptx.cuh"

namespace sphb200 {

struct VjpParams {
    const void* dsph;
    const void* grad_sph;
    void* grad_xyz;
    int64_t n;
    int L;
    int warps_per_cta;
    uint32_t tile_bytes;  // 4 * 32 * L * sizeof(T), multiple of 128
};

constexpr int VJP_MAX_THREADS = 512;
constexpr int VJP_NBUF = 2;

template <typename T>
__global__ void __launch_bounds__(VJP_MAX_THREADS, 1) sph_vjp_kernel(const VjpParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int L = prm.L;
    const int64_t n = prm.n;
    const int64_t n_tiles = (n + 31) >> 5;
    const T* __restrict__ dsph = static_cast<const T*>(prm.dsph);
    const T* __restrict__ gsph = static_cast<const T*>(prm.grad_sph);
    T* __restrict__ gxyz = static_cast<T*>(prm.grad_xyz);

    // [warps][NBUF] images, then [warps][NBUF] mbarriers
    unsigned char* my = smem + (size_t)warp * VJP_NBUF * prm.tile_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)prm.warps_per_cta * VJP_NBUF * prm.tile_bytes) +
                     warp * VJP_NBUF;
    if (lane == 0) {
        for (int b = 0; b < VJP_NBUF; ++b) mbar_init(&bars[b], 1);
        fence_mbar_init();
    }
    __syncwarp();

    const uint32_t g_bytes = 32u * L * sizeof(T);  // grad_sph part of an image; dsph part is 3x
    const int64_t stride = (int64_t)gridDim.x * prm.warps_per_cta;
    const int64_t first = (int64_t)warp * gridDim.x + blockIdx.x;

    auto issue = [&](int64_t tile, int b) {  // lane 0 only; full tiles only
        unsigned char* img = my + (size_t)b * prm.tile_bytes;
        mbar_arrive_expect_tx(&bars[b], 4u * g_bytes);
        bulk_load(img, gsph + tile * 32 * L, g_bytes, &bars[b]);
        bulk_load(img + g_bytes, dsph + tile * 32 * 3 * L, 3u * g_bytes, &bars[b]);
    };
    auto is_full = [&](int64_t tile) { return (tile + 1) * 32 <= n; };

    if (lane == 0 && first < n_tiles && is_full(first)) issue(first, 0);
    uint32_t phase_bits = 0;  // bit b = parity to wait for on bars[b]
    int buf = 0;
    for (int64_t tile = first; tile < n_tiles; tile += stride) {
        const int64_t next = tile + stride;
        if (lane == 0 && next < n_tiles && is_full(next)) issue(next, buf ^ 1);
        const int64_t p = tile * 32 + lane;
        double ax = 0.0, ay = 0.0, az = 0.0;
        if (is_full(tile)) {
            mbar_wait(&bars[buf], (phase_bits >> buf) & 1u);
            phase_bits ^= 1u << buf;
            const T* img = reinterpret_cast<const T*>(my + (size_t)buf * prm.tile_bytes);
            const T* g = img + lane * L;
            const T* d = img + 32 * L + lane * 3 * L;
#pragma unroll 4
            for (int k = 0; k < L; ++k) {
                const double w = static_cast<double>(g[k]);
                ax = fma(static_cast<double>(d[k]), w, ax);
                ay = fma(static_cast<double>(d[L + k]), w, ay);
                az = fma(static_cast<double>(d[2 * L + k]), w, az);
            }
        } else if (p < n) {  // ragged last tile: straight from global memory
            const T* g = gsph + p * L;
            const T* d = dsph + p * 3 * L;
            for (int k = 0; k < L; ++k) {
                const double w = static_cast<double>(g[k]);
                ax = fma(static_cast<double>(d[k]), w, ax);
                ay = fma(static_cast<double>(d[L + k]), w, ay);
                az = fma(static_cast<double>(d[2 * L + k]), w, az);
            }
        }
        if (p < n) {
            gxyz[3 * p + 0] = static_cast<T>(ax);
            gxyz[3 * p + 1] = static_cast<T>(ay);
            gxyz[3 * p + 2] = static_cast<T>(az);
        }
        __syncwarp();  // every lane is done with this image before it is refilled
        buf ^= 1;
    }
}

}  // namespace sphb200
