// "tp" forward kernel: one THREAD per point, one WARP per tile of 32 consecutive points.
//
// Why this shape on B200: the path is bound by the HBM write of the
// row-major outputs (784..1296 B per point against ~1.5..2 kflop).  A tile of 32
// consecutive points owns ONE contiguous byte range of sph ([32,L]) and one of dsph ([32,3,L]),
// so each warp
//   1. runs the recurrences of its 32 points in registers (eval_point_columns, O(1) state),
//   2. writes every output element into a shared-memory image laid out exactly like global memory
//      (thread p writes word p*L+k: conflict-free because L = (l_max+1)^2 is odd for even l_max),
//   3. hands the image to the TMA engine as one or two 1-D bulk stores (cp.async.bulk, full
//      128-byte lines, no LSU store instructions) and goes on with its next tile.
// Warps are independent (no CTA-wide barrier); the grid is one persistent CTA per SM with as many
// warps as shared memory allows, tiles dealt round-robin across SMs.
// The paper's A100 kernel also staged outputs in shared memory, but with 1 thread in 8
// computing and the others copying; here the copy costs no thread at all.
#pragma once
#include "ptx.cuh"
#include "sph_core.cuh"

namespace sphb200 {

// one translation unit (api.cu) includes this header, so the constant bank is defined here
__constant__ SphTables c_tables;

template <typename T> struct SmemEmit {
    T* S;
    T* G;
    int L;
    __device__ __forceinline__ void val(int k, double v) { S[k] = static_cast<T>(v); }
    __device__ __forceinline__ void grad(int a, int k, double v) { G[a * L + k] = static_cast<T>(v); }
};

struct TpParams {
    const void* xyz;
    void* sph;
    void* dsph;
    int64_t n;
    int l_max;
    int warps_per_cta;
    int nbuf;              // shared-memory images per warp (1 or 2)
    uint32_t tile_bytes;   // bytes of one image (sph part + dsph part), multiple of 128
};

constexpr int TP_MAX_THREADS = 512;

template <typename T, typename R, int DERIV, bool NORM>
__global__ void __launch_bounds__(TP_MAX_THREADS, 1) sph_tp_kernel(const TpParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const int64_t n = prm.n;
    const int64_t n_tiles = (n + 31) >> 5;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    T* __restrict__ dsph = static_cast<T*>(prm.dsph);

    const uint32_t s_bytes = 32u * L * sizeof(T);
    unsigned char* my = smem + (size_t)warp * prm.nbuf * prm.tile_bytes;
    const uint64_t policy = policy_evict_first();

    // tiles are dealt so that consecutive tiles land on different SMs: slot = warp*gridDim + cta
    const int64_t stride = (int64_t)gridDim.x * prm.warps_per_cta;
    int buf = 0;
    for (int64_t tile = (int64_t)warp * gridDim.x + blockIdx.x; tile < n_tiles; tile += stride) {
        // the image we are about to overwrite must have been read out by its bulk store
        if (lane == 0) {
            if (prm.nbuf == 1) bulk_wait_read<0>();
            else bulk_wait_read<1>();
        }
        __syncwarp();
        T* S = reinterpret_cast<T*>(my + (size_t)buf * prm.tile_bytes);
        T* G = reinterpret_cast<T*>(my + (size_t)buf * prm.tile_bytes + s_bytes);

        const int64_t p = tile * 32 + lane;
        double x = 0.0, y = 0.0, z = 1.0;  // lanes past the end compute a harmless point
        if (p < n) {
            x = static_cast<double>(xyz[3 * p + 0]);
            y = static_cast<double>(xyz[3 * p + 1]);
            z = static_cast<double>(xyz[3 * p + 2]);
        }
        SmemEmit<T> emit{S + lane * L, G + lane * 3 * L, L};
        eval_point_columns<R, DERIV, NORM>(x, y, z, l_max, c_tables, emit);

        fence_proxy_async_smem();
        __syncwarp();
        const int64_t p0 = tile * 32;
        const int np = (n - p0 >= 32) ? 32 : (int)(n - p0);
        if (np == 32) {
            if (lane == 0) {
                bulk_store_hint(sph + p0 * L, S, s_bytes, policy);
                if (DERIV >= 1) bulk_store_hint(dsph + p0 * 3 * L, G, 3u * s_bytes, policy);
                bulk_commit();
            }
        } else {  // ragged last tile: byte count need not be a multiple of 16 -> plain stores
            for (int i = lane; i < np * L; i += 32) st_cs(sph + p0 * L + i, S[i]);
            if (DERIV >= 1)
                for (int i = lane; i < np * 3 * L; i += 32) st_cs(dsph + p0 * 3 * L + i, G[i]);
            __syncwarp();
        }
        buf = (buf + 1 == prm.nbuf) ? 0 : buf + 1;
    }
    // shared memory must outlive the bulk stores that read it
    if (lane == 0) bulk_wait_all<0>();
}

}  // namespace sphb200
