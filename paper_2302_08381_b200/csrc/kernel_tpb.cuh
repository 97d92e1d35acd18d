// "tpb" forward kernel: TWO threads per point (one per branch of Eq. 5), l_max a compile-time
// constant, 16 points per warp.  Values, or values + gradients.
//
// Why (profiles/r1_*): the path is bound by the HBM write of the row-major
// outputs, and a tile of consecutive points owns one contiguous byte range of sph and one of dsph.
// The thread-per-point kernel (kernel_tp.cuh) stages a 32-point tile per warp; at 1296 B per point
// (C2) that is 41 KB per warp, so only 5 warps fit in an SM's shared memory and the SM idles on
// instruction latency (ncu: 6 % occupancy, 27 % issue-active).  Here
//   * lane = p + 16 b: point p of a 16-point tile, branch b (0: the m >= 0 / cos outputs,
//     1: the m < 0 / sin outputs).  Both lanes of a point run the same instruction stream on the
//     same Legendre column and differ only in the azimuthal factor (c_m | s_m) they multiply by,
//     so there is no divergence, and a warp's image is half as large: twice the warps per SM;
//   * l_max is a template parameter: the (l,m) triangle is fully unrolled, every table entry is a
//     constant-bank operand, every shared-memory offset an immediate, and column m+1 (needed by
//     Eq. 10 for d/dx, d/dy) is computed once and reused as the next column;
//   * the image is laid out exactly like global memory and leaves as 1-D TMA bulk stores.
// For normalised output the chain rule is folded into the assembly:
//     dY/dx = [(q1 - l Q) x A + Q A_x] / r,  dY/dz = (qz - l Q z) A / r,
// with q1 = F Q_{l-1}^{m+1}, qz = F (l+m) Q_{l-1}^m, A = c_m | s_m (Eq. 10 + Euler, sph_core.cuh).
#pragma once
#include <type_traits>

#include "ptx.cuh"
#include "sph_core.cuh"

namespace sphb200 {

// compile-time loop: f(std::integral_constant<int, I>{}) for I in [BEGIN, END)
template <int BEGIN, int END, typename F> __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (BEGIN < END) {
        f(std::integral_constant<int, BEGIN>{});
        static_for<BEGIN + 1, END>(f);
    }
}

// every translation unit that instantiates these kernels carries its own copy of the tables
static __constant__ SphTables c_tables_tpb;

struct TpbParams {
    const void* xyz;
    void* sph;
    void* dsph;
    int64_t n;
};

constexpr int TPB_PTS = 16;            // points per warp tile
constexpr int TPB_SMEM_BUDGET = 226 * 1024;

// launch shape fixed by (element size, DERIV, LMAX)
template <int ESIZE, int DERIV, int LMAX> struct TpbShape {
    static constexpr int L = (LMAX + 1) * (LMAX + 1);
    static constexpr int tile_bytes = TPB_PTS * L * ESIZE * (DERIV ? 4 : 1);
    static constexpr int fit = TPB_SMEM_BUDGET / tile_bytes;
    static constexpr int nbuf = (fit >= 32) ? 2 : 1;                       // two images if 16 warps still fit
    static constexpr int warps = (fit / nbuf) >= 16 ? 16 : (fit / nbuf);   // 0 => does not fit
    static constexpr int smem = warps * nbuf * tile_bytes;
};

template <typename T, typename R, int DERIV, bool NORM, int LMAX>
__global__ void __launch_bounds__(TpbShape<sizeof(T), DERIV, LMAX>::warps * 32, 1)
    sph_tpb_kernel(const TpbParams prm) {
    using RT = rec<R>;
    using Shape = TpbShape<sizeof(T), DERIV, LMAX>;
    constexpr int L = Shape::L;
    constexpr int WARPS = Shape::warps;
    constexpr int NBUF = Shape::nbuf;
    constexpr uint32_t S_BYTES = TPB_PTS * L * sizeof(T);
    const SphTables& TB = c_tables_tpb;
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int pl = lane & (TPB_PTS - 1);   // point inside the tile
    const bool sinb = lane >= TPB_PTS;     // branch
    const int64_t n = prm.n;
    const int64_t n_tiles = (n + TPB_PTS - 1) / TPB_PTS;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    T* __restrict__ dsph = static_cast<T*>(prm.dsph);
    unsigned char* my = smem + (size_t)warp * NBUF * Shape::tile_bytes;
    const uint64_t policy = policy_evict_first();

    const int64_t stride = (int64_t)gridDim.x * WARPS;
    int buf = 0;
    for (int64_t tile = (int64_t)warp * gridDim.x + blockIdx.x; tile < n_tiles; tile += stride) {
        const int64_t p = tile * TPB_PTS + pl;
        double x = 0.0, y = 0.0, z = 1.0;  // lanes past the end compute a harmless point
        if (p < n) {
            x = static_cast<double>(__ldg(xyz + 3 * p + 0));
            y = static_cast<double>(__ldg(xyz + 3 * p + 1));
            z = static_cast<double>(__ldg(xyz + 3 * p + 2));
        }
        R X, Y, Z, r2;
        double rinv = 1.0;
        if (NORM) {
            RT::normalize(x, y, z, X, Y, Z, rinv);
            r2 = RT::make(1.0, 0.0);
        } else {
            X = RT::make(x, 0.0);
            Y = RT::make(y, 0.0);
            Z = RT::make(z, 0.0);
            r2 = RT::r2_of(X, Y, Z);
        }
        const double xd = to_double(X), yd = to_double(Y), zd = to_double(Z);

        // the image we are about to overwrite must have been read out by its bulk store
        if (lane == 0) bulk_wait_read<NBUF - 1>();
        __syncwarp();
        T* S = reinterpret_cast<T*>(my + (size_t)buf * Shape::tile_bytes) + pl * L;
        T* G = reinterpret_cast<T*>(my + (size_t)buf * Shape::tile_bytes + S_BYTES) + pl * 3 * L;

        double Qc[LMAX + 1];   // column m:   Qc[l] = Qt_l^m     (0 for l < m)
        double Qn[LMAX + 1];   // column m+1: Qn[l] = Qt_l^{m+1} (0 for l < m+1)
        // column M of the folded Eq. 7 into dst[M..LMAX] (static_for: every index is a constant, so
        // the arrays live in registers)
        auto column = [&](auto Mc, double* dst) {
            constexpr int M = decltype(Mc)::value;
            R q = RT::make(TB.D_hi[M], TB.D_lo[M]), qp = RT::make(0.0, 0.0);
            static_for<M, LMAX + 1>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                dst[l] = to_double(q);
                if constexpr (l < LMAX) {
                    constexpr int t1 = SPH_TRI(l + 1, M);
                    const R a = RT::make(TB.A_hi[t1], TB.A_lo[t1]);
                    R qn;
                    if constexpr (l == M) {
                        qn = a * (Z * q);
                    } else {
                        const R w = NORM ? qp : r2 * qp;
                        qn = a * (Z * q) - RT::make(TB.B_hi[t1], TB.B_lo[t1]) * w;
                    }
                    qp = q;
                    q = qn;
                }
            });
        };
        column(std::integral_constant<int, 0>{}, Qc);
        R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
        double c1 = 0.0, s1 = 0.0;  // c_{m-1}, s_{m-1}
        static_for<0, LMAX + 1>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            // column m+1, computed once: Eq. 10 needs Qt_{l-1}^{m+1} now, and it is the next column
            if constexpr (m < LMAX) column(std::integral_constant<int, m + 1>{}, Qn);
            // azimuthal factor of this lane's branch and its x/y derivatives (Eq. 9, Eq. 10)
            const double cd = to_double(c), sd = to_double(s);
            const double dm = (double)m;
            const double A = sinb ? sd : (m == 0 ? SPH_INV_SQRT2 : cd);
            double Ax = dm * (sinb ? s1 : c1);
            double Ay = dm * (sinb ? c1 : -s1);
            double xA = xd * A, yA = yd * A, Az = A;
            if (NORM && DERIV >= 1) {
                xA *= rinv;
                yA *= rinv;
                Az *= rinv;
                Ax *= rinv;
                Ay *= rinv;
            }
            const bool emit = (m > 0) || !sinb;   // the sin branch has no m = 0 output
            static_for<m, LMAX + 1>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                constexpr int kc = l * (l + 1) + m, ks = l * (l + 1) - m;
                const int k = sinb ? ks : kc;
                const double Q = Qc[l];
                if (emit) S[k] = static_cast<T>(Q * A);
                if constexpr (DERIV >= 1) {
                    constexpr int t = SPH_TRI(l, m);
                    double q1 = 0.0, qz = 0.0;
                    if constexpr (l >= m + 2) q1 = TB.G1[t] * Qn[l - 1];   // F_l^m Q_{l-1}^{m+1}
                    if constexpr (l >= m + 1) qz = TB.Gz[t] * Qc[l - 1];   // F_l^m (l+m) Q_{l-1}^m
                    double gx, gy, gz;
                    if (NORM) {
                        const double lQ = (double)l * Q;
                        const double t1 = q1 - lQ;
                        const double tz = SPH_FMA(-lQ, zd, qz);
                        gx = SPH_FMA(t1, xA, Q * Ax);
                        gy = SPH_FMA(t1, yA, Q * Ay);
                        gz = tz * Az;
                    } else {
                        gx = SPH_FMA(q1, xA, Q * Ax);
                        gy = SPH_FMA(q1, yA, Q * Ay);
                        gz = qz * Az;
                    }
                    if (emit) {
                        G[k] = static_cast<T>(gx);
                        G[L + k] = static_cast<T>(gy);
                        G[2 * L + k] = static_cast<T>(gz);
                    }
                }
            });
            // next column, next power of (x + i y): Eq. 9
            if constexpr (m < LMAX) {
                static_for<m + 1, LMAX + 1>([&](auto lc) { Qc[decltype(lc)::value] = Qn[decltype(lc)::value]; });
                c1 = cd;
                s1 = sd;
                const R cn = X * c - Y * s;
                const R sn = X * s + Y * c;
                c = cn;
                s = sn;
            }
        });

        fence_proxy_async_smem();
        __syncwarp();
        const int64_t p0 = tile * TPB_PTS;
        T* S0 = reinterpret_cast<T*>(my + (size_t)buf * Shape::tile_bytes);
        T* G0 = reinterpret_cast<T*>(my + (size_t)buf * Shape::tile_bytes + S_BYTES);
        if (n - p0 >= TPB_PTS) {
            if (lane == 0) {
                bulk_store_hint(sph + p0 * L, S0, S_BYTES, policy);
                if (DERIV >= 1) bulk_store_hint(dsph + p0 * 3 * L, G0, 3u * S_BYTES, policy);
                bulk_commit();
            }
        } else {  // ragged last tile: byte count need not be a multiple of 16 -> plain stores
            const int np = (int)(n - p0);
            for (int i = lane; i < np * L; i += 32) st_cs(sph + p0 * L + i, S0[i]);
            if (DERIV >= 1)
                for (int i = lane; i < np * 3 * L; i += 32) st_cs(dsph + p0 * 3 * L + i, G0[i]);
            __syncwarp();
        }
        buf = (buf + 1 == NBUF) ? 0 : buf + 1;
    }
    // shared memory must outlive the bulk stores that read it
    if (lane == 0) bulk_wait_all<0>();
}

}  // namespace sphb200
