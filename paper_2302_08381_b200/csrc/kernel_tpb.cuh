// "tpb" forward kernel: TWO threads per point (one per branch of Eq. 5), l_max a compile-time
// constant, 16 points per tile.  Values, or values + gradients.
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
    void* ddsph;
    int64_t n;
    int tiles_per_cta;   // consecutive tiles one CTA works through
    int pdl;             // launched as a programmatic dependent launch (tpb_inst.cu)
};

constexpr int TPB_PTS = 16;                 // points per tile
constexpr int TPB_SMEM_PER_SM = 228 * 1024; // B200: 228 KB per SM, 1 KB of it reserved per resident CTA

// Launch shape fixed by (element size, DERIV, LMAX, SPLIT).
//
// The grid is NOT persistent: a CTA owns `tiles_per_cta` consecutive tiles and there are many more
// CTAs than fit on the machine, so the hardware block scheduler hands tiles out as SMs free up.
// Measured on B200 with a store-only probe: under a static, equal split of a large output the SMs
// finish at 247k / 283k / 346k cycles depending on where they sit (6.2 TB/s overall); handing the
// same tiles out dynamically reaches 7.3-7.4 TB/s.
//
// SPLIT = warps that share one tile.  SPLIT == 2: warp 0 takes the columns m < cut, warp 1 the
// columns m >= cut of the (l,m) triangle (balanced by the number of (l,m) pairs), so a tile's
// latency halves for the same shared-memory footprint; the only duplicated work is column `cut`
// and the first `cut` steps of Eq. 9.
template <int LMAX, int SPLIT> struct TpbCut {
    static constexpr int pairs(int m0, int m1) {   // (l,m) pairs with m0 <= m < m1
        int s = 0;
        for (int m = m0; m < m1; ++m) s += LMAX + 1 - m;
        return s;
    }
    static constexpr int cut() {
        if (SPLIT == 1) return LMAX + 1;
        const int total = pairs(0, LMAX + 1);
        int c = 1;
        while (c < LMAX && 2 * pairs(0, c) < total) ++c;
        // the nearer of c-1 and c to an even split
        const int over = 2 * pairs(0, c) - total, under = total - 2 * pairs(0, c - 1);
        return (c > 1 && under < over) ? c - 1 : c;
    }
};

template <int ESIZE, int DERIV, int LMAX, int SPLIT, bool BB = false> struct TpbShape {
    static constexpr int L = (LMAX + 1) * (LMAX + 1);
    // BB: ONE lane per point does both branches of Eq. 5 (32 points per tile): the Legendre
    // recurrences run once for the two -- for the kernels that are bound by them (double-double)
    static constexpr int pts = BB ? 32 : TPB_PTS;
    // Shared-memory banks: lane p writes word p * (row pitch) + k; the lanes of a branch collide 8- or
    // 16-way when the pitch in 32-bit words is 0 or 16 modulo 32, i.e. for l_max = 3 (mod 4)
    // (measured: f32 l_max = 7 ran at 2.0 TB/s where l_max = 6 and 8 reach 6.7 and 6.9).  Those row
    // lengths get 16 bytes of padding per point (pitch = 4 or 20 mod 32: 2-way), the image is then
    // no longer byte-identical to global memory and leaves as one bulk store per point and array where a
    // point's rows are long enough (`row_bulk`), by 16-byte vector stores otherwise.  Measured, vector ->
    // bulk rows: f32 V+G l_max 7 / 11: 6.2 / 4.4 -> 6.9 / 5.2 TB/s, f32 V l_max 15: 5.7 -> 6.2, f32 V+G+H
    // l_max 3: 5.2 -> 6.0, f64 V+G l_max 7: 5.3 -> 5.9; but f32 V l_max 3 / 7 / 11 (rows of 64-576 bytes):
    // 4.2 / 6.1 / 5.4 -> 3.3 / 5.5 / 5.0, f64 V+G l_max 3: 6.2 -> 5.5, f64 V l_max 11: 4.7 -> 4.5.
    static constexpr int words = L * ESIZE / 4;
    static constexpr bool pad = (words % 32 == 0) || (words % 32 == 16);
    static constexpr int pad_elems = pad ? 16 / ESIZE : 0;
    static constexpr int point_bytes = L * ESIZE * (DERIV == 0 ? 1 : (DERIV == 1 ? 4 : 13));
    static constexpr bool row_bulk = pad && (DERIV == 0 ? (ESIZE == 4 && point_bytes >= 1024) : point_bytes >= 800);
    static constexpr int pitch_s = L + pad_elems;          // elements between the points' rows of sph
    static constexpr int pitch_g = 3 * L + pad_elems;      // ... of dsph
    static constexpr int s_bytes = pts * pitch_s * ESIZE;
    static constexpr int pitch_h = 9 * L + pad_elems;      // ... of ddsph
    static constexpr int g_bytes = DERIV >= 1 ? pts * pitch_g * ESIZE : 0;
    static constexpr int h_bytes = DERIV >= 2 ? pts * pitch_h * ESIZE : 0;
    static constexpr int tile_bytes = s_bytes + g_bytes + h_bytes;
    static constexpr int fit = TPB_SMEM_PER_SM / (tile_bytes + 1024);   // resident CTAs per SM by shared memory
    static constexpr int cap = 16 / SPLIT;                              // ... and by registers (<= 128 each)
    static constexpr int min_ctas = fit < 1 ? 1 : (fit < cap ? fit : cap);
    static constexpr int cut = TpbCut<LMAX, SPLIT>::cut();
};

template <typename T, typename R, int DERIV, bool NORM, int LMAX, int SPLIT, bool BB = false>
__global__ void __launch_bounds__(SPLIT * 32, TpbShape<sizeof(T), DERIV, LMAX, SPLIT, BB>::min_ctas)
    sph_tpb_kernel(const TpbParams prm) {
    using RT = rec<R>;
    using Shape = TpbShape<sizeof(T), DERIV, LMAX, SPLIT, BB>;
    constexpr int PTS = Shape::pts;
    constexpr int L = Shape::L;
    constexpr int CUT = Shape::cut;
    constexpr uint32_t S_BYTES = Shape::s_bytes;
    constexpr int PS = Shape::pitch_s, PG = Shape::pitch_g, PH = Shape::pitch_h;
    constexpr uint32_t G_BYTES = Shape::g_bytes;
    const SphTables& TB = c_tables_tpb;
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int part = threadIdx.x >> 5;     // which share of the columns (warp-uniform)
    const int pl = lane & (PTS - 1);             // point inside the tile
    const bool sinb = BB ? false : lane >= PTS;   // branch (BB: cos here, sin alongside)
    const int64_t n = prm.n;
    const int64_t n_tiles = (n + PTS - 1) / PTS;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    T* __restrict__ dsph = static_cast<T*>(prm.dsph);
    T* __restrict__ ddsph = static_cast<T*>(prm.ddsph);
    const uint64_t policy = policy_evict_first();
    auto cta_sync = [&]() {
        if constexpr (SPLIT == 1) __syncwarp();
        else __syncthreads();
    };

    // programmatic dependent launch (tpb_inst.cu): let the next kernel's CTAs become resident as
    // ours retire, and do not touch memory before the previous kernel in the stream has completed
    if (prm.pdl) {
        grid_launch_dependents();
        grid_dependency_wait();
    }

    const int64_t t_begin = (int64_t)blockIdx.x * prm.tiles_per_cta;
    int64_t t_end = t_begin + prm.tiles_per_cta;
    if (t_end > n_tiles) t_end = n_tiles;

    // lanes past the end compute a harmless point
    auto load_xyz = [&](int64_t tile, T& a, T& b, T& c) {
        const int64_t p = tile * PTS + pl;
        a = T(0), b = T(0), c = T(1);
        if (p < n) {
            a = __ldg(xyz + 3 * p + 0);
            b = __ldg(xyz + 3 * p + 1);
            c = __ldg(xyz + 3 * p + 2);
        }
    };
    T xn, yn, zn;
    if (t_begin < t_end) load_xyz(t_begin, xn, yn, zn);

    for (int64_t tile = t_begin; tile < t_end; ++tile) {
        const double x = static_cast<double>(xn), y = static_cast<double>(yn), z = static_cast<double>(zn);
        if (tile + 1 < t_end) load_xyz(tile + 1, xn, yn, zn);   // in flight while this tile computes
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
        if (tile > t_begin) {
            // (padded images: one thread per point has issued stores; the others wait on nothing)
            if (Shape::row_bulk || threadIdx.x == 0) bulk_wait_read<0>();
            cta_sync();
        }
        T* S = reinterpret_cast<T*>(smem) + pl * PS;
        T* G = reinterpret_cast<T*>(smem + S_BYTES) + pl * PG;
        T* H = reinterpret_cast<T*>(smem + S_BYTES + G_BYTES) + pl * PH;

        double Qc[LMAX + 1];   // column m:   Qc[l] = Qt_l^m     (0 for l < m)
        double Qn[DERIV >= 1 ? LMAX + 1 : 1];   // column m+1: Qn[l] = Qt_l^{m+1} (0 for l < m+1)
        double Qnn[DERIV >= 2 ? LMAX + 1 : 1];   // column m+2 (Hessians: Eq. 10 twice needs Qt_{l-2}^{m+2})
        // column M of the folded Eq. 7 into dst[M..LMAX] (static_for: every index is a constant, so
        // the arrays live in registers)
        auto column = [&](auto Mc, double* dst) {
            constexpr int M = decltype(Mc)::value;
            R q = RT::make(TB.D_hi[M], TB.D_lo[M]), qp = RT::make(0.0, 0.0);
            static_for<M, LMAX + 1>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                dst[l] = pair_value(q);   // (q: unnormalised pair from rec_step_u)
                if constexpr (l < LMAX) {
                    constexpr int t1 = SPH_TRI(l + 1, M);
                    const R a = RT::make(TB.A_hi[t1], TB.A_lo[t1]);
                    R qn;
                    if constexpr (l == M) {
                        qn = a * (Z * q);
                    } else {
                        const R w = NORM ? qp : r2 * qp;
                        qn = rec_step_u(TB.A_hi[t1], TB.A_lo[t1], TB.B_hi[t1], TB.B_lo[t1], Z, q, w);   // (dd.cuh: short dependency chain)
                    }
                    qp = q;
                    q = qn;
                }
            });
        };
        // the columns M0 <= m < M1 of the triangle: values (Eq. 5) and gradients (Eq. 10) of this
        // lane's branch into the image
        auto columns = [&](auto M0c, auto M1c) {
            constexpr int M0 = decltype(M0c)::value, M1 = decltype(M1c)::value;
            R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
            double c1 = 0.0, s1 = 0.0;  // c_{m-1}, s_{m-1}
            double c2 = 0.0, s2 = 0.0;  // c_{m-2}, s_{m-2} (Hessians)
            static_for<0, M0>([&](auto) {   // Eq. 9 up to (x + i y)^M0
                c2 = c1;
                s2 = s1;
                c1 = to_double(c);
                s1 = to_double(s);
                const R cn = X * c - Y * s;
                const R sn = X * s + Y * c;
                c = cn;
                s = sn;
            });
            column(std::integral_constant<int, M0>{}, Qc);
            if constexpr (DERIV >= 2 && M0 < LMAX) column(std::integral_constant<int, M0 + 1>{}, Qn);
            static_for<M0, M1>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                // column m+1, computed once: Eq. 10 needs Qt_{l-1}^{m+1} now, and it is the next column
                // (Hessians: columns m+1 and m+2 are carried, m+2 is the new one)
                // (values only: no second column at all, column m+1 is computed in place afterwards)
                if constexpr (DERIV == 1) {
                    if constexpr (m < LMAX) column(std::integral_constant<int, m + 1>{}, Qn);
                } else if constexpr (DERIV >= 2) {
                    if constexpr (m + 2 <= LMAX) column(std::integral_constant<int, m + 2>{}, Qnn);
                }
                // azimuthal factor of this lane's branch and its x/y derivatives (Eq. 9, Eq. 10)
                const double cd = to_double(c), sd = to_double(s);
                const double dm = (double)m;
                const double sc = (NORM && DERIV == 1) ? rinv : 1.0;   // gradients only: the chain rule's 1/r, folded in
                // one branch of Eq. 5 for every l of this column: A = c_m | s_m | 1/sqrt2, its x/y
                // derivatives, (c,s)_{m-2} for the second derivatives
                auto branch = [&](bool sin_branch, bool emit) {
                    const double A = sin_branch ? sd : (m == 0 ? SPH_INV_SQRT2 : cd);
                    const double Ax = dm * (sin_branch ? s1 : c1) * sc;
                    const double Ay = dm * (sin_branch ? c1 : -s1) * sc;
                    const double xA = xd * A * sc, yA = yd * A * sc, Az = A * sc;
                    double y_prev = 0.0;   // Ytilde_{l-1}^m of this branch (Eq. 11 shortcut below)
                    static_for<m, LMAX + 1>([&](auto lc) {
                        constexpr int l = decltype(lc)::value;
                        constexpr int kc = l * (l + 1) + m, ks = l * (l + 1) - m;
                        const int k = sin_branch ? ks : kc;
                        const double Q = Qc[l];
                        if constexpr (DERIV >= 2) {
                            constexpr int t = SPH_TRI(l, m);
                            double q1 = 0.0, qz = 0.0, q2 = 0.0, qxz = 0.0, qzz = 0.0;
                            if constexpr (l >= m + 2) q1 = TB.G1[t] * Qn[l - 1];     // F_l^m Q_{l-1}^{m+1}
                            if constexpr (l >= m + 1) qz = TB.Gz[t] * Qc[l - 1];     // F_l^m (l+m) Q_{l-1}^m
                            if constexpr (l >= m + 4) q2 = TB.H2[t] * Qnn[l - 2];    // F_l^m Q_{l-2}^{m+2}
                            if constexpr (l >= m + 3) qxz = TB.Hxz[t] * Qn[l - 2];   // F_l^m (l+m) Q_{l-2}^{m+1}
                            if constexpr (l >= m + 2) qzz = TB.Hzz[t] * Qc[l - 2];   // F_l^m (l+m)(l+m-1) Q_{l-2}^m
                            const double dmm = dm * (dm - 1.0);
                            // Eq. 10 twice: cos: A_xx = m(m-1) c_{m-2}, A_xy = -m(m-1) s_{m-2}; sin: s_{m-2}, c_{m-2}
                            const double Axx = dmm * (sin_branch ? s2 : c2);
                            const double Axy = dmm * (sin_branch ? c2 : -s2);
                            double o[10];
                            assemble_scalars<NORM>(l, Q, q1, qz, q2, qxz, qzz, A, Ax, Ay, Axx, Axy, xd, yd, zd, rinv, o);
                            if (emit) {
                                S[k] = static_cast<T>(o[0]);
                                G[k] = static_cast<T>(o[1]);
                                G[L + k] = static_cast<T>(o[2]);
                                G[2 * L + k] = static_cast<T>(o[3]);
                                // o[4..9] = xx xy xz yy yz zz ; rows = xx xy xz yx yy yz zx zy zz
                                H[k] = static_cast<T>(o[4]);
                                H[L + k] = static_cast<T>(o[5]);
                                H[2 * L + k] = static_cast<T>(o[6]);
                                H[3 * L + k] = static_cast<T>(o[5]);
                                H[4 * L + k] = static_cast<T>(o[7]);
                                H[5 * L + k] = static_cast<T>(o[8]);
                                H[6 * L + k] = static_cast<T>(o[6]);
                                H[7 * L + k] = static_cast<T>(o[8]);
                                H[8 * L + k] = static_cast<T>(o[9]);
                            }
                        } else {
                            const double Yl = Q * A;
                            if (emit) S[k] = static_cast<T>(Yl);
                            if constexpr (DERIV >= 1) {
                                constexpr int t = SPH_TRI(l, m);
                                double q1 = 0.0, qz = 0.0;
                                if constexpr (l >= m + 2) q1 = TB.G1[t] * Qn[l - 1];   // F_l^m Q_{l-1}^{m+1}
                                if constexpr (NORM && l >= m + 1) qz = TB.Gz[t] * Qc[l - 1];   // F_l^m (l+m) Q_{l-1}^m
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
                                    // Eq. 11 (reading E2): d/dz Ytilde_l^m = (F_l^m / F_{l-1}^m)(l+|m|) Ytilde_{l-1}^m,
                                    // the ratio being the table Gz: the value of the previous degree, already
                                    // in a register, times one constant (one multiply less than F (l+m) Q_{l-1}^m A)
                                    gz = TB.Gz[t] * y_prev;
                                }
                                y_prev = Yl;
                                if (emit) {
                                    G[k] = static_cast<T>(gx);
                                    G[L + k] = static_cast<T>(gy);
                                    G[2 * L + k] = static_cast<T>(gz);
                                }
                            }
                        }
                    });
                };
                if constexpr (BB) {
                    branch(false, true);
                    if constexpr (m > 0) branch(true, true);   // the sin branch has no m = 0 output
                } else {
                    branch(sinb, (m > 0) || !sinb);
                }
                // next column, next power of (x + i y): Eq. 9
                if constexpr (m + 1 < M1) {
                    if constexpr (DERIV == 0) column(std::integral_constant<int, m + 1>{}, Qc);
                    else static_for<m + 1, LMAX + 1>([&](auto lc) { Qc[decltype(lc)::value] = Qn[decltype(lc)::value]; });
                    if constexpr (DERIV >= 2)
                        static_for<m + 2, LMAX + 1>([&](auto lc) { Qn[decltype(lc)::value] = Qnn[decltype(lc)::value]; });
                    c2 = c1;
                    s2 = s1;
                    c1 = cd;
                    s1 = sd;
                    const R cn = X * c - Y * s;
                    const R sn = X * s + Y * c;
                    c = cn;
                    s = sn;
                }
            });
        };
        if constexpr (SPLIT == 1) {
            columns(std::integral_constant<int, 0>{}, std::integral_constant<int, LMAX + 1>{});
        } else {
            if (part == 0) columns(std::integral_constant<int, 0>{}, std::integral_constant<int, CUT>{});
            else columns(std::integral_constant<int, CUT>{}, std::integral_constant<int, LMAX + 1>{});
        }

        fence_proxy_async_smem();
        cta_sync();
        const int64_t p0 = tile * PTS;
        T* S0 = reinterpret_cast<T*>(smem);
        T* G0 = reinterpret_cast<T*>(smem + S_BYTES);
        T* H0 = reinterpret_cast<T*>(smem + S_BYTES + G_BYTES);
        if constexpr (Shape::row_bulk) {
            // padded image (rows 16 bytes further apart than in global memory; row lengths are multiples of
            // 64 bytes here), long rows: every point's rows leave as bulk stores of their own, issued by one
            // thread per point
            const int np = (int)((n - p0 < PTS) ? n - p0 : PTS);
            if ((int)threadIdx.x < np) {
                const int r = threadIdx.x;
                bulk_store_hint(sph + (p0 + r) * L, S0 + r * PS, (uint32_t)(L * sizeof(T)), policy);
                if (DERIV >= 1) bulk_store_hint(dsph + (p0 + r) * 3 * L, G0 + r * PG, (uint32_t)(3 * L * sizeof(T)), policy);
                if (DERIV >= 2) bulk_store_hint(ddsph + (p0 + r) * 9 * L, H0 + r * PH, (uint32_t)(9 * L * sizeof(T)), policy);
                bulk_commit();
            }
        } else if constexpr (Shape::pad) {
            // padded image, short rows: 16-byte vectors (row lengths are multiples of 16 bytes here)
            constexpr int VE = 16 / (int)sizeof(T);        // elements per vector
            const int np = (int)((n - p0 < PTS) ? n - p0 : PTS);
            constexpr int VS = L / VE, VG = 3 * L / VE;    // vectors per point
            for (int i = threadIdx.x; i < np * VS; i += SPLIT * 32) {
                const int r = i / VS, v = i - r * VS;
                __stcs(reinterpret_cast<float4*>(sph + (p0 + r) * L) + v, reinterpret_cast<const float4*>(S0 + r * PS)[v]);
            }
            if (DERIV >= 1)
                for (int i = threadIdx.x; i < np * VG; i += SPLIT * 32) {
                    const int r = i / VG, v = i - r * VG;
                    __stcs(reinterpret_cast<float4*>(dsph + (p0 + r) * 3 * L) + v,
                           reinterpret_cast<const float4*>(G0 + r * PG)[v]);
                }
            if (DERIV >= 2) {
                constexpr int VH = 9 * L / VE;
                for (int i = threadIdx.x; i < np * VH; i += SPLIT * 32) {
                    const int r = i / VH, v = i - r * VH;
                    __stcs(reinterpret_cast<float4*>(ddsph + (p0 + r) * 9 * L) + v,
                           reinterpret_cast<const float4*>(H0 + r * PH)[v]);
                }
            }
            cta_sync();
        } else if (n - p0 >= PTS) {
            if (threadIdx.x == 0) {
                bulk_store_hint(sph + p0 * L, S0, S_BYTES, policy);
                if (DERIV >= 1) bulk_store_hint(dsph + p0 * 3 * L, G0, 3u * S_BYTES, policy);
                if (DERIV >= 2) bulk_store_hint(ddsph + p0 * 9 * L, H0, 9u * S_BYTES, policy);
                bulk_commit();
            }
        } else {  // ragged last tile: byte count need not be a multiple of 16 -> plain stores
            const int np = (int)(n - p0);
            for (int i = threadIdx.x; i < np * L; i += SPLIT * 32) st_cs(sph + p0 * L + i, S0[i]);
            if (DERIV >= 1)
                for (int i = threadIdx.x; i < np * 3 * L; i += SPLIT * 32) st_cs(dsph + p0 * 3 * L + i, G0[i]);
            if (DERIV >= 2)
                for (int i = threadIdx.x; i < np * 9 * L; i += SPLIT * 32) st_cs(ddsph + p0 * 9 * L + i, H0[i]);
            cta_sync();
        }
    }
    // shared memory must outlive the bulk stores' reads of it
    if (Shape::row_bulk || threadIdx.x == 0) bulk_wait_read<0>();
}

}  // namespace sphb200
