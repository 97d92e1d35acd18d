// "tpg" forward kernel: SEVERAL lanes per point, any l_max at run time.  Values, or values +
// gradients, for the l_max that have no compile-time-unrolled tpb kernel (kernel_tpb.cuh).
//
// Why: the path is bound by the HBM write of the row-major outputs and wants many small tiles in
// flight (kernel_tpb.cuh).  With gradients at l_max = 16 a 16-point f32 tile is already 74 KB; the
// one-warp-per-point kernels (kernel_w.cuh, kernel_wc.cuh) are built for rows of ~100 KB per point
// and reach ~1 TB/s here.  So a point is given LP = 2, 4 or 8 lanes:
//     lane = p + PTS c,   PTS = 32 / LP points per tile,
//     c = column class: the lane owns the columns m = c, c + C, c + 2C, ... of the (l,m) triangle,
//         C = LP, and writes BOTH branches of Eq. 5 (the m >= 0 / cos and the m < 0 / sin outputs)
//         of its columns: the Legendre recurrences, the bulk of a column's cost, run once for the two
//         (template flag BB; with BB = false a lane does one branch and C = LP / 2 -- measured
//         25-55 % slower: f32 values l_max = 24 2.3 -> 3.2 TB/s with BB).
// A column is run with O(1) state as in eval_point_columns (sph_core.cuh): Qt_l^m by the folded
// Eq. 7 and, for the gradients, column m+1 one row behind it (Eq. 10 needs Qt_{l-1}^{m+1}); the
// powers (x + i y)^m of Eq. 9 advance C at a time.  All lanes run the same loops (trip counts
// differ by < C), the tile's image is laid out exactly like global memory and leaves as 1-D TMA
// bulk stores; non-persistent grid, one tile per warp.
#pragma once
#include <cstdlib>

#include "options.h"
#include "ptx.cuh"
#include "sph_core.cuh"

namespace sphb200 {

struct TpgParams {
    const void* xyz;
    void* sph;
    void* dsph;
    const SphTables* tab;   // global-memory copy of the tables
    int64_t n;
    int l_max;
    int warps_per_cta;
};

// coefficient tables in shared memory (lanes of a warp sit on different (l,m): a constant bank
// would serialise them)
template <typename R> struct TpgTabs;
template <> struct TpgTabs<double> {
    const double *A, *B, *D, *G1, *Gz;
    static constexpr int n_tri = 4, n_col = 1;
    __device__ void carve(double* base, int tsz, int ncol) {
        A = base, B = A + tsz, G1 = B + tsz, Gz = G1 + tsz, D = Gz + tsz;
    }
    __device__ void fill(double* base, const SphTables* t, int tsz, int ncol) {
        for (int i = threadIdx.x; i < tsz; i += blockDim.x) {
            base[i] = t->A_hi[i], base[tsz + i] = t->B_hi[i], base[2 * tsz + i] = t->G1[i], base[3 * tsz + i] = t->Gz[i];
        }
        for (int i = threadIdx.x; i < ncol; i += blockDim.x) base[4 * tsz + i] = t->D_hi[i];
    }
    __device__ double a(int t) const { return A[t]; }
    __device__ double b(int t) const { return B[t]; }
    __device__ double d(int m) const { return D[m]; }
};
template <> struct TpgTabs<dd> {
    const double *Ah, *Al, *Bh, *Bl, *Dh, *Dl, *G1, *Gz;
    static constexpr int n_tri = 6, n_col = 2;
    __device__ void carve(double* base, int tsz, int ncol) {
        Ah = base, Al = Ah + tsz, Bh = Al + tsz, Bl = Bh + tsz, G1 = Bl + tsz, Gz = G1 + tsz, Dh = Gz + tsz, Dl = Dh + ncol;
    }
    __device__ void fill(double* base, const SphTables* t, int tsz, int ncol) {
        for (int i = threadIdx.x; i < tsz; i += blockDim.x) {
            base[i] = t->A_hi[i], base[tsz + i] = t->A_lo[i], base[2 * tsz + i] = t->B_hi[i], base[3 * tsz + i] = t->B_lo[i];
            base[4 * tsz + i] = t->G1[i], base[5 * tsz + i] = t->Gz[i];
        }
        for (int i = threadIdx.x; i < ncol; i += blockDim.x) base[6 * tsz + i] = t->D_hi[i], base[6 * tsz + ncol + i] = t->D_lo[i];
    }
    __device__ dd a(int t) const { return dd{Ah[t], Al[t]}; }
    __device__ dd b(int t) const { return dd{Bh[t], Bl[t]}; }
    __device__ dd d(int m) const { return dd{Dh[m], Dl[m]}; }
};

// bytes of one tile's image; rows whose pitch in 32-bit words would be 0 or 16 modulo 32
// (l_max = 3 mod 4) get 16 bytes of padding per point against 8/16-way bank conflicts, and such an
// image leaves by vector stores instead of TMA (see TpbShape in kernel_tpb.cuh)
__host__ __device__ inline int tpg_pad_elems(int L, int esize) {
    const int words = L * esize / 4;
    return (words % 32 == 0 || words % 32 == 16) ? 16 / esize : 0;
}
__host__ __device__ inline int tpg_tile_bytes(int pts, int L, int esize, int deriv) {
    const int pe = tpg_pad_elems(L, esize);
    return pts * (L + pe) * esize + (deriv ? pts * (3 * L + pe) * esize : 0);
}

__host__ __device__ inline int tpg_tab_bytes(int l_max, bool is_dd) {
    const int tsz = (l_max + 1) * (l_max + 2) / 2, ncol = l_max + 1;
    return (((is_dd ? 6 : 4) * tsz + (is_dd ? 2 : 1) * ncol) * 8 + 15) & ~15;
}

template <typename T, typename R, int DERIV, bool NORM, int LP, bool BB>
__global__ void __launch_bounds__(128, 4) sph_tpg_kernel(const TpgParams prm) {
    using RT = rec<R>;
    constexpr int PTS = 32 / LP;   // points per tile
    constexpr int C = BB ? LP : LP / 2;   // column classes (BB: a lane does BOTH branches of its columns)
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const int tsz = (l_max + 1) * (l_max + 2) / 2;
    const int64_t n = prm.n;

    // ---- coefficient tables -> shared memory (once per CTA) -----------------------------------
    TpgTabs<R> TB;
    TB.fill(reinterpret_cast<double*>(smem), prm.tab, tsz, l_max + 1);
    TB.carve(reinterpret_cast<double*>(smem), tsz, l_max + 1);
    __syncthreads();

    const int64_t tile = (int64_t)blockIdx.x * prm.warps_per_cta + warp;
    const int64_t p0 = tile * PTS;
    if (p0 >= n) return;
    const int pad_e = tpg_pad_elems(L, (int)sizeof(T));
    const int PS = L + pad_e, PG = 3 * L + pad_e;   // elements between the points' rows of sph / dsph
    const uint32_t S_BYTES = (uint32_t)(PTS * PS * sizeof(T));
    unsigned char* img = smem + tpg_tab_bytes(l_max, sizeof(R) == sizeof(dd)) +
                         (size_t)warp * tpg_tile_bytes(PTS, L, (int)sizeof(T), DERIV);
    const int pl = lane % PTS;          // point inside the tile
    const int role = lane / PTS;
    const bool sinb = BB ? false : (role & 1);   // branch (BB: cos here, sin alongside)
    const int cls = BB ? role : (role >> 1);     // column class
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    T* __restrict__ dsph = static_cast<T*>(prm.dsph);
    const int64_t p = p0 + pl;

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

    // powers of (x + i y) (Eq. 9): w^cls and w^(cls-1) to start with, w^C to advance by,
    // w^(C-1) for the class that starts at m = 0 (its "w^(m-1)" exists from the second column on)
    R cm = RT::make(1.0, 0.0), sm = RT::make(0.0, 0.0);     // w^m
    R cm1 = RT::make(0.0, 0.0), sm1 = RT::make(0.0, 0.0);   // w^(m-1)
    R cC = RT::make(1.0, 0.0), sC = RT::make(0.0, 0.0);     // w^C
    R cCm = RT::make(1.0, 0.0), sCm = RT::make(0.0, 0.0);   // w^(C-1)
#pragma unroll
    for (int j = 0; j < C; ++j) {
        if (j == cls) cm = cC, sm = sC;
        if (j + 1 == cls) cm1 = cC, sm1 = sC;
        if (j == C - 1) cCm = cC, sCm = sC;
        const R cn = X * cC - Y * sC;
        const R sn = X * sC + Y * cC;
        cC = cn;
        sC = sn;
    }

    T* S = reinterpret_cast<T*>(img) + pl * PS;
    T* G = reinterpret_cast<T*>(img + S_BYTES) + pl * PG;

    for (int m = cls; m <= l_max; m += C) {
        const double cd = to_double(cm), sd = to_double(sm);
        const double c1 = to_double(cm1), s1 = to_double(sm1);
        const double dm = (double)m;
        const double sc = (NORM && DERIV >= 1) ? rinv : 1.0;   // the chain rule's 1/r, folded into the factors
        // azimuthal factor of a branch and its x/y derivatives (Eq. 9, Eq. 10): {A, xA, yA, Az, Ax, Ay}
        // first = this lane's branch (BB: the cos branch), second = the sin branch (BB only)
        const double A0 = sinb ? sd : (m == 0 ? SPH_INV_SQRT2 : cd);
        const double Ax0 = dm * (sinb ? s1 : c1) * sc, Ay0 = dm * (sinb ? c1 : -s1) * sc;
        const double xA0 = xd * A0 * sc, yA0 = yd * A0 * sc, Az0 = A0 * sc;
        const double A1 = sd;
        const double Ax1 = dm * s1 * sc, Ay1 = dm * c1 * sc;
        const double xA1 = xd * A1 * sc, yA1 = yd * A1 * sc, Az1 = A1 * sc;
        const bool emit0 = (m > 0) || !sinb;   // the sin branch has no m = 0 output
        const bool emit1 = BB && m > 0;
        R q = TB.d(m);                   // Qt_l^m, starting at Qt_m^m
        R qp = RT::make(0.0, 0.0);       // Qt_{l-1}^m
        R pc = RT::make(0.0, 0.0);       // Qt_{l-1}^{m+1}
        R pp = RT::make(0.0, 0.0);       // Qt_{l-2}^{m+1}
        // running indices: t = TRI(l, m) (so TRI(l+1, m) = t + l + 1 and TRI(l, m+1) = t + 1) and
        // the output indices k = l (l + 1) +- m, which advance by 2 (l + 1)
        int t = SPH_TRI(m, m);
        T* Sk0 = S + m * (m + 1) + (sinb ? -m : m);
        T* Gk0 = G + m * (m + 1) + (sinb ? -m : m);
        T* Sk1 = S + m * (m + 1) - m;
        T* Gk1 = G + m * (m + 1) - m;
#pragma unroll 2
        for (int l = m; l <= l_max; ++l) {
            const double Q = to_double(q);
            double q1 = 0.0, qz = 0.0, lQ = 0.0;
            if (DERIV >= 1) {
                q1 = TB.G1[t] * to_double(pc);   // F_l^m Q_{l-1}^{m+1}
                qz = TB.Gz[t] * to_double(qp);   // F_l^m (l+m) Q_{l-1}^m
                if (NORM) {   // (q1 - l Q) and (qz - l Q z): Eq. 10 + Euler, as in kernel_tpb.cuh
                    lQ = (double)l * Q;
                    q1 -= lQ;
                    qz = SPH_FMA(-lQ, zd, qz);
                }
            }
            if (emit0) {
                *Sk0 = static_cast<T>(Q * A0);   // Eq. 5
                if (DERIV >= 1) {
                    Gk0[0] = static_cast<T>(SPH_FMA(q1, xA0, Q * Ax0));
                    Gk0[L] = static_cast<T>(SPH_FMA(q1, yA0, Q * Ay0));
                    Gk0[2 * L] = static_cast<T>(qz * Az0);
                }
            }
            if (emit1) {
                *Sk1 = static_cast<T>(Q * A1);
                if (DERIV >= 1) {
                    Gk1[0] = static_cast<T>(SPH_FMA(q1, xA1, Q * Ax1));
                    Gk1[L] = static_cast<T>(SPH_FMA(q1, yA1, Q * Ay1));
                    Gk1[2 * L] = static_cast<T>(qz * Az1);
                }
            }
            if (l < l_max) {
                const int t1 = t + l + 1;   // TRI(l + 1, m)
                R qn;
                if (l == m) {
                    qn = TB.a(t1) * (Z * q);
                } else {
                    const R w = NORM ? qp : r2 * qp;
                    qn = rec_step2(TB.a(t1), TB.b(t1), Z, q, w);   // (dd.cuh)
                }
                qp = q;
                q = qn;
                if (DERIV >= 1) {  // column m+1 reaches row l
                    R pn;
                    if (l == m) {
                        pn = RT::make(0.0, 0.0);
                    } else if (l == m + 1) {
                        pn = TB.d(m + 1);
                    } else {
                        const R w2 = NORM ? pp : r2 * pp;
                        pn = rec_step2(TB.a(t + 1), TB.b(t + 1), Z, pc, w2);   // TRI(l, m + 1) = t + 1
                    }
                    pp = pc;
                    pc = pn;
                }
            }
            t += l + 1;
            Sk0 += 2 * (l + 1);
            Gk0 += 2 * (l + 1);
            Sk1 += 2 * (l + 1);
            Gk1 += 2 * (l + 1);
        }
        // the next column of this class: w^(m+C), w^(m+C-1)
        if (m == 0) {
            cm1 = cCm, sm1 = sCm;
        } else {
            const R cn1 = cm1 * cC - sm1 * sC;
            const R sn1 = cm1 * sC + sm1 * cC;
            cm1 = cn1, sm1 = sn1;
        }
        const R cn = cm * cC - sm * sC;
        const R sn = cm * sC + sm * cC;
        cm = cn, sm = sn;
    }

    fence_proxy_async_smem();
    __syncwarp();
    T* S0 = reinterpret_cast<T*>(img);
    T* G0 = reinterpret_cast<T*>(img + S_BYTES);
    if (pad_e) {
        // padded image: rows leave as 16-byte vectors (row lengths are multiples of 16 bytes here)
        const int VE = 16 / (int)sizeof(T);
        const int np = (int)((n - p0 < PTS) ? n - p0 : PTS);
        const int VS = L / VE, VG = 3 * L / VE;
        for (int i = lane; i < np * VS; i += 32) {
            const int r = i / VS, v = i - r * VS;
            __stcs(reinterpret_cast<float4*>(sph + (p0 + r) * L) + v, reinterpret_cast<const float4*>(S0 + r * PS)[v]);
        }
        if (DERIV >= 1)
            for (int i = lane; i < np * VG; i += 32) {
                const int r = i / VG, v = i - r * VG;
                __stcs(reinterpret_cast<float4*>(dsph + (p0 + r) * 3 * L) + v, reinterpret_cast<const float4*>(G0 + r * PG)[v]);
            }
    } else if (n - p0 >= PTS) {
        if (lane == 0) {
            const uint64_t policy = policy_evict_first();
            bulk_store_hint(sph + p0 * L, S0, S_BYTES, policy);
            if (DERIV >= 1) bulk_store_hint(dsph + p0 * 3 * L, G0, 3u * S_BYTES, policy);
            bulk_commit();
            bulk_wait_read<0>();   // shared memory must outlive the bulk stores' reads of it
        }
    } else {  // ragged last tile: byte count need not be a multiple of 16 -> plain stores
        const int np = (int)(n - p0);
        for (int i = lane; i < np * L; i += 32) st_cs(sph + p0 * L + i, S0[i]);
        if (DERIV >= 1)
            for (int i = lane; i < np * 3 * L; i += 32) st_cs(dsph + p0 * 3 * L + i, G0[i]);
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef void (*TpgKernel)(const TpgParams);

struct TpgLaunch {
    const void* func;
    TpgKernel kern;
    TpgParams prm;
    int64_t grid;
    int threads;
    size_t smem;
};

template <typename T, typename R, int LP, bool BB> static TpgKernel tpg_pick2(int deriv, int norm) {
    if (deriv == 0) return norm ? sph_tpg_kernel<T, R, 0, true, LP, BB> : sph_tpg_kernel<T, R, 0, false, LP, BB>;
    return norm ? sph_tpg_kernel<T, R, 1, true, LP, BB> : sph_tpg_kernel<T, R, 1, false, LP, BB>;
}
template <typename T, typename R> static TpgKernel tpg_pick(int deriv, int norm, int lp) {
    if (lp == 2) return tpg_pick2<T, R, 2, true>(deriv, norm);
    if (lp == 4) return tpg_pick2<T, R, 4, true>(deriv, norm);
    return tpg_pick2<T, R, 8, true>(deriv, norm);
}


// returns 0 and fills *out if the kernel applies: values or values + gradients whose smallest tile
// (4 points) still leaves room for several tiles per SM; 1 otherwise
static inline int tpg_plan(int smem_optin, int64_t n, int l_max, int normalized, int dtype, void* sph, void* dsph,
                           const void* xyz, const SphTables* d_tab, TpgLaunch* out) {
    const int deriv = dsph ? 1 : 0;
    const int esize = dtype == 0 ? 4 : 8;
    const int L = (l_max + 1) * (l_max + 1);
    const int64_t per_pt = (int64_t)L * esize * (deriv ? 4 : 1);
    // lanes per point: the most points per tile (16, 8, 4) whose image stays under 12 KB (measured:
    // the kernel is latency-bound, so small tiles = more warps in flight wins almost everywhere)
    int lp = g_opt.tpg_lp;
    if (lp != 2 && lp != 4 && lp != 8) {
        lp = 2;
        while (lp < 8 && (32 / lp) * per_pt > 12 * 1024) lp *= 2;
    }
    const int64_t tile_bytes = tpg_tile_bytes(32 / lp, L, esize, deriv);
    // longer rows go to the warp-per-point kernels (measured: f64 gradients at l_max = 16, a 37 KB
    // tile: 1.5 TB/s here, 1.8 there; f32 gradients at l_max = 24, 40 KB: 1.9 here, 1.0 there)
    if (tile_bytes > (dtype != 0 && deriv ? 32 : 48) * 1024) return 1;
    const int tab_bytes = tpg_tab_bytes(l_max, dtype != 0);
    int warps = 4;
    while (warps > 1 && tab_bytes + warps * tile_bytes > (smem_optin - 1024) / 2) warps >>= 1;   // >= 2 CTAs per SM
    if (tab_bytes + warps * tile_bytes > smem_optin - 1024) return 1;
    out->kern = dtype == 0 ? tpg_pick<float, double>(deriv, normalized, lp) : tpg_pick<double, dd>(deriv, normalized, lp);
    out->func = (const void*)out->kern;
    out->prm.xyz = xyz;
    out->prm.sph = sph;
    out->prm.dsph = dsph;
    out->prm.tab = d_tab;
    out->prm.n = n;
    out->prm.l_max = l_max;
    out->prm.warps_per_cta = warps;
    const int pts = 32 / lp;
    const int64_t n_tiles = (n + pts - 1) / pts;
    out->grid = (n_tiles + warps - 1) / warps;
    if (out->grid > 0x7fffffff) return 1;
    out->threads = warps * 32;
    out->smem = (size_t)tab_bytes + (size_t)warps * tile_bytes;
    return 0;
}

static inline void tpg_launch(const TpgLaunch& lw, cudaStream_t stream) {
    lw.kern<<<(unsigned)lw.grid, lw.threads, lw.smem, stream>>>(lw.prm);
}

}  // namespace sphb200
