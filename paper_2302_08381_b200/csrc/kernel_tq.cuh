// "tq" forward kernel: two phases per batch of points, the whole CTA on both.  Any l_max, values /
// + gradients / + Hessians, run-time l_max (12 instantiations in all).
//
// Why (profiles/r2_*): the unrolled tpb kernels keep a point's whole Legendre
// column in registers and stage 16 points per warp, so from l_max ~ 11 (gradients) / 6 (Hessians)
// they run at 168-255 registers with 43-74 KB images: 3-8 warps per SM, latency-bound.  The
// run-time kernels that took over there (tpg, w) tie the recurrences and the assembly to the same
// lanes (lane = column class, or lane = m), so most lanes idle through one of the two.  Here the two
// are separate phases with their own mapping, and the image is sized by the store engine's needs
// (a contiguous byte range per output array, 16-byte aligned), not by the warp width:
//
//   phase A  lane = POINT.  The batch's points (32, 16 for the longest rows) run Eq. 9 and
//            the folded Eq. 7 (tables.h) -- double for f32 I/O, double-double for f64 I/O --
//            with warp-uniform coefficient loads from the constant bank; the columns m of the
//            triangle are dealt to the CTA's warps in snake order (balanced lengths).  Qt_l^m, (c_m, s_m)
//            and (u, 1/r) of every point go to a scratch in shared memory as f64.
//   phase B  lane = one (l, m >= 0) PAIR of one point of the current tile (tile = the fewest points
//            whose rows are a 16-byte multiple: 4 f32 / 2 f64, or more while the image stays
//            small).  A lane assembles every requested component of both harmonics (l, +-m): the
//            Legendre side of Eq. 10 -- and, for the normalised variant, the chain rule of
//            P:108 folded into it -- is computed once per pair as a handful of coefficients, each
//            branch of Eq. 5 is then 1 / 6 / 21 multiply-adds on (A, A_x, A_y, A_xx, A_xy).
//            Lanes of a warp hold consecutive m of one row, so scratch reads and image writes are
//            conflict-free for every row length (no padding, unlike tpb at l_max = 3 mod 4).
//   store    the tile's image is byte-identical to global memory: 1 / 2 / 3 bulk stores (TMA, SASS
//            UBLKCP); two images, so a tile drains while the next is assembled; ONE barrier per tile.
//
// Folded chain rule (derivation in DESIGN.md section 5): with Q, q1, qz, q2, qxz, qzz as in
// sph_core.cuh (the table ratios applied), at the evaluation point (x,y,z) (= u for normalised),
//   solid       E1 = q1,  EZ = qz,  F2 = q2,  FXZ = qxz,  FZZ = qzz
//   normalised  lQ = l Q, w = (l+2) lQ,
//               E1 = q1 - lQ,  EZ = qz - lQ z,  F2 = q2 - 2 l q1 + w,
//               FXZ = qxz - l qz + z (w - l q1),  FZZ = qzz + z (w z - 2 l qz) - lQ
//   Y   = Q A
//   g_x = x E1 A + Q A_x,  g_y = y E1 A + Q A_y,  g_z = EZ A                          (times 1/r)
//   H_xx = (E1 + x^2 F2) A + 2 x E1 A_x + Q A_xx,   H_yy = (E1 + y^2 F2) A + 2 y E1 A_y - Q A_xx,
//   H_xy = x y F2 A + x E1 A_y + y E1 A_x + Q A_xy,
//   H_xz = x FXZ A + EZ A_x,  H_yz = y FXZ A + EZ A_y,  H_zz = FZZ A                   (times 1/r^2)
// which is Eq. 10 once / twice for the solid harmonics and the Euler-simplified chain rule of
// sph_core.cuh for the normalised ones, regrouped by the azimuthal factor they multiply.
#pragma once
#include "options.h"
#include "ptx.cuh"
#include "sph_core.cuh"

namespace sphb200 {

struct TqParams {
    const void* xyz;
    void* sph;
    void* dsph;
    void* ddsph;
    const SphTables* tab;        // global-memory copy of the tables (phase B: G1, Gz, H2, Hxz, Hzz)
    const unsigned short* lm;    // [(l_max+1)(l_max+2)/2]: l | m << 8 of triangle index t
    int64_t n;
    int l_max;
    int batch;                   // points per phase-A batch: 32, 16 or 8
    int pts_tile;                // points per image; divides batch
    int batches_per_cta;         // consecutive batches one CTA works through
};

constexpr int TQ_MAX_WARPS = 8;

// shared-memory carve-up (bytes), identical on host and device
struct TqSmem {
    int T, TP, CP;
    size_t q_bytes, cs_bytes, pt_bytes, img_bytes, total;
    __host__ __device__ TqSmem(int l_max, int deriv, int esize, int batch, int pts_tile) {
        T = (l_max + 1) * (l_max + 2) / 2;
        TP = (T + 3) | 1;          // doubles per point: three finite pad entries, odd pitch (conflict-free lane = point stores)
        CP = (l_max + 1) | 1;      // (c, s) pairs per point, odd pitch
        q_bytes = (size_t)batch * TP * 8;
        cs_bytes = (size_t)batch * CP * 16;
        pt_bytes = (size_t)batch * 32;
        const int rows = deriv == 0 ? 1 : (deriv == 1 ? 4 : 13);
        const size_t L = (size_t)(l_max + 1) * (l_max + 1);
        img_bytes = ((size_t)pts_tile * rows * L * esize + 127) & ~(size_t)127;
        total = ((q_bytes + cs_bytes + pt_bytes + 127) & ~(size_t)127) + 2 * img_bytes;
    }
    __host__ __device__ size_t img_offset() const { return (q_bytes + cs_bytes + pt_bytes + 127) & ~(size_t)127; }
};

template <typename T, typename R, int DERIV, bool NORM>
__global__ void __launch_bounds__(TQ_MAX_WARPS * 32, 2) sph_tq_kernel(const TqParams prm) {
    using RT = rec<R>;
    constexpr int ES = (int)sizeof(T);
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int W = blockDim.x >> 5;
    const int l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const int B = prm.batch, P = prm.pts_tile;
    const TqSmem lay(l_max, DERIV, ES, B, P);
    const int TT = lay.T, TP = lay.TP, CP = lay.CP;
    double* __restrict__ Qs = reinterpret_cast<double*>(smem);
    double2* __restrict__ CS = reinterpret_cast<double2*>(smem + lay.q_bytes);
    double4* __restrict__ PT = reinterpret_cast<double4*>(smem + lay.q_bytes + lay.cs_bytes);
    unsigned char* img0 = smem + lay.img_offset();
    const int64_t n = prm.n;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    T* __restrict__ dsph = static_cast<T*>(prm.dsph);
    T* __restrict__ ddsph = static_cast<T*>(prm.ddsph);
    const SphTables& TB = c_tables;
    const uint64_t policy = policy_evict_first();

    // pad entries behind every point's triangle: read (times a zero coefficient) by phase B
    for (int i = threadIdx.x; i < B * 3; i += blockDim.x) Qs[(i / 3) * TP + TT + (i % 3)] = 0.0;

    const uint32_t s_bytes = (uint32_t)P * L * ES;
    int tile_no = 0;   // tiles this CTA has issued: parity picks the image
    for (int bi = 0; bi < prm.batches_per_cta; ++bi) {
        const int64_t b0 = ((int64_t)blockIdx.x * prm.batches_per_cta + bi) * B;
        if (b0 >= n) break;

        // ---- phase A: lane = point --------------------------------------------------------------
        __syncthreads();   // the previous batch's phase B has finished reading the scratch
        if (lane < B) {
            const int64_t p = b0 + lane;
            double x = 0.0, y = 0.0, z = 1.0;   // lanes past the end compute a harmless point
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
            if (warp == W - 1) {   // Eq. 9 and the point itself: the warp with the shortest columns
                PT[lane] = make_double4(to_double(X), to_double(Y), to_double(Z), rinv);
                R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
                double2* cs = CS + lane * CP;
                for (int m = 0; m <= l_max; ++m) {
                    cs[m] = make_double2(to_double(c), to_double(s));
                    const R cn = X * c - Y * s;
                    const R sn = X * s + Y * c;
                    c = cn;
                    s = sn;
                }
            }
            // columns of the folded Eq. 7, dealt to the warps in snake order: m = w, 2W-1-w, 2W+w, ...
            double* q_out = Qs + lane * TP;
            for (int i = 0; i * W <= l_max; ++i) {
                const int m = (i & 1) ? (i + 1) * W - 1 - warp : i * W + warp;
                if (m > l_max) continue;
                int t = SPH_TRI(m, m);
                R q = RT::make(TB.D_hi[m], TB.D_lo[m]), qp = RT::make(0.0, 0.0);
                q_out[t] = to_double(q);
                for (int l = m + 1; l <= l_max; ++l) {
                    t += l;   // SPH_TRI(l, m) - SPH_TRI(l-1, m) = l
                    const R a = RT::make(TB.A_hi[t], TB.A_lo[t]);
                    R qn;
                    if (l == m + 1) {
                        qn = a * (Z * q);
                    } else {
                        const R w = NORM ? qp : r2 * qp;
                        qn = a * (Z * q) - RT::make(TB.B_hi[t], TB.B_lo[t]) * w;
                    }
                    qp = q;
                    q = qn;
                    q_out[t] = to_double(q);
                }
            }
        }
        __syncthreads();

        // ---- phase B: lane = (point of the tile, pair) --------------------------------------------
        const int n_tiles = B / P;
        for (int ti = 0; ti < n_tiles; ++ti) {
            const int64_t p0 = b0 + (int64_t)ti * P;
            if (p0 >= n) break;
            unsigned char* img = img0 + (size_t)(tile_no & 1) * lay.img_bytes;
            T* __restrict__ S0 = reinterpret_cast<T*>(img);
            T* __restrict__ G0 = reinterpret_cast<T*>(img + s_bytes);
            T* __restrict__ H0 = reinterpret_cast<T*>(img + 4u * s_bytes);
            const int items = P * TT;
            for (int e0 = warp * 32; e0 < items; e0 += W * 32) {
                const int e = e0 + lane;
                if (e >= items) break;
                int pi = e0 / TT;           // warp-uniform division, then at most a few steps
                int t = e - pi * TT;
                while (t >= TT) {
                    t -= TT;
                    ++pi;
                }
                const int pb = ti * P + pi;   // point inside the batch
                const double4 pt = PT[pb];
                const double x = pt.x, y = pt.y, z = pt.z, ri = pt.w;
                const unsigned lmv = __ldg(prm.lm + t);
                const int l = (int)(lmv & 0xffu), m = (int)(lmv >> 8);
                const double* __restrict__ Qp = Qs + pb * TP;
                const double2* __restrict__ cs = CS + pb * CP;
                const double Q = Qp[t];
                const double2 cs0 = cs[m];
                const double Ac = (m == 0) ? SPH_INV_SQRT2 : cs0.x, As = cs0.y;
                const int kc = l * (l + 1) + m, ks = kc - 2 * m;
                T* __restrict__ S = S0 + pi * L;
                S[kc] = static_cast<T>(Q * Ac);
                if (m > 0) S[ks] = static_cast<T>(Q * As);
                if constexpr (DERIV >= 1) {
                    const double dl = (double)l, dm = (double)m;
                    const int t1 = t - l;
                    const double q1 = __ldg(&prm.tab->G1[t]) * Qp[t1 + 1];   // F_l^m Q_{l-1}^{m+1}
                    const double qz = __ldg(&prm.tab->Gz[t]) * Qp[t1];       // F_l^m (l+m) Q_{l-1}^m
                    const double2 cs1 = cs[m >= 1 ? m - 1 : 0];
                    // Eq. 10: cos: A_x = m c_{m-1}, A_y = -m s_{m-1}; sin: A_x = m s_{m-1}, A_y = m c_{m-1}
                    const double mc1 = dm * cs1.x, ms1 = dm * cs1.y;
                    const double lQ = dl * Q;
                    const double E1 = NORM ? q1 - lQ : q1;
                    const double EZ = NORM ? SPH_FMA(-lQ, z, qz) : qz;
                    const double sg = NORM ? ri : 1.0;
                    const double E1g = E1 * sg;
                    const double ax = x * E1g, ay = y * E1g, az = EZ * sg, Qg = Q * sg;
                    T* __restrict__ G = G0 + pi * 3 * L;
                    G[kc] = static_cast<T>(SPH_FMA(ax, Ac, Qg * mc1));
                    G[L + kc] = static_cast<T>(SPH_FMA(ay, Ac, -(Qg * ms1)));
                    G[2 * L + kc] = static_cast<T>(az * Ac);
                    if (m > 0) {
                        G[ks] = static_cast<T>(SPH_FMA(ax, As, Qg * ms1));
                        G[L + ks] = static_cast<T>(SPH_FMA(ay, As, Qg * mc1));
                        G[2 * L + ks] = static_cast<T>(az * As);
                    }
                    if constexpr (DERIV >= 2) {
                        const int t2 = t1 - l + 1;
                        const double q2 = __ldg(&prm.tab->H2[t]) * Qp[t2 + 2];    // F_l^m Q_{l-2}^{m+2}
                        const double qxz = __ldg(&prm.tab->Hxz[t]) * Qp[t2 + 1];  // F_l^m (l+m) Q_{l-2}^{m+1}
                        const double qzz = __ldg(&prm.tab->Hzz[t]) * Qp[t2];      // F_l^m (l+m)(l+m-1) Q_{l-2}^m
                        const double2 cs2 = cs[m >= 2 ? m - 2 : 0];
                        const double dmm = dm * (dm - 1.0);
                        // Eq. 10 twice: cos: A_xx = m(m-1) c_{m-2}, A_xy = -m(m-1) s_{m-2}; sin: s_{m-2}, c_{m-2}
                        const double mmc2 = dmm * cs2.x, mms2 = dmm * cs2.y;
                        double F2 = q2, FXZ = qxz, FZZ = qzz;
                        if (NORM) {
                            const double w = (dl + 2.0) * lQ;
                            F2 = SPH_FMA(-2.0 * dl, q1, q2 + w);
                            FXZ = SPH_FMA(z, SPH_FMA(-dl, q1, w), SPH_FMA(-dl, qz, qxz));
                            FZZ = SPH_FMA(z, SPH_FMA(w, z, -2.0 * dl * qz), qzz) - lQ;
                        }
                        const double sh = NORM ? ri * ri : 1.0;
                        const double E1h = E1 * sh, F2h = F2 * sh, Qh = Q * sh;
                        const double cxx = SPH_FMA(x * x, F2h, E1h), cyy = SPH_FMA(y * y, F2h, E1h), cxy = (x * y) * F2h;
                        const double bx = x * E1h, by = y * E1h, bx2 = bx + bx, by2 = by + by;
                        const double FXZh = FXZ * sh;
                        const double cxz = x * FXZh, cyz = y * FXZh, ezh = EZ * sh, czz = FZZ * sh;
                        T* __restrict__ H = H0 + pi * 9 * L;
                        auto put = [&](int k, double A, double Ax, double Ay, double Axx, double Axy) {
                            const double QAxx = Qh * Axx;
                            const T hxx = static_cast<T>(SPH_FMA(cxx, A, SPH_FMA(bx2, Ax, QAxx)));
                            const T hyy = static_cast<T>(SPH_FMA(cyy, A, SPH_FMA(by2, Ay, -QAxx)));
                            const T hxy = static_cast<T>(SPH_FMA(cxy, A, SPH_FMA(bx, Ay, SPH_FMA(by, Ax, Qh * Axy))));
                            const T hxz = static_cast<T>(SPH_FMA(cxz, A, ezh * Ax));
                            const T hyz = static_cast<T>(SPH_FMA(cyz, A, ezh * Ay));
                            const T hzz = static_cast<T>(czz * A);
                            // rows = xx xy xz yx yy yz zx zy zz (both triangles stored, exactly equal)
                            H[k] = hxx;
                            H[L + k] = hxy;
                            H[2 * L + k] = hxz;
                            H[3 * L + k] = hxy;
                            H[4 * L + k] = hyy;
                            H[5 * L + k] = hyz;
                            H[6 * L + k] = hxz;
                            H[7 * L + k] = hyz;
                            H[8 * L + k] = hzz;
                        };
                        put(kc, Ac, mc1, -ms1, mmc2, -mms2);
                        if (m > 0) put(ks, As, ms1, mc1, mms2, mmc2);
                    }
                }
            }
            // the other image's stores (issued one tile ago) must have read it before anyone writes
            // there again; this tile's image must be visible to the async proxy
            fence_proxy_async_smem();
            if (threadIdx.x == 0) bulk_wait_read<0>();
            __syncthreads();
            const bool full = n - p0 >= P;
            if (full && ((s_bytes & 15u) == 0)) {
                if (threadIdx.x == 0) {
                    bulk_store_hint(sph + p0 * L, S0, s_bytes, policy);
                    if (DERIV >= 1) bulk_store_hint(dsph + p0 * 3 * L, G0, 3u * s_bytes, policy);
                    if (DERIV >= 2) bulk_store_hint(ddsph + p0 * 9 * L, H0, 9u * s_bytes, policy);
                    bulk_commit();
                }
            } else {   // ragged last tile (or a row length that is not a 16-byte multiple per tile): plain stores
                const int np = (int)(full ? P : n - p0);
                for (int i = threadIdx.x; i < np * L; i += blockDim.x) st_cs(sph + p0 * L + i, S0[i]);
                if (DERIV >= 1)
                    for (int i = threadIdx.x; i < np * 3 * L; i += blockDim.x) st_cs(dsph + p0 * 3 * L + i, G0[i]);
                if (DERIV >= 2)
                    for (int i = threadIdx.x; i < np * 9 * L; i += blockDim.x) st_cs(ddsph + p0 * 9 * L + i, H0[i]);
                __syncthreads();   // the image is free again only when every thread has copied its share
            }
            ++tile_no;
        }
    }
    // shared memory must outlive the bulk stores' reads of it
    if (threadIdx.x == 0) bulk_wait_read<0>();
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef void (*TqKernel)(const TqParams);

struct TqLaunch {
    const void* func;
    TqKernel kern;
    TqParams prm;
    int64_t grid;
    int threads;
    size_t smem;
};

template <typename T, typename R> static TqKernel tq_pick(int deriv, int norm) {
    if (deriv == 0) return norm ? sph_tq_kernel<T, R, 0, true> : sph_tq_kernel<T, R, 0, false>;
    if (deriv == 1) return norm ? sph_tq_kernel<T, R, 1, true> : sph_tq_kernel<T, R, 1, false>;
    return norm ? sph_tq_kernel<T, R, 2, true> : sph_tq_kernel<T, R, 2, false>;
}

// returns 0 and fills *out if a launch shape fits: the smallest tile whose arrays are 16-byte
// multiples (4 points f32, 2 f64; 1 when the row itself is one), doubled while the image stays
// under ~20 KB; the largest batch (32, 16, 8 points) that leaves room for two CTAs per SM, or for
// one if that is all that fits; 1 otherwise (rows too long for two full-row images)
static inline int tq_plan(int sm_count, int smem_optin, int64_t n, int l_max, int normalized, int dtype, void* sph,
                          void* dsph, void* ddsph, const void* xyz, const SphTables* d_tab, const unsigned short* d_lm,
                          TqLaunch* out) {
    const int deriv = ddsph ? 2 : (dsph ? 1 : 0);
    const int esize = dtype == 0 ? 4 : 8;
    const int rows = deriv == 0 ? 1 : (deriv == 1 ? 4 : 13);
    const int64_t L = (int64_t)(l_max + 1) * (l_max + 1);
    const int64_t row_bytes = L * esize;
    int pts = 16 / esize;
    if (row_bytes % 16 == 0) pts = 1;
    else if ((2 * row_bytes) % 16 == 0) pts = 2;
    while (pts < 32 && 2 * pts * rows * row_bytes <= 20 * 1024) pts *= 2;
    if (g_opt.tq_points > 0) pts = g_opt.tq_points;
    if (pts > 32 || 32 % pts != 0) return 1;
    const int budget = smem_optin - 1024;
    int batch = 0;
    for (int want_ctas = 2; want_ctas >= 1 && !batch; --want_ctas)
        for (int b = 32; b >= 8 && b >= pts; b >>= 1) {
            TqSmem lay(l_max, deriv, esize, b, pts);
            if ((int64_t)lay.total * want_ctas + 1024 * want_ctas <= (want_ctas == 1 ? budget : 227 * 1024)) {
                if ((int64_t)lay.total > budget) continue;
                batch = b;
                break;
            }
        }
    if (!batch) return 1;
    TqSmem lay(l_max, deriv, esize, batch, pts);
    out->kern = dtype == 0 ? tq_pick<float, double>(deriv, normalized) : tq_pick<double, dd>(deriv, normalized);
    out->func = (const void*)out->kern;
    out->prm.xyz = xyz;
    out->prm.sph = sph;
    out->prm.dsph = dsph;
    out->prm.ddsph = ddsph;
    out->prm.tab = d_tab;
    out->prm.lm = d_lm;
    out->prm.n = n;
    out->prm.l_max = l_max;
    out->prm.batch = batch;
    out->prm.pts_tile = pts;
    const int64_t n_batches = (n + batch - 1) / batch;
    // a few batches per CTA amortise the pad initialisation and the launch; keep >= ~8 CTAs per SM
    int64_t bpc = n_batches / ((int64_t)sm_count * 16);
    if (bpc > 4) bpc = 4;
    if (bpc < 1) bpc = 1;
    out->prm.batches_per_cta = (int)bpc;
    out->grid = (n_batches + bpc - 1) / bpc;
    if (out->grid > 0x7fffffff) return 1;
    out->threads = TQ_MAX_WARPS * 32;
    out->smem = lay.total;
    return 0;
}

static inline void tq_launch(const TqLaunch& lw, cudaStream_t stream) {
    lw.kern<<<(unsigned)lw.grid, lw.threads, lw.smem, stream>>>(lw.prm);
}

}  // namespace sphb200
