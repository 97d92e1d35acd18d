// Fused density expansion (Eq. 1) for ANY l_max <= 32 with the contraction on the f64 tensor-core
// path, run-time l_max: the companion of kernel_expand.cuh (compile-time l_max <= 8, whose accumulators
// for every degree fit in registers).  Here the degrees are cut into BANDS of at most NTB N-tiles (8
// consecutive m of one degree each) and a CTA row (blockIdx.y) owns one band:
//     c[s, n, lm] = sum over the points k of segment s of  R[k, n, l] * Y_l^m(r_k / |r_k|),  l in the band.
// One warp per range of segments (persistent grid, ranges of equal point count, as kernel_expand.cuh).
// Per tile of 16 points:
//   1. two lanes per point (the even | the odd columns m) run the columns of the folded Eq. 7 with
//      run-time loops -- coefficients from the constant bank -- from the diagonal up to the band's last
//      degree, and store the band's harmonics (both branches of Eq. 5) into a [16][<= 8 NTB] image;
//      the powers of x + iy by Eq. 9.  Every band re-runs the recurrences (they are the smaller
//      part of a tile; what a band saves is the accumulators: NTB x MT x 2 doubles per lane);
//   2. the tile's radial values ([16][n_rad][l_max+1], one contiguous range) arrive as one bulk load,
//      requested after the previous tile's contraction;
//   3. per N-tile t of the band:  C_t [8 MT x 8] += R_l^T [8 MT x 16] . Y_t [16 x 8]  by mma.sync m8n8k4
//      (SASS DMMA), K = 4 points per step, accumulators in registers for the whole segment.
// At the end of a segment the accumulators go out by plain stores (a band's share of a coefficient row is
// neither contiguous over n nor 16-byte aligned).
#pragma once
#include "kernel_expand.cuh"

namespace sphb200 {

constexpr int EXRT_MAX_BANDS = 24;   // l_max = 32: 153 N-tiles in 11 bands of <= 16; 22 bands of <= 9 (n_rad > 8)
constexpr int EXRT_MAX_NTB = 16;     // N-tiles per band at most

struct ExpandRtParams {
    const void* xyz;        // [n, 3]
    const void* radial;     // [n, n_rad, l_max+1]
    const int64_t* seg_ptr; // [n_seg + 1]
    void* coeff;            // [n_seg, n_rad, L]
    int64_t n_seg;
    int n_rad, l_max;
    int warps_per_cta;
    int n_bands;
    unsigned char band_l0[EXRT_MAX_BANDS], band_l1[EXRT_MAX_BANDS];   // degrees of band b: l0 .. l1
    unsigned char band_tiles[EXRT_MAX_BANDS];                         // N-tiles of band b
    // N-tile t of band b: degree | sub-tile << 6 (m-indices 8 sub .. 8 sub + 7 of that degree) | first column in
    // the band's image << 10.  Read with a compile-time t: one uniform constant-bank load per use, so that the
    // unrolled loops over the tiles carry no running state.
    uint32_t tile_desc[EXRT_MAX_BANDS][EXRT_MAX_NTB];
};
__host__ __device__ constexpr int exrt_tile_l(uint32_t d) { return (int)(d & 63u); }
__host__ __device__ constexpr int exrt_tile_sub(uint32_t d) { return (int)((d >> 6) & 15u); }
__host__ __device__ constexpr int exrt_tile_col(uint32_t d) { return (int)(d >> 10); }

// shared memory of one warp: image of the band's harmonics [16][YP], radial image, mbarrier
template <int ESIZE, int NTB> struct ExpandRtShape {
    static constexpr int YP = 8 * NTB + 8 + 1;   // columns per point: the band's, 8 that a last fragment may over-read, odd pitch
    static constexpr int y_bytes = (TPB_PTS * YP * ESIZE + 15) & ~15;
    __host__ __device__ static constexpr int r_bytes(int n_rad, int l_max, int nrad_max) {
        return ((TPB_PTS * n_rad + nrad_max) * (l_max + 1) * ESIZE + 15) & ~15;
    }
    __host__ __device__ static constexpr int warp_bytes(int n_rad, int l_max, int nrad_max) {
        return y_bytes + r_bytes(n_rad, l_max, nrad_max) + 16;
    }
};

// MT: M-tiles of 8 radial indices (n_rad <= 8 MT); NTB: N-tiles per band
template <typename T, typename R, int MT, int NTB>
__global__ void __launch_bounds__(64, 8) sph_expand_rt_kernel(const ExpandRtParams prm) {
    using RT = rec<R>;
    using Shape = ExpandRtShape<sizeof(T), NTB>;
    constexpr int NRAD_MAX = 8 * MT, YP = Shape::YP;
    const SphTables& TB = c_tables_tpb;
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int n_rad = prm.n_rad, l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const int l0 = prm.band_l0[blockIdx.y], l1 = prm.band_l1[blockIdx.y];   // this CTA row's degrees
    // the warps of one CTA row share the segments in contiguous ranges of (nearly) equal point counts
    const int64_t W = (int64_t)gridDim.x * prm.warps_per_cta, w = (int64_t)blockIdx.x * prm.warps_per_cta + warp;
    const int64_t n_pts = __ldg(prm.seg_ptr + prm.n_seg);
    auto first_at_or_after = [&](int64_t v) {   // first segment whose first point is >= v
        int64_t lo = 0, hi = prm.n_seg;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (__ldg(prm.seg_ptr + mid) >= v) hi = mid;
            else lo = mid + 1;
        }
        return lo;
    };
    const int64_t seg0 = w == 0 ? 0 : first_at_or_after((n_pts * w + W - 1) / W);
    const int64_t seg1 = w == W - 1 ? prm.n_seg : first_at_or_after((n_pts * (w + 1) + W - 1) / W);
    const int cnt = (int)(seg1 - seg0);
    if (cnt <= 0) return;
    auto SP = [&](int j) { return __ldg(prm.seg_ptr + seg0 + j); };

    unsigned char* my = smem + (size_t)warp * Shape::warp_bytes(n_rad, l_max, NRAD_MAX);
    T* Ys = reinterpret_cast<T*>(my);
    T* Rs = reinterpret_cast<T*>(my + Shape::y_bytes);
    uint64_t* bar = reinterpret_cast<uint64_t*>(my + Shape::y_bytes + Shape::r_bytes(n_rad, l_max, NRAD_MAX));
    const int pl = lane & (TPB_PTS - 1);   // point inside the tile
    const int par = lane >> 4;             // which of the point's two lanes: it takes the columns m = par (mod 2)
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    const T* __restrict__ radial = static_cast<const T*>(prm.radial);
    T* __restrict__ coeff = static_cast<T*>(prm.coeff);
    const int rstride = n_rad * (l_max + 1);   // radial values per point
    const bool r_bulk = (rstride * (int)sizeof(T)) % 16 == 0;
    if (lane == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    uint32_t phase = 0u;
    __syncwarp();

    const int fr = lane >> 2, fk = lane & 3;   // fragment coordinates of this lane
    double acc[MT][NTB][2];
    auto zero_acc = [&]() {
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int t = 0; t < NTB; ++t) acc[mt][t][0] = acc[mt][t][1] = 0.0;
    };
    const uint32_t* desc = prm.tile_desc[blockIdx.y];   // (constant bank)
    const int n_tiles = prm.band_tiles[blockIdx.y];
    // c[seg, n, lm] of segment j: lane holds C[n = fr + 8 mt][m-index 8 sub + 2 fk + {0, 1}] of every tile
    auto flush = [&](int j) {
        const int64_t seg = seg0 + j;
#pragma unroll
        for (int t = 0; t < NTB; ++t) {
            if (t < n_tiles) {
                const uint32_t d = desc[t];
                const int tl = exrt_tile_l(d), jm0 = 8 * exrt_tile_sub(d) + 2 * fk;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int n = fr + 8 * mt;
#pragma unroll
                    for (int e = 0; e < 2; ++e)
                        if (n < n_rad && jm0 + e < 2 * tl + 1)
                            coeff[(seg * n_rad + n) * L + tl * tl + jm0 + e] = static_cast<T>(acc[mt][t][e]);
                }
            }
        }
    };
    auto settle = [&](int& j, int64_t& k0) {
        while (j < cnt && k0 >= SP(j + 1)) {
            ++j;
            if (j < cnt) k0 = SP(j);
        }
    };
    auto fetch_radial = [&](int j, int64_t k0) {
        const int np = (int)min((int64_t)TPB_PTS, SP(j + 1) - k0);
        if (r_bulk) {
            if (lane == 0) {
                const uint32_t bytes = (uint32_t)(np * rstride * (int)sizeof(T));
                mbar_arrive_expect_tx(bar, bytes);
                bulk_load(Rs, radial + k0 * rstride, bytes, bar);
            }
        } else {
            for (int i = lane; i < np * rstride; i += 32) cp_async_elem(Rs + i, radial + k0 * rstride + i);
            cp_async_commit();
        }
        for (int i = np * rstride + lane; i < TPB_PTS * rstride; i += 32) Rs[i] = T(0);
    };
    auto fetch_xyz = [&](int j, int64_t k0, T& xa, T& ya, T& za) {
        const int np = (int)min((int64_t)TPB_PTS, SP(j + 1) - k0);
        xa = T(0), ya = T(0), za = T(1);   // lanes past the end compute a harmless point
        if (pl < np) {
            xa = __ldg(xyz + 3 * (k0 + pl) + 0);
            ya = __ldg(xyz + 3 * (k0 + pl) + 1);
            za = __ldg(xyz + 3 * (k0 + pl) + 2);
        }
    };

    int j = 0;
    int64_t k0 = SP(0);
    settle(j, k0);
    T xn = T(0), yn = T(0), zn = T(1);
    if (j < cnt) {
        fetch_radial(j, k0);
        fetch_xyz(j, k0, xn, yn, zn);
    }
    zero_acc();
    const int col_base = l0 * l0;   // column of harmonic (l, m) in the image: l (l + 1) + m - l0^2
    while (j < cnt) {
        const int np = (int)min((int64_t)TPB_PTS, SP(j + 1) - k0);
        const double x = static_cast<double>(xn), y = static_cast<double>(yn), z = static_cast<double>(zn);
        int jn = j;
        int64_t kn = k0 + TPB_PTS;
        settle(jn, kn);
        if (jn < cnt) fetch_xyz(jn, kn, xn, yn, zn);   // in flight through this tile
        // ---- harmonics of the band for the tile's points: two lanes per point ---------------------
        {
            R X, Y, Z;
            double rinv;
            RT::normalize(x, y, z, X, Y, Z, rinv);
            T* S = Ys + pl * YP;
            // The two lanes of a point share the COLUMNS: lane `par` takes m = par, par + 2, ... and stores both
            // harmonics (l, +m) and (l, -m) of every entry, so that no recurrence runs twice (with run-time
            // loops the two lanes may run different columns: no divergence beyond the trip counts).
            // Its powers (c_m, s_m) advance by (x + iy)^2.
            const R X2 = X * X - Y * Y, Y2 = (X * Y) * 2.0;
            R c = par ? X : RT::make(1.0, 0.0), s = par ? Y : RT::make(0.0, 0.0);
            for (int m = par; m <= l1; m += 2) {
                const double Ac = m == 0 ? SPH_INV_SQRT2 : to_double(c), As = to_double(s);
                // column m of the folded Eq. 7 (r^2 = 1 on the unit sphere) from the diagonal to the band's end;
                // Qt_{m-1}^m = 0, so the first step needs no special case
                R q = RT::make(TB.D_hi[m], TB.D_lo[m]), qp = RT::make(0.0, 0.0);
                int t1 = SPH_TRI(m, m);
                auto advance = [&](int l) {   // (q, qp) = (Qt_l^m, Qt_{l-1}^m) -> (Qt_{l+1}^m, Qt_l^m)
                    t1 += l + 1;              // SPH_TRI(l + 1, m)
                    const R qn = rec_step(TB.A_hi[t1], TB.A_lo[t1], TB.B_hi[t1], TB.B_lo[t1], Z, q, qp);
                    qp = q;
                    q = qn;
                };
                int l = m;
#pragma unroll 2
                for (; l < l0; ++l) advance(l);          // the rows below the band: recurrence only
                // the band's rows: harmonic (l, +-m) sits in column l (l + 1) +- m - l0^2; + 2 (l + 1) per row
                int sc = l * (l + 1) + m - col_base;
                const int dm2 = 2 * m;
#pragma unroll 2
                for (;; ++l) {
                    const double Q = to_double(q);
                    S[sc - dm2] = static_cast<T>(Q * As);   // Eq. 5; for m = 0 the cos store that follows overwrites it
                    S[sc] = static_cast<T>(Q * Ac);
                    if (l == l1) break;
                    advance(l);
                    sc += 2 * l + 2;
                }
                const R cn = X2 * c - Y2 * s;   // Eq. 9, two steps at once
                const R sn = X2 * s + Y2 * c;
                c = cn;
                s = sn;
            }
        }
        if (r_bulk) {   // this tile's radial image has landed (it was in flight through this evaluation)
            mbar_wait(bar, phase);
            phase ^= 1u;
        } else {
            cp_async_wait_all();
        }
        __syncwarp();
        // ---- contract over the tile's points, 4 at a time (K of the DMMA) -------------------------
        // What a fragment reads outside the valid ranges (n >= n_rad: the next point's radial values or
        // the padding; m-index beyond 2l+1: the next degree's harmonics or the image's slack) only reaches
        // rows / columns of C that are never stored.
#pragma unroll
        for (int ks = 0; ks < TPB_PTS / 4; ++ks) {
            if (4 * ks < np) {
                const int p = 4 * ks + fk;
                const T* rp = Rs + p * rstride + fr * (l_max + 1);
                const T* yp = Ys + p * YP + fr;
#pragma unroll
                for (int t = 0; t < NTB; ++t) {
                    if (t < n_tiles) {
                        const uint32_t d = desc[t];
                        const int tl = exrt_tile_l(d);
                        double a[MT];   // (re-read for every sub-tile of a degree: cheaper than carrying the state)
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) a[mt] = static_cast<double>(rp[8 * mt * (l_max + 1) + tl]);
                        const double bv = static_cast<double>(yp[exrt_tile_col(d)]);
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) dmma_m8n8k4(acc[mt][t], a[mt], bv);
                    }
                }
            }
        }
        __syncwarp();   // every lane is done with the radial image and the image of the harmonics
        if (jn < cnt) fetch_radial(jn, kn);   // lands while the next tile's harmonics are evaluated
        if (jn != j) {   // the segment is complete
            flush(j);
            zero_acc();
        }
        j = jn;
        k0 = kn;
    }
    // empty segments: zeros (the CTA row of the first band writes the whole rows)
    if (blockIdx.y == 0)
        for (int je = 0; je < cnt; ++je) {
            if (SP(je) == SP(je + 1))
                for (int i = lane; i < n_rad * L; i += 32) coeff[(seg0 + je) * n_rad * L + i] = T(0);
        }
}

}  // namespace sphb200
