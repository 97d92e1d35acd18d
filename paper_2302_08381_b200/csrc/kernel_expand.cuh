// Fused density expansion (Eq. 1):
//     c[s, n, lm] = sum over the points k of segment s of  R[k, n, l] * Y_l^m(r_k / |r_k|)
// with the radial values R_nl(r_k) supplied by the caller (the paper leaves the radial basis to the
// application) and segments given by ascending offsets (e.g. the neighbour list of centre s).
// The harmonics never reach HBM: per point the kernel reads 3 + n_rad (l_max+1) values, and it
// writes n_rad L values per SEGMENT -- against L values written and read back per POINT when
// sphericart_cuda_compute is followed by a separate contraction.
//
// Persistent grid: every warp takes a contiguous range of segments of (nearly) equal POINT count.  Per
// tile of 16 points of a segment
//   1. two lanes per point (cos | sin branch of Eq. 5, as in kernel_tpb.cuh, l_max compile-time)
//      evaluate the normalised harmonics into a [16][L] image in shared memory (f64 / double-double
//      recurrences, stored in the I/O type; in f64 for l_max <= 3), while the tile's radial values
//      ([16][n_rad][l_max+1], one contiguous range of global memory) land next to it as ONE bulk load
//      (TMA, mbarrier), requested right after the previous tile's contraction;
//   2. the contraction over the tile's points is, for every degree l, a small dense product
//          C_l [n_rad x (2l+1)]  +=  R_l^T [n_rad x 16]  .  Y_l [16 x (2l+1)]
//      and runs on the f64 tensor-core path: mma.sync m8n8k4 (SASS DMMA), M = radial index n, N = 8
//      consecutive m of one l, K = 4 points per step; fragments come straight from the two images
//      (widened to f64 as they are read), accumulators stay in registers for the whole segment.
//      (Measured on B200: DMMA sustains the same 18 T FMA/s as DFMA, but one instruction does 256 FMAs
//      instead of 32 and needs 2 operand loads instead of 2 per 32: the first version of this kernel,
//      lane = harmonic with one LDS per DFMA, was bound by the LSU pipe and by issue slots, not by f64
//      throughput.)
// At the end of a segment the accumulators are staged in shared memory and leave as one bulk store.
// l_max > 8: kernel_expand_rt.cuh (the degrees in bands, run-time loops).
#pragma once
#include "kernel_tpb.cuh"

namespace sphb200 {

struct ExpandParams {
    const void* xyz;        // [n, 3]
    const void* radial;     // [n, n_rad, l_max+1]
    const int64_t* seg_ptr; // [n_seg + 1]
    void* coeff;            // [n_seg, n_rad, L]
    int64_t n_seg;
    int n_rad;
    int warps_per_cta;
};

constexpr int EXP_MAX_RAD = 16;   // two M-tiles of 8 radial indices

// N-tiles of the contraction: degree l has ceil((2l+1)/8) tiles of 8 consecutive m
template <int LMAX> struct ExpandTiles {
    __host__ __device__ static constexpr int of(int l) { return (2 * l + 1 + 7) / 8; }
    __host__ __device__ static constexpr int first(int l) {
        int s = 0;
        for (int i = 0; i < l; ++i) s += of(i);
        return s;
    }
    static constexpr int total = first(LMAX + 1);
};

// D (8x8, f64) += A (8x4, row) * B (4x8, col): lane holds A[lane/4][lane%4], B[lane%4][lane/4],
// D[lane/4][2 (lane%4) + {0,1}]
__device__ __forceinline__ void dmma_m8n8k4(double (&d)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d[0]), "+d"(d[1])
                 : "d"(a), "d"(b));
}

template <int ESIZE, int LMAX> struct ExpandShape {
    static constexpr int L = (LMAX + 1) * (LMAX + 1);
    static constexpr int passes = (L + 31) / 32;
    // per warp: Y image [16][L] + ONE radial image [16][n_rad][LMAX+1], both in the I/O type (the
    // next tile's radial values are requested after this tile's contraction and arrive -- one bulk load
    // -- while the next tile's harmonics are evaluated),
    // the radial image followed by nrad_max rows of padding (the unrolled contraction reads
    // nrad_max rows per point whatever n_rad is; what it reads past n_rad only reaches rows of C
    // that are dropped), + the warp's segment offsets
    // The image of the harmonics is held in the I/O type, except for l_max <= 3 where it is f64 (rows an odd
    // number of doubles apart): the tolerance 5e-6 (l_max + 1) is tightest there, an f32 image alone uses it up
    // (measured: l_max = 1, n_rad = 16: 1.001e-5 against 1.0e-5), and the image is at most 2 KB anyway.
    static constexpr bool y_f64 = LMAX <= 3;
    static constexpr int y_size = y_f64 ? 8 : ESIZE;
    static constexpr int y_pitch = y_f64 ? (L | 1) : L;
    static constexpr int y_bytes = (TPB_PTS * y_pitch * y_size + 15) & ~15;
    __host__ __device__ static constexpr int r_bytes(int n_rad, int nrad_max) {
        return ((TPB_PTS * n_rad + nrad_max) * (LMAX + 1) * ESIZE + 15) & ~15;
    }
    // + a staging image of one segment's coefficients [n_rad][L] (leaves as one bulk store) + two
    // mbarriers (one per radial image: the image arrives as ONE bulk load)
    __host__ __device__ static constexpr int c_bytes(int n_rad) { return (n_rad * L * ESIZE + 15) & ~15; }
    __host__ __device__ static constexpr int warp_bytes(int n_rad, int nrad_max) {
        return y_bytes + r_bytes(n_rad, nrad_max) + c_bytes(n_rad) + 16;
    }
};

template <typename T, typename R, int LMAX, int NRAD_MAX>
__global__ void __launch_bounds__(128, 4) sph_expand_kernel(const ExpandParams prm) {
    using RT = rec<R>;
    using Shape = ExpandShape<sizeof(T), LMAX>;
    constexpr int L = Shape::L;
    const SphTables& TB = c_tables_tpb;
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int n_rad = prm.n_rad;
    // Persistent grid: the warps share the segments in contiguous ranges of (nearly) equal POINT counts
    // -- warp w of W takes the segments whose first point lies in [w n / W, (w+1) n / W) -- so that all
    // of them finish together whatever the segment lengths (a grid of one CTA per few segments ran 3.5
    // waves and idled through the last one).  Two binary searches over seg_ptr per warp.
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
    const int cnt = (int)(seg1 - seg0);   // this warp's segments j = 0 .. cnt-1 are the points SP(j) .. SP(j+1)-1
    if (cnt <= 0) return;
    auto SP = [&](int j) { return __ldg(prm.seg_ptr + seg0 + j); };
    unsigned char* my = smem + (size_t)warp * Shape::warp_bytes(n_rad, NRAD_MAX);
    using YT = std::conditional_t<Shape::y_f64, double, T>;   // element type of the image of the harmonics
    constexpr int LY = Shape::y_pitch;
    YT* Ys = reinterpret_cast<YT*>(my);
    // ONE radial image: the next tile's values are requested right after this tile's contraction and
    // land while the next tile's harmonics are evaluated (a second image would cost a resident CTA)
    T* Rs = reinterpret_cast<T*>(my + Shape::y_bytes);
    T* Cs = reinterpret_cast<T*>(my + Shape::y_bytes + Shape::r_bytes(n_rad, NRAD_MAX));
    uint64_t* bar = reinterpret_cast<uint64_t*>(my + Shape::y_bytes + Shape::r_bytes(n_rad, NRAD_MAX) + Shape::c_bytes(n_rad));
    const int pl = lane & (TPB_PTS - 1);   // point inside the tile
    const bool sinb = lane >= TPB_PTS;     // branch
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    const T* __restrict__ radial = static_cast<const T*>(prm.radial);
    T* __restrict__ coeff = static_cast<T*>(prm.coeff);
    const int rstride = n_rad * (LMAX + 1);   // radial values per point
    // a tile's radial values are one contiguous range of global memory: where a point's share is a
    // multiple of 16 bytes the range is 16-byte aligned whatever its first point, and it arrives as ONE
    // bulk load (TMA) signalled on an mbarrier; otherwise element by element (cp.async)
    const bool r_bulk = (rstride * (int)sizeof(T)) % 16 == 0;
    // likewise a segment's coefficients leave as ONE bulk store from the staging image
    const bool c_bulk = (n_rad * L * (int)sizeof(T)) % 16 == 0;
    if (lane == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    uint32_t phase = 0u;   // parity of the mbarrier
    __syncwarp();

    using Tiles = ExpandTiles<LMAX>;
    constexpr int MT = NRAD_MAX / 8;   // M-tiles
    constexpr int NT = Tiles::total;   // N-tiles
    const int fr = lane >> 2, fk = lane & 3;   // fragment coordinates of this lane
    double acc[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int t = 0; t < NT; ++t) acc[mt][t][0] = acc[mt][t][1] = 0.0;

    auto zero_acc = [&]() {
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int t = 0; t < NT; ++t) acc[mt][t][0] = acc[mt][t][1] = 0.0;
    };
    // c[seg, n, lm] of segment j: lane holds C[n = fr + 8 mt][m-index 8 t + 2 fk + {0, 1}] of every tile
    auto flush = [&](int j) {
        const int64_t seg = seg0 + j;
        if (c_bulk) {
            if (lane == 0) bulk_wait_read<0>();   // the previous segment's store has read the staging image
            __syncwarp();
            static_for<0, LMAX + 1>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                constexpr int NTL = Tiles::of(l), T0 = Tiles::first(l);
                static_for<0, NTL>([&](auto tc) {
                    constexpr int t = decltype(tc)::value;
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        const int n = fr + 8 * mt;
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int jm = 8 * t + 2 * fk + e;
                            if (n < n_rad && jm < 2 * l + 1) Cs[n * L + l * l + jm] = static_cast<T>(acc[mt][T0 + t][e]);
                        }
                    }
                });
            });
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
                bulk_store(coeff + seg * n_rad * L, Cs, (uint32_t)(n_rad * L * (int)sizeof(T)));
                bulk_commit();
            }
            return;
        }
        static_for<0, LMAX + 1>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            constexpr int NTL = Tiles::of(l), T0 = Tiles::first(l);
            static_for<0, NTL>([&](auto tc) {
                constexpr int t = decltype(tc)::value;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int n = fr + 8 * mt;
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int jm = 8 * t + 2 * fk + e;
                        if (n < n_rad && jm < 2 * l + 1)
                            coeff[(seg * n_rad + n) * L + l * l + jm] = static_cast<T>(acc[mt][T0 + t][e]);
                    }
                }
            });
        });
    };
    // the tiles of this warp in order: (segment j, first point k0); advance() steps to the next one
    // (j == cnt: none left).  Empty segments are skipped here and zero-filled at the end.
    auto settle = [&](int& j, int64_t& k0) {
        while (j < cnt && k0 >= SP(j + 1)) {
            ++j;
            if (j < cnt) k0 = SP(j);
        }
    };
    // inputs of a tile: its radial values into the image (absent points' rows zeroed: they contribute
    // 0), its points into registers
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
    while (j < cnt) {
        const int np = (int)min((int64_t)TPB_PTS, SP(j + 1) - k0);
        const double x = static_cast<double>(xn), y = static_cast<double>(yn), z = static_cast<double>(zn);
        // the next tile (of this segment or of the warp's next non-empty one): its inputs are in
        // flight while this tile is evaluated and contracted
        int jn = j;
        int64_t kn = k0 + TPB_PTS;
        settle(jn, kn);
        if (jn < cnt) fetch_xyz(jn, kn, xn, yn, zn);   // in flight through this tile
        // ---- harmonics of the tile: two lanes per point ----------------------------------------
        R X, Y, Z;
        double rinv;
        RT::normalize(x, y, z, X, Y, Z, rinv);
        YT* S = Ys + pl * LY;
        double Qc[LMAX + 1];
        R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
        static_for<0, LMAX + 1>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            // column m of the folded Eq. 7 (r^2 = 1 on the unit sphere), as in kernel_tpb.cuh
            {
                R q = RT::make(TB.D_hi[m], TB.D_lo[m]), qp = RT::make(0.0, 0.0);
                static_for<m, LMAX + 1>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    Qc[l] = to_double(q);
                    if constexpr (l < LMAX) {
                        constexpr int t1 = SPH_TRI(l + 1, m);
                        const R a = RT::make(TB.A_hi[t1], TB.A_lo[t1]);
                        R qn;
                        if constexpr (l == m) qn = a * (Z * q);
                        else qn = rec_step(TB.A_hi[t1], TB.A_lo[t1], TB.B_hi[t1], TB.B_lo[t1], Z, q, qp);   // (dd.cuh)
                        qp = q;
                        q = qn;
                    }
                });
            }
            const double A = sinb ? to_double(s) : (m == 0 ? SPH_INV_SQRT2 : to_double(c));
            const bool emit = (m > 0) || !sinb;   // the sin branch has no m = 0 output
            static_for<m, LMAX + 1>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                constexpr int kc = l * (l + 1) + m, ks = l * (l + 1) - m;
                if (emit) S[sinb ? ks : kc] = static_cast<YT>(Qc[l] * A);   // Eq. 5
            });
            if constexpr (m < LMAX) {   // Eq. 9
                const R cn = X * c - Y * s;
                const R sn = X * s + Y * c;
                c = cn;
                s = sn;
            }
        });
        if (r_bulk) {   // this tile's radial image has landed (it was in flight through this evaluation)
            mbar_wait(bar, phase);
            phase ^= 1u;
        } else {
            cp_async_wait_all();
        }
        __syncwarp();
        // ---- contract over the tile's points, 4 at a time (K of the DMMA) --------------------------
        // What a fragment reads outside the valid ranges (n >= n_rad: the next point's radial values
        // or the padding; m beyond 2l+1: the next degree's harmonics) only reaches rows / columns of
        // C that are never stored.
#pragma unroll
        for (int ks = 0; ks < TPB_PTS / 4; ++ks) {
            if (4 * ks < np) {
                const int p = 4 * ks + fk;
                static_for<0, LMAX + 1>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    double a[MT];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) a[mt] = static_cast<double>(Rs[p * rstride + (fr + 8 * mt) * (LMAX + 1) + l]);
                    constexpr int NTL = Tiles::of(l), T0 = Tiles::first(l);
                    static_for<0, NTL>([&](auto tc) {
                        constexpr int t = decltype(tc)::value;
                        const double bv = static_cast<double>(Ys[p * LY + l * l + 8 * t + fr]);
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) dmma_m8n8k4(acc[mt][T0 + t], a[mt], bv);
                    });
                });
            }
        }
        __syncwarp();   // every lane is done with the radial image and the Y image
        if (jn < cnt) fetch_radial(jn, kn);   // lands while the next tile's harmonics are evaluated
        if (jn != j) {   // the segment is complete
            flush(j);
            zero_acc();
        }
        j = jn;
        k0 = kn;
    }
    if (c_bulk && lane == 0) bulk_wait_read<0>();   // shared memory must outlive the bulk stores' reads of it
    // empty segments: zeros
    for (int je = 0; je < cnt; ++je) {
        if (SP(je) == SP(je + 1))
            for (int i = lane; i < n_rad * L; i += 32) coeff[(seg0 + je) * n_rad * L + i] = T(0);
    }
}

}  // namespace sphb200
