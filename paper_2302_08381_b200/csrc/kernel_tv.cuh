// "tv" forward kernel: VALUES only, any l_max, run-time l_max; built for the cells where the values
// are bound by the recurrences themselves (f64 I/O: double-double, ~23 operations per Legendre entry
// for two outputs) and the two-phase kernel's second pass over a scratch costs more than it saves.
//
//   lane = (point of the batch, column class), as phase A of kernel_tq.cuh (batches of 32 / 16 / 8
//   points: 1 / 2 / 4 lanes per point), two columns of the folded Eq. 7 at a time per lane.
//   Every entry Qt_l^m goes STRAIGHT into the image as the two harmonics (l, +-m) = Qt c_m | Qt s_m
//   (Eq. 5): no scratch for the triangle, no second phase.
//   The powers (c_m, s_m) (Eq. 9) of batch i+1 are computed WHILE batch i's columns run: by
//   dedicated warps in segments for f64 I/O (double-double: ~50 operations per power, see
//   kernel_tq.cuh), on the side by one lane class for f32 I/O; two sets of them in shared memory.
//   Image: one row per point, rows a pitch apart that keeps lane = point stores conflict-free and
//   leaves each row 16 bytes of slack, so that it is staged at the offset its global address has
//   from a 16-byte boundary; every row leaves as one bulk store (TMA) issued by a thread of its own.
#pragma once
#include "kernel_tq.cuh"

namespace sphb200 {

struct TvParams {
    const void* xyz;
    void* sph;
    const double2* ab_hi;   // {A, B}[t] of the folded Eq. 7, high parts (tables.h)
    const double2* ab_lo;   // ... low parts
    int64_t n;
    int l_max;
    int batch;              // 32, 16 or 8 points
    int cs_warps;           // f64 I/O: warps that run Eq. 9 only
    int batches_per_cta;
};

struct TvSmem {
    int CP;                 // (c, s) pairs per point and set
    uint32_t pitch;         // bytes between the rows of the image
    bool contig;            // rows end to end (odd L)
    size_t cs_off, img_off, total;
    __host__ __device__ TvSmem(int l_max, int esize, int batch) {
        CP = (l_max + 1) | 1;   // odd pitch: conflict-free lane = point stores
        const uint32_t L = (uint32_t)(l_max + 1) * (l_max + 1);
        // row + 16 bytes of slack, rounded up to 16, then to an odd number of 16-byte units: lanes of
        // one class (consecutive points) then fall into different banks for 4- and 8-byte elements alike
        uint32_t units = (L * esize + 16 + 15) / 16;
        units |= 1;
        pitch = units * 16;
        // Odd L (even l_max): the rows are an odd number of elements long, so laid end to end -- the image
        // byte-identical to global memory -- lane = point stores are conflict-free as they are, no row needs
        // staging at an offset, and a whole batch leaves as ONE bulk store (a batch starts at a multiple of
        // 8 points: 16-byte aligned).  Even L keeps the padded rows above, each its own (aligned) bulk store.
        contig = (L & 1u) != 0;
        if (contig) pitch = L * esize;
        cs_off = 0;
        img_off = ((size_t)2 * batch * CP * 16 + 127) & ~(size_t)127;
        total = img_off + (size_t)batch * pitch;
    }
};

template <typename T, typename R, bool NORM>
__global__ void __launch_bounds__(TQ_MAX_WARPS * 32, 1) sph_tv_kernel(const TvParams prm) {
    using RT = rec<R>;
    constexpr int ES = (int)sizeof(T);
    constexpr bool DD = sizeof(R) > sizeof(double);
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const int l_max = prm.l_max, L = (l_max + 1) * (l_max + 1), B = prm.batch;
    const TvSmem lay(l_max, ES, B);
    const int CP = lay.CP;
    const uint32_t s0 = smem_u32(smem), sCS = s0 + (uint32_t)lay.cs_off, sIMG = s0 + (uint32_t)lay.img_off;
    const int64_t n = prm.n;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    const SphTables& TB = c_tables_tq;
    const uint64_t policy = policy_evict_first();
    const int pt_l = lane & (B - 1), cls = lane / B, NC = 32 / B;
    const int WC = DD ? prm.cs_warps : 0, Wq = W - WC;
    const bool cs_lane = DD ? warp >= Wq : (warp == W - 1 && cls == NC - 1);
    const bool col_lane = warp < Wq;
    const int V = Wq * NC, v = warp * NC + cls;
    const uint32_t row_b = (uint32_t)L * ES;

    // the point of this lane in batch b0 (lanes past the end: a harmless point)
    auto load_point = [&](int64_t b0, R& X, R& Y, R& Z, R& r2) {
        const int64_t p = b0 + pt_l;
        double x = 0.0, y = 0.0, z = 1.0;
        if (p < n) {
            x = static_cast<double>(__ldg(xyz + 3 * p + 0));
            y = static_cast<double>(__ldg(xyz + 3 * p + 1));
            z = static_cast<double>(__ldg(xyz + 3 * p + 2));
        }
        if (NORM) {
            double rinv;
            RT::normalize(x, y, z, X, Y, Z, rinv);
            r2 = RT::make(1.0, 0.0);
        } else {
            X = RT::make(x, 0.0), Y = RT::make(y, 0.0), Z = RT::make(z, 0.0);
            r2 = RT::r2_of(X, Y, Z);
        }
    };
    // Eq. 9 for batch b0 into set `set`: this lane's segment of the powers (kernel_tq.cuh, phase A)
    auto powers = [&](int64_t b0, int set) {
        if (b0 >= n) return;
        R X, Y, Z, r2;
        load_point(b0, X, Y, Z, r2);
        const int seg = DD ? (warp - Wq) * NC + cls : 0, nseg = DD ? WC * NC : 1;
        // segments of h = 2^sq powers, the largest power of two <= ceil((l_max + 1) / nseg); the last
        // segment takes what is left
        int h = 1, sq = 0;
        while (2 * h * nseg <= l_max + nseg) h <<= 1, ++sq;
        R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
        if (seg > 0) {
            R pr = X, pi = Y;
            for (int i = 0; i < sq; ++i) {
                const R prn = pr * pr - pi * pi;
                const R pin = (pr * pi) * 2.0;
                pr = prn, pi = pin;
            }
            c = pr, s = pi;
            for (int i = 1; i < seg; ++i) {
                const R cn = c * pr - s * pi;
                const R sn = c * pi + s * pr;
                c = cn, s = sn;
            }
        }
        const int m0 = seg * h, m1 = seg == nseg - 1 ? l_max + 1 : min(m0 + h, l_max + 1);
        uint32_t a = sCS + ((set * B + pt_l) * CP + m0) * 16;
        for (int m = m0; m < m1; ++m, a += 16) {
            // (the m = 0 slot holds the factor of Eq. 5 for m = 0, 1/sqrt2, instead of c_0 = 1)
            tq_sts2(a, m == 0 ? SPH_INV_SQRT2 : to_double(c), to_double(s));
            const R cn = X * c - Y * s;
            const R sn = X * s + Y * c;
            c = cn, s = sn;
        }
    };

    const int64_t b_first = (int64_t)blockIdx.x * prm.batches_per_cta * B;
    if (b_first >= n) return;
    if (cs_lane) powers(b_first, 0);
    __syncthreads();

    for (int bi = 0; bi < prm.batches_per_cta; ++bi) {
        const int64_t b0 = b_first + (int64_t)bi * B;
        if (b0 >= n) break;
        const int set = bi & 1;
        if (cs_lane && bi + 1 < prm.batches_per_cta) powers(b0 + B, set ^ 1);   // the next batch's, meanwhile
        if (col_lane) {
            R X, Y, Z, r2;
            load_point(b0, X, Y, Z, r2);
            // The previous batch's rows must have been read out of the image before anyone writes there again:
            // the threads that issued their bulk stores wait for that HERE, after this batch's points are
            // loaded and normalised (the stores' reads run under that work), and only the column warps meet at
            // a barrier of their own -- the warps that run Eq. 9 never touch the image and are not held up.
            if (bi > 0) {
                if ((int)threadIdx.x < B) bulk_wait_read<0>();
                named_bar_sync(1, Wq * 32);
            }
            // this point's row, staged at the offset its global address has from a 16-byte boundary
            const uint32_t shift = lay.contig ? 0u : (uint32_t)(((b0 + pt_l) & 15) * row_b) & 15u;
            const uint32_t row = sIMG + pt_l * lay.pitch + shift;
            const uint32_t cs_row = sCS + ((set * B + pt_l) * CP) * 16;
            // one entry of column m at row l: the harmonics (l, +m) and (l, -m); the sin one first, so that
            // for m = 0 (s_0 = 0, same slot) the cos store that follows overwrites it
            auto emit = [&](R q, double Ac, double As, uint32_t ac, uint32_t as) {
                const double Q = pair_value(q);   // (unnormalised pair from rec_step_u)
                tq_sts(as, static_cast<T>(Q * As));
                tq_sts(ac, static_cast<T>(Q * Ac));
            };
            // one step of the folded Eq. 7: Qt_l^m from (q, qp) = (Qt_{l-1}^m, Qt_{l-2}^m), t = TRI(l, m)
            auto next = [&](int t, const R& q, const R& qp) -> R {
                const double2 hi = __ldg(prm.ab_hi + t);
                double2 lo = make_double2(0.0, 0.0);
                if constexpr (DD) lo = __ldg(prm.ab_lo + t);
                const R w = NORM ? qp : r2 * qp;
                return rec_step_u(hi.x, lo.x, hi.y, lo.y, Z, q, w);   // (B_{m+1}^m = 0)
            };
            // Columns in ADJACENT pairs (2k, 2k+1): both chains of a pair run over (nearly) the same rows, so a
            // lane has two independent recurrences in flight for the whole of its loop, not only where a long
            // and a short column happen to overlap.  Pair k takes M - 2k row steps (M = l_max + 1); the pairs
            // are dealt to the V column classes in snake order (class v: k = v, 2V-1-v, 2V+v, ...), which
            // balances the classes' step counts where V <= ~M/4.  The row loop is unrolled by two with the
            // roles of (q, qp) exchanged, so that no register is copied from one step to the next.
            const int n_pairs = l_max / 2 + 1;
            for (int i = 0; i * V < n_pairs; ++i) {
                const int k = (i & 1) ? (i + 1) * V - 1 - v : i * V + v;
                if (k >= n_pairs) continue;
                const int ma = 2 * k, mb = ma + 1;
                const bool has_b = mb <= l_max;
                double Aca, Asa, Acb = 0.0, Asb = 0.0;
                tq_lds2(cs_row + ma * 16, Aca, Asa);
                if (has_b) tq_lds2(cs_row + mb * 16, Acb, Asb);
                R qa = RT::make(TB.D_hi[ma], TB.D_lo[ma]), qpa = RT::make(0.0, 0.0);
                // byte addresses of (l, +m) and (l, -m) in the row; from row l to l + 1 both move by 2 (l + 1) elements
                uint32_t aca = row + (uint32_t)(ma * (ma + 1) + ma) * ES, asa = row + (uint32_t)(ma * (ma + 1) - ma) * ES;
                emit(qa, Aca, Asa, aca, asa);
                if (!has_b) continue;
                // row l = mb: the second entry of column a, the first of column b
                int ta = SPH_TRI(ma, ma) + mb, tb = SPH_TRI(mb, mb);
                qpa = next(ta, qa, qpa);                           // (newest in qpa, the one before in qa)
                R qb = RT::make(TB.D_hi[mb], TB.D_lo[mb]), qpb = RT::make(0.0, 0.0);
                aca += 2u * mb * ES, asa += 2u * mb * ES;
                uint32_t acb = row + (uint32_t)(mb * (mb + 1) + mb) * ES, asb = row + (uint32_t)(mb * (mb + 1) - mb) * ES;
                emit(qpa, Aca, Asa, aca, asa);
                emit(qb, Acb, Asb, acb, asb);
                int l = mb + 1;
                if (l <= l_max) {   // one single step brings column a back to (newest in qa)
                    ta += l, tb += l;
                    qa = next(ta, qpa, qa);
                    qpb = next(tb, qb, qpb);                       // (column b: newest in qpb)
                    aca += 2u * l * ES, asa += 2u * l * ES, acb += 2u * l * ES, asb += 2u * l * ES;
                    emit(qa, Aca, Asa, aca, asa);
                    emit(qpb, Acb, Asb, acb, asb);
                    ++l;
                }
                for (; l + 1 <= l_max; l += 2) {   // a: newest in qa; b: newest in qpb
                    ta += l, tb += l;
                    qpa = next(ta, qa, qpa);
                    qb = next(tb, qpb, qb);
                    aca += 2u * l * ES, asa += 2u * l * ES, acb += 2u * l * ES, asb += 2u * l * ES;
                    emit(qpa, Aca, Asa, aca, asa);
                    emit(qb, Acb, Asb, acb, asb);
                    ta += l + 1, tb += l + 1;
                    qa = next(ta, qpa, qa);
                    qpb = next(tb, qb, qpb);
                    aca += 2u * (l + 1) * ES, asa += 2u * (l + 1) * ES, acb += 2u * (l + 1) * ES, asb += 2u * (l + 1) * ES;
                    emit(qa, Aca, Asa, aca, asa);
                    emit(qpb, Acb, Asb, acb, asb);
                }
                if (l <= l_max) {   // the last row of an odd count
                    ta += l, tb += l;
                    qpa = next(ta, qa, qpa);
                    qb = next(tb, qpb, qb);
                    aca += 2u * l * ES, asa += 2u * l * ES, acb += 2u * l * ES, asb += 2u * l * ES;
                    emit(qpa, Aca, Asa, aca, asa);
                    emit(qb, Acb, Asb, acb, asb);
                }
            }
        }
        fence_proxy_async_smem();
        __syncthreads();   // the image is complete; so are the next batch's powers
        if (lay.contig) {
            const int np = (int)min((int64_t)B, n - b0);
            const T* src = reinterpret_cast<const T*>(smem + lay.img_off);
            if (np == B) {   // (B x L x ES is a multiple of 16 bytes: B >= 8)
                if (threadIdx.x == 0) {
                    bulk_store_hint(sph + b0 * L, src, (uint32_t)B * row_b, policy);
                    bulk_commit();
                }
            } else {         // ragged last batch: plain stores (read before the next barrier: nothing left in flight)
                for (int i = threadIdx.x; i < np * L; i += blockDim.x) st_cs(sph + b0 * L + i, src[i]);
            }
        } else if (threadIdx.x < B) {
            const int64_t p = b0 + threadIdx.x;
            if (p < n) {
                const uint32_t d = (uint32_t)((p & 15) * row_b) & 15u;
                const T* src = reinterpret_cast<const T*>(smem + lay.img_off + threadIdx.x * lay.pitch + d);
                T* g = sph + p * L;
                uint32_t head = (16u - d) & 15u;
                if (head > row_b) head = row_b;
                const uint32_t body = (row_b - head) & ~15u;
                for (uint32_t i = 0; i < head / ES; ++i) st_cs(g + i, src[i]);
                if (body) bulk_store_hint(g + head / ES, src + head / ES, body, policy);
                for (uint32_t i = (head + body) / ES; i < row_b / ES; ++i) st_cs(g + i, src[i]);
                bulk_commit();
            }
        }
        // (the points parked in shared memory two batches ahead, so that no lane waits on global memory at the
        // top of a batch, were measured: 3 % slower -- other CTAs cover that latency already)
        // (two images, so that a batch drains while the next is computed, were measured: slower everywhere --
        // the shared memory they take costs more resident CTAs than the second barrier costs time)
    }
    // shared memory must outlive the bulk stores' reads of it
    if ((int)threadIdx.x < B) bulk_wait_read<0>();
}

}  // namespace sphb200
