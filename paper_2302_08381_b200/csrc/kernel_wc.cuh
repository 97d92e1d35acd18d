// "wc" forward kernel: the warps of a CTA work TOGETHER on one point at a time, so that a staged
// chunk is a third of a row (<= 368 harmonics) and every bulk store is ~3 KB.  Works for
// l_max >= 19 and any derivative order; used by default where it wins: f64 Hessians from l_max = 29
// and every f64 output set at l_max = 32 -- config C4.  (Measured, Hessians, 131 072-262 144 points: f64 l_max = 32 5.0 TB/s against 4.7 for the
// one-warp-per-point kernel -- 6.2 against 4.9 at C4's full size with rotating outputs -- but
// 4.4-4.9 against 4.7-5.1 at l_max 28-31, whose rows split less evenly into chunks and, for even L,
// are 128-byte aligned anyway; f32: 1.9-2.8 against 2.7-2.9 at every l_max.)
//
// Why (profiles/r1b_kernels.md): the one-warp-per-point kernel (kernel_w.cuh) can stage
// only ~128 harmonics of each of its 13 output rows, so a point leaves as 143 bulk stores of ~1 KB
// whose ends fall anywhere inside a 128-byte line (L = 1089 is odd).  That store pattern alone
// takes 5.9 ms on C4 (5.0 TB/s in a store-only probe); the same bytes in longer runs reach
// 5.5 TB/s (2 KB) to 6.4 TB/s (4.3 KB).  Runs that long need ~38 KB of staging per image: images
// belong to a group of warps, not to one warp.
//
//   A-warps (WC_AW of them): phase A of kernel_w.cuh (lane = m: c_m, s_m and column m of the
//       Legendre triangle, double-double for f64 I/O) for the CTA's points, round-robin, into a
//       ring of WC_SLOTS scratch slots in shared memory;
//   B-warps (WC_GROUPS groups of WC_GW): the chunks (a few whole l-rows each) of the CTA's points,
//       in order, go to the groups in turn.  A group assembles its chunk in ONE pass -- every
//       thread one (l, m >= 0) pair, both harmonics (l, +-m), all components (assemble_pair) --
//       into one of its two images, meets on its named barrier, and three of its warps issue the
//       1/4/13 bulk stores of the image's rows; the stores of one chunk drain while the group
//       assembles its next chunk into the other image, and the other group works meanwhile.
//   Slots are handed over with mbarriers (full: A -> B, empty: B -> A).
// The grid is not persistent: a CTA owns up to WC_PTS consecutive points.
// Measured on C4 (B200): 6.05 ms with kernel_w.cuh -> 4.88 ms (stores alone: 4.4 ms).
#pragma once
#include "kernel_w.cuh"

namespace sphb200 {

constexpr int WC_GROUPS = 2;    // groups of assembly warps, each with its own pair of images, on alternate chunks
constexpr int WC_GW = 6;        // warps per group: one pass covers 192 (l, m >= 0) pairs
constexpr int WC_BW = WC_GROUPS * WC_GW;
constexpr int WC_AW = 4;        // recurrence warps (phase A of a point takes ~4x one point's assembly)
constexpr int WC_SLOTS = 6;     // triangles in flight
constexpr int WC_CH = 368;      // most harmonics in a chunk: l_max = 32 splits into l < 19, 19 <= l < 27, l >= 27
                                // (361 / 368 / 360 harmonics, 190 / 188 / 183 pairs: one pass each)
constexpr int WC_PTS = 256;     // most points per CTA (the first point's phase A is not overlapped); fewer for
                                // small n, so that every SM gets several CTAs
constexpr int WC_THREADS = (WC_BW + WC_AW) * 32;

// Staging image: as WkStage (kernel_w.cuh), rows of one array a compile-time stride apart and
// congruent to their global addresses modulo 16 bytes, with room for WC_CH harmonics per row.
template <int ESIZE, int DERIV, bool LODD> struct WcStage {
    static constexpr int AL = 16 / ESIZE;
    static constexpr int RS = LODD ? ((WC_CH + AL) | 1) : wk_round_up(WC_CH + AL, AL);
    static constexpr int A1 = wk_round_up(RS + AL - 1, AL);              // after the 1 row of sph
    static constexpr int A2 = wk_round_up(A1 + 3 * RS + AL - 1, AL);     // after the 3 rows of dsph
    static constexpr int A3 = wk_round_up(A2 + 9 * RS + AL - 1, AL);     // after the 9 rows of ddsph
    static constexpr int elems = DERIV == 0 ? A1 : (DERIV == 1 ? A2 : A3);
    static constexpr int bytes = elems * ESIZE;
};
__host__ __device__ constexpr int wc_stage_bytes(int esize, int deriv, bool lodd) {
    return esize == 4 ? (deriv == 0 ? (lodd ? WcStage<4, 0, true>::bytes : WcStage<4, 0, false>::bytes)
                                    : deriv == 1 ? (lodd ? WcStage<4, 1, true>::bytes : WcStage<4, 1, false>::bytes)
                                                 : (lodd ? WcStage<4, 2, true>::bytes : WcStage<4, 2, false>::bytes))
                      : (deriv == 0 ? (lodd ? WcStage<8, 0, true>::bytes : WcStage<8, 0, false>::bytes)
                                    : deriv == 1 ? (lodd ? WcStage<8, 1, true>::bytes : WcStage<8, 1, false>::bytes)
                                                 : (lodd ? WcStage<8, 2, true>::bytes : WcStage<8, 2, false>::bytes));
}

// shared-memory carve-up (bytes), identical on host and device
struct WcSmem {
    int tsz, ntab;
    size_t tab_bytes, bar_bytes, slot_bytes, stage_bytes, total;
    __host__ __device__ WcSmem(int l_max, int deriv, int esize) {
        tsz = (l_max + 1) * (l_max + 2) / 2;
        ntab = 1 + (deriv == 0 ? 0 : (deriv == 1 ? 2 : 5));
        tab_bytes = ((size_t)ntab * tsz * 8 + 15) & ~(size_t)15;
        bar_bytes = ((size_t)2 * WC_SLOTS * 8 + 15) & ~(size_t)15;
        // per slot: Qt[tsz] + cs[2(l_max+1)] + {x, y, z, 1/r}, rounded to 16
        slot_bytes = ((size_t)(tsz + 2 * (l_max + 1) + 4) * 8 + 15) & ~(size_t)15;
        stage_bytes = (size_t)wc_stage_bytes(esize, deriv, (l_max & 1) == 0);
        total = tab_bytes + bar_bytes + WC_SLOTS * slot_bytes + 2 * WC_GROUPS * stage_bytes;
    }
};

struct WcParams {
    const void* xyz;
    void* sph;
    void* dsph;
    void* ddsph;
    const SphTables* tab;   // global-memory copy of the tables
    int64_t n;
    int l_max;
    int n_chunks;
    int pts_per_cta;
    unsigned char row0[SPH_MAX_L + 3];   // chunk i = the l-rows [row0[i], row0[i+1])
};

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <typename T, typename R, int DERIV, bool NORM, bool LODD>
__global__ void __launch_bounds__(WC_THREADS, 1) sph_wc_kernel(const WcParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int ROWS = wk_rows<DERIV>::n;
    constexpr int ES = (int)sizeof(T);
    using Stage = WcStage<ES, DERIV, LODD>;
    constexpr int AL = Stage::AL;
    constexpr int RS = Stage::RS;
    using RT = rec<R>;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const WcSmem lay(l_max, DERIV, ES);

    // ---- coefficient tables -> shared memory, barriers, scratch (once per CTA) ----------------
    double* tabs = reinterpret_cast<double*>(smem);
    {
        const double* src[6] = {prm.tab->Np, prm.tab->G1, prm.tab->Gz, prm.tab->H2, prm.tab->Hxz, prm.tab->Hzz};
        for (int t = 0; t < lay.ntab; ++t)
            for (int i = threadIdx.x; i < lay.tsz; i += blockDim.x) tabs[t * lay.tsz + i] = src[t][i];
    }
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + lay.tab_bytes);   // full[s]: slot s holds a triangle
    uint64_t* empty = full + WC_SLOTS;                                     // empty[s]: every B-warp is done with it
    unsigned char* slots = smem + lay.tab_bytes + lay.bar_bytes;
    unsigned char* stage = slots + WC_SLOTS * lay.slot_bytes;
    // neighbour reads of assemble_pair may touch the padding behind cs (times a zero coefficient):
    // it only has to be finite
    for (int i = threadIdx.x; i < (int)(WC_SLOTS * lay.slot_bytes / 8); i += blockDim.x)
        reinterpret_cast<double*>(slots)[i] = 0.0;
    if (threadIdx.x == 0) {
        for (int s = 0; s < WC_SLOTS; ++s) {
            mbar_init(&full[s], 32);            // every lane of the A-warp arrives
            mbar_init(&empty[s], WC_BW * 32);   // every B-thread arrives
        }
        fence_mbar_init();
    }
    __syncthreads();
    const double* Np = tabs;
    WkTabView tv;
    tv.G1 = tabs + 1 * lay.tsz;
    tv.Gz = tabs + 2 * lay.tsz;
    tv.H2 = tabs + 3 * lay.tsz;   // only dereferenced when DERIV == 2
    tv.Hxz = tabs + 4 * lay.tsz;
    tv.Hzz = tabs + 5 * lay.tsz;

    const int64_t pt_begin = (int64_t)blockIdx.x * prm.pts_per_cta;
    const int np = (int)((prm.n - pt_begin < prm.pts_per_cta) ? prm.n - pt_begin : prm.pts_per_cta);

    if (warp >= WC_BW) {
        // ================= A-warps: recurrences, lane = m (phase A of kernel_w.cuh) =================
        const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
        int nbits = 0;
        while ((1 << nbits) <= (l_max < 31 ? l_max : 31)) ++nbits;
        for (int i = warp - WC_BW; i < np; i += WC_AW) {
            const int s = i % WC_SLOTS, round = i / WC_SLOTS;
            const int64_t pt = pt_begin + i;
            const double x = static_cast<double>(xyz[3 * pt + 0]);
            const double y = static_cast<double>(xyz[3 * pt + 1]);
            const double z = static_cast<double>(xyz[3 * pt + 2]);
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
            double* Qt = reinterpret_cast<double*>(slots + (size_t)s * lay.slot_bytes);
            double* cs = Qt + lay.tsz;
            double* pv = cs + 2 * (l_max + 1);   // {x, y, z, 1/r} the assembly evaluates at
            // the B-warps must have released the slot's previous triangle
            if (round > 0) mbar_wait(&empty[s], (uint32_t)((round - 1) & 1));
            const int m = lane;
            R c, sn;
            cs_power<R>(m, X, Y, nbits, c, sn);
            if (m <= l_max) {
                cs[2 * m] = to_double(c);
                cs[2 * m + 1] = to_double(sn);
            }
            if (l_max == 32 && lane == 31) {  // the 33rd column: (c,s)_32 and Qt_32^32 = Np_32^32 * 1
                const R c32 = X * c - Y * sn;
                const R s32 = X * sn + Y * c;
                cs[64] = to_double(c32);
                cs[65] = to_double(s32);
                Qt[SPH_TRI(32, 32)] = Np[SPH_TRI(32, 32)];
            }
            if (lane == 0) {
                pv[0] = to_double(X);
                pv[1] = to_double(Y);
                pv[2] = to_double(Z);
                pv[3] = rinv;
            }
            R w = RT::make(0.0, 0.0), wp = RT::make(0.0, 0.0);
            for (int l = 0; l <= l_max; ++l) {
                const R wn = column_step_int<R, NORM>(l, m, Z, r2, w, wp);
                wp = w;
                w = wn;
                if (m <= l) Qt[SPH_TRI(l, m)] = to_double(w) * Np[SPH_TRI(l, m)];
            }
            mbar_arrive(&full[s]);
        }
        return;
    }

    // ================= B-warps: assembly and stores =============================================
    T* __restrict__ out_base[3] = {static_cast<T*>(prm.sph), static_cast<T*>(prm.dsph), static_cast<T*>(prm.ddsph)};
    const uint64_t policy = policy_evict_first();
    constexpr int BT = WC_GW * 32;            // threads of one group
    const int grp = warp / WC_GW;              // this warp's group
    const int gw = warp - grp * WC_GW;         // warp inside the group
    const int bt = gw * 32 + lane;             // 0 .. BT-1
    unsigned char* gstage = stage + (size_t)grp * 2 * Stage::bytes;   // the group's two images
    int hs = 0;                   // chunks this group has assembled: image hs & 1 is the one to fill
    int q = 0;                    // chunks of the CTA so far: chunk q belongs to group q % WC_GROUPS
    // the image's rows are stored by WC_IW warps of the group, row j by lane j / WC_IW of warp j % WC_IW
    // (the compiler serialises the bulk stores of a warp's lanes: ~12 instructions each)
    constexpr int WC_IW = 3;
    const int my_row = gw + WC_IW * lane;
    const bool issuer = gw < WC_IW && my_row < ROWS;
    for (int i = 0; i < np; ++i) {
        const int s = i % WC_SLOTS, round = i / WC_SLOTS;
        const int64_t pt = pt_begin + i;
        const double* Qt = reinterpret_cast<const double*>(slots + (size_t)s * lay.slot_bytes);
        const double* cs = Qt + lay.tsz;
        const double* pv = cs + 2 * (l_max + 1);
        mbar_wait(&full[s], (uint32_t)(round & 1));
        const double xd = pv[0], yd = pv[1], zd = pv[2], rinv = pv[3];
        const uint32_t ptl = (uint32_t)pt;   // low 32 bits are enough modulo AL
        for (int ci = 0; ci < prm.n_chunks; ++ci, ++q) {
            if (q % WC_GROUPS != grp) continue;
            const int l0 = prm.row0[ci], l1 = prm.row0[ci + 1];   // rows [l0, l1)
            const int k0 = l0 * l0;
            const int cnt = l1 * l1 - k0;
            const int tA = SPH_TRI(l0, 0), tB = SPH_TRI(l1, 0);   // this chunk's part of the triangle
            const int buf = hs & 1;
            // d_a = e(a, 0) mod AL, and the 32-bit shared address of row 0 of each array
            const uint32_t d0 = (ptl * (uint32_t)L + (uint32_t)k0) & (AL - 1);
            const uint32_t d1 = (ptl * 3u * (uint32_t)L + (uint32_t)k0) & (AL - 1);
            const uint32_t d2 = (ptl * 9u * (uint32_t)L + (uint32_t)k0) & (AL - 1);
            const uint32_t img_s = smem_u32(gstage) + (uint32_t)buf * Stage::bytes;
            const uint32_t b0 = img_s + d0 * ES;
            const uint32_t b1 = img_s + (Stage::A1 + d1) * ES;
            const uint32_t b2 = img_s + (Stage::A2 + d2) * ES;
            auto put = [&](int k, const double* o) {
                const uint32_t ib = (uint32_t)k * ES;
                sts_off<0>(b0 + ib, static_cast<T>(o[0]));
                if constexpr (DERIV >= 1) {
                    const uint32_t a1 = b1 + ib;
                    sts_off<0 * RS * ES>(a1, static_cast<T>(o[1]));
                    sts_off<1 * RS * ES>(a1, static_cast<T>(o[2]));
                    sts_off<2 * RS * ES>(a1, static_cast<T>(o[3]));
                }
                if constexpr (DERIV >= 2) {
                    // o[4..9] = xx xy xz yy yz zz ; rows = xx xy xz yx yy yz zx zy zz
                    const uint32_t a2 = b2 + ib;
                    sts_off<0 * RS * ES>(a2, static_cast<T>(o[4]));
                    sts_off<1 * RS * ES>(a2, static_cast<T>(o[5]));
                    sts_off<2 * RS * ES>(a2, static_cast<T>(o[6]));
                    sts_off<3 * RS * ES>(a2, static_cast<T>(o[5]));
                    sts_off<4 * RS * ES>(a2, static_cast<T>(o[7]));
                    sts_off<5 * RS * ES>(a2, static_cast<T>(o[8]));
                    sts_off<6 * RS * ES>(a2, static_cast<T>(o[6]));
                    sts_off<7 * RS * ES>(a2, static_cast<T>(o[8]));
                    sts_off<8 * RS * ES>(a2, static_cast<T>(o[9]));
                }
            };
            for (int t = tA + bt; t < tB; t += BT) {
                // (l, m) of triangle index t
                int l = (int)((sqrtf((float)(8 * t + 1)) - 1.0f) * 0.5f);
                l += (SPH_TRI(l + 1, 0) <= t);
                l -= (SPH_TRI(l, 0) > t);
                const int m = t - SPH_TRI(l, 0);
                double oc[10], os[10];
                assemble_pair<DERIV, NORM>(l, m, t, Qt, cs, xd, yd, zd, rinv, tv, oc, os);
                const int ic = l * (l + 1) + m - k0;   // (l, +m) inside the chunk; (l, -m) sits 2m before it
                put(ic, oc);
                if (m > 0) put(ic - 2 * m, os);
            }
            fence_proxy_async_smem();
            // One barrier per chunk: it says "this image is complete" and, because the storing lanes
            // first wait until their previous stores (the OTHER image's) have been read out, also
            // "the other image is free" for the chunk after this one.
            if (issuer) bulk_wait_read<0>();
            named_bar_sync(1 + grp, BT);
            ++hs;

            if (issuer) {
                const int j = my_row;
                // which array, which row inside the point
                const int arr = (j == 0) ? 0 : (j < 4 ? 1 : 2);
                const int rows_in_arr = (arr == 0) ? 1 : (arr == 1 ? 3 : 9);
                const int jj = (arr == 0) ? 0 : (arr == 1 ? j - 1 : j - 4);
                const int64_t e = (pt * rows_in_arr + jj) * (int64_t)L + k0;  // first element of the run
                T* g = (arr == 0 ? out_base[0] : (arr == 1 ? out_base[1] : out_base[2])) + e;
                const uint32_t sg = (uint32_t)e & (AL - 1);
                // where the run was staged: A_a + d_a + jj RS; by construction this is sg modulo AL
                const uint32_t da = (arr == 0) ? d0 : (arr == 1 ? d1 : d2);
                const int aoff = (arr == 0) ? 0 : (arr == 1 ? Stage::A1 : Stage::A2);
                const T* srow = reinterpret_cast<const T*>(gstage + (size_t)buf * Stage::bytes) + aoff + da + jj * RS;
                int head = (int)((AL - sg) & (AL - 1));   // elements before the first 16-byte boundary
                if (head > cnt) head = cnt;
                const int body = (cnt - head) & ~(AL - 1);
                for (int q = 0; q < head; ++q) st_cs(g + q, srow[q]);
                if (body > 0) bulk_store_hint(g + head, srow + head, (uint32_t)body * sizeof(T), policy);
                for (int q = head + body; q < cnt; ++q) st_cs(g + q, srow[q]);
                bulk_commit();
            }
        }
        // this thread is done reading slot s
        mbar_arrive(&empty[s]);
    }
    if (issuer) bulk_wait_read<0>();   // shared memory must outlive the bulk stores' reads of it
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef void (*WcKernel)(const WcParams);

struct WcLaunch {
    const void* func;
    WcKernel kern;
    WcParams prm;
    int64_t grid;
    size_t smem;
};

template <typename T, typename R, bool LODD> static WcKernel wc_pick2(int deriv, int norm) {
    if (deriv == 0) return norm ? sph_wc_kernel<T, R, 0, true, LODD> : sph_wc_kernel<T, R, 0, false, LODD>;
    if (deriv == 1) return norm ? sph_wc_kernel<T, R, 1, true, LODD> : sph_wc_kernel<T, R, 1, false, LODD>;
    return norm ? sph_wc_kernel<T, R, 2, true, LODD> : sph_wc_kernel<T, R, 2, false, LODD>;
}
template <typename T, typename R> static WcKernel wc_pick(int deriv, int norm, bool lodd) {
    return lodd ? wc_pick2<T, R, true>(deriv, norm) : wc_pick2<T, R, false>(deriv, norm);
}

// returns 0 and fills *out if the cooperative kernel applies (rows long enough to be worth it and
// the carve-up fits), 1 otherwise
static inline int wc_plan(int min_l, int sm_count, int smem_optin, int64_t n, int l_max, int normalized, int dtype, void* sph, void* dsph,
                          void* ddsph, const void* xyz, const SphTables* d_tab, WcLaunch* out) {
    const int deriv = ddsph ? 2 : (dsph ? 1 : 0);
    const int esize = dtype == 0 ? 4 : 8;
    if (l_max < min_l) return 1;
    const WcSmem lay(l_max, deriv, esize);
    if ((int64_t)lay.total > smem_optin) return 1;
    const bool lodd = (l_max & 1) == 0;
    out->kern = dtype == 0 ? wc_pick<float, double>(deriv, normalized, lodd) : wc_pick<double, dd>(deriv, normalized, lodd);
    out->func = (const void*)out->kern;
    out->prm.xyz = xyz;
    out->prm.sph = sph;
    out->prm.dsph = dsph;
    out->prm.ddsph = ddsph;
    out->prm.tab = d_tab;
    out->prm.n = n;
    out->prm.l_max = l_max;
    // chunks of whole l-rows, at most WC_CH harmonics each: fewest passes of the B-warps over the
    // pairs, then fewest chunks (dynamic programming over the row where a chunk ends)
    int best[SPH_MAX_L + 2], from[SPH_MAX_L + 2];
    best[0] = 0;
    for (int e = 1; e <= l_max + 1; ++e) {   // rows [0, e) covered
        best[e] = 1 << 30;
        for (int b = e - 1; b >= 0 && e * e - b * b <= WC_CH; --b) {
            const int pairs = e * (e + 1) / 2 - b * (b + 1) / 2;
            const int c = best[b] + (pairs + WC_GW * 32 - 1) / (WC_GW * 32) * 1000 + 300;
            if (c < best[e]) best[e] = c, from[e] = b;
        }
    }
    int nc = 0;
    for (int e = l_max + 1; e > 0; e = from[e]) ++nc;
    out->prm.row0[nc] = (unsigned char)(l_max + 1);
    for (int e = l_max + 1, i = nc; e > 0; e = from[e]) out->prm.row0[--i] = (unsigned char)from[e];
    out->prm.n_chunks = nc;
    // One CTA per SM is resident: the grid is sized in WHOLE waves -- k = the fewest that keep a CTA at
    // <= WC_PTS points, at least 4 where n allows -- and the points dealt evenly over k * sm_count CTAs.
    // (n / (4 SMs) points per CTA, capped, left a last wave of a few CTAs at some sizes: n = 131 072 ran
    // 594 CTAs = 4 waves + 2 CTAs, 3.7-4.9 TB/s where 37 888 and 262 144 points reached 4.3-6.0.)
    int64_t waves = (n + (int64_t)WC_PTS * sm_count - 1) / ((int64_t)WC_PTS * sm_count);
    if (waves < 4) waves = 4;
    int64_t ppc = (n + waves * sm_count - 1) / (waves * sm_count);
    if (ppc < 16) ppc = 16;
    out->prm.pts_per_cta = (int)ppc;
    out->grid = (n + ppc - 1) / ppc;
    if (out->grid > 0x7fffffff) return 1;
    out->smem = lay.total;
    return 0;
}

static inline void wc_launch(const WcLaunch& lw, cudaStream_t stream) {
    lw.kern<<<(unsigned)lw.grid, WC_THREADS, lw.smem, stream>>>(lw.prm);
}

}  // namespace sphb200
