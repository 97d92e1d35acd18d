// "w" forward kernel: one WARP per point.  Any l_max <= 32, values / +gradients / +Hessians.
//
// Used when a point's outputs are too large for the thread-per-point kernel (config C4:
// 13 * 1089 * 8 B = 113 KB per point) or its row length is even.  Per point the warp runs
//   phase A  lane = m: c_m, s_m by square-and-multiply and column m of the Legendre triangle by the
//            integer-coefficient form of Eq. 7 (tables.h), all lanes stepping l together; the
//            triangle Qt and (c,s) go to a per-warp scratch in shared memory as f64;
//   phase B  a chunk = a few whole l-rows (<= CH harmonics); lane = one (l, m >= 0) of the chunk's
//            part of the triangle: it assembles ALL components (Y, 3 gradient, 6 unique Hessian) of
//            BOTH harmonics (l, +m) and (l, -m) from the scratch (assemble_pair: the Legendre side
//            of Eq. 10 is shared by the two) and writes them into per-component staging rows;
//   store    each of the 1/4/13 global rows of the chunk is a contiguous run of elements; lane j
//            issues row j as one 1-D TMA bulk store.  A run starts at element (n*rows+j)*L + k0,
//            which is 16-byte aligned only up to an element offset; the staging image (WkStage)
//            places every run so that shared and global addresses agree mod 16, the aligned body
//            goes out by TMA and at most AL-1 elements at either end by plain stores.
#pragma once
#include <atomic>

#include "options.h"
#include "ptx.cuh"
#include "sph_core.cuh"

namespace sphb200 {

struct WkParams {
    const void* xyz;
    void* sph;
    void* dsph;
    void* ddsph;
    const SphTables* tab;   // global-memory copy of the tables
    int64_t n;
    int l_max;
    int warps_per_cta;
    int nbuf;               // staging images per warp
    int pts_per_warp;       // consecutive rounds of warps_per_cta points one CTA works through
    int n_chunks;
    unsigned char row0[SPH_MAX_L + 3];   // chunk i = the l-rows [row0[i], row0[i+1])
};

struct WkTabView {  // phase-B coefficient tables, copied to shared memory once per CTA
    const double *G1, *Gz, *H2, *Hxz, *Hzz;
};

constexpr int WK_MAX_THREADS = 384;
constexpr int WK_CH = 128;   // most harmonics in a chunk (whole l-rows; the row l = 32 has 65)

template <int DERIV> struct wk_rows {  // global rows per point / staging rows
    static constexpr int n = DERIV == 0 ? 1 : (DERIV == 1 ? 4 : 13);
};

// Staging image of one chunk: one row per output component, laid out so that EVERY row's
// shared-memory address agrees with its global address modulo 16 bytes (what a bulk store needs)
// while the rows of one array sit a COMPILE-TIME stride apart:
//   row jj of array a (a = 0 sph, 1 dsph, 2 ddsph) starts at global element
//       e(a, jj) = (pt rows_a + jj) L + k0,            so  e(a, jj) = e(a, 0) + jj L;
//   it is staged at element  A_a + d_a + jj RS  with  d_a = e(a, 0) mod AL  (AL = elements per
//   16 bytes) and a row stride RS = L (mod AL): RS = CH + 1 for odd L (odd squares are 1 mod 8),
//   RS = CH + AL for even L (even squares are 0 mod 4).
// One base register per array then addresses all of its rows with immediate offsets.
__host__ __device__ constexpr int wk_round_up(int v, int a) { return (v + a - 1) / a * a; }
template <int ESIZE, int DERIV, bool LODD> struct WkStage {
    static constexpr int AL = 16 / ESIZE;
    static constexpr int RS = LODD ? WK_CH + 1 : WK_CH + AL;
    static constexpr int A1 = wk_round_up(RS + AL - 1, AL);              // after the 1 row of sph
    static constexpr int A2 = wk_round_up(A1 + 3 * RS + AL - 1, AL);     // after the 3 rows of dsph
    static constexpr int A3 = wk_round_up(A2 + 9 * RS + AL - 1, AL);     // after the 9 rows of ddsph
    static constexpr int elems = DERIV == 0 ? A1 : (DERIV == 1 ? A2 : A3);
    static constexpr int bytes = elems * ESIZE;
};
__host__ __device__ constexpr int wk_stage_bytes(int esize, int deriv, bool lodd) {
    return esize == 4 ? (deriv == 0 ? (lodd ? WkStage<4, 0, true>::bytes : WkStage<4, 0, false>::bytes)
                                    : deriv == 1 ? (lodd ? WkStage<4, 1, true>::bytes : WkStage<4, 1, false>::bytes)
                                                 : (lodd ? WkStage<4, 2, true>::bytes : WkStage<4, 2, false>::bytes))
                      : (deriv == 0 ? (lodd ? WkStage<8, 0, true>::bytes : WkStage<8, 0, false>::bytes)
                                    : deriv == 1 ? (lodd ? WkStage<8, 1, true>::bytes : WkStage<8, 1, false>::bytes)
                                                 : (lodd ? WkStage<8, 2, true>::bytes : WkStage<8, 2, false>::bytes));
}

// shared-memory carve-up (bytes), identical on host and device
struct WkSmem {
    int tsz;            // (l_max+1)(l_max+2)/2
    int ntab;           // coefficient tables kept in smem: Np + {0,2,5}
    size_t tab_bytes;
    size_t scratch_bytes;   // per warp: Qt[tsz] + cs[2(l_max+1)], rounded to 16
    size_t stage_bytes;     // per warp: nbuf staging images
    size_t warp_bytes;
    __host__ __device__ WkSmem(int l_max, int deriv, int esize, int nbuf) {
        tsz = (l_max + 1) * (l_max + 2) / 2;
        ntab = 1 + (deriv == 0 ? 0 : (deriv == 1 ? 2 : 5));
        tab_bytes = ((size_t)ntab * tsz * 8 + 15) & ~(size_t)15;
        scratch_bytes = ((size_t)(tsz + 2 * (l_max + 1)) * 8 + 15) & ~(size_t)15;
        stage_bytes = (size_t)nbuf * wk_stage_bytes(esize, deriv, (l_max & 1) == 0);
        warp_bytes = scratch_bytes + stage_bytes;
    }
};

// shared-memory stores through 32-bit shared addresses with an immediate byte offset
template <int OFF> __device__ __forceinline__ void sts_off(uint32_t addr, float v) {
    asm volatile("st.shared.f32 [%0+%2], %1;" ::"r"(addr), "f"(v), "n"(OFF) : "memory");
}
template <int OFF> __device__ __forceinline__ void sts_off(uint32_t addr, double v) {
    asm volatile("st.shared.f64 [%0+%2], %1;" ::"r"(addr), "d"(v), "n"(OFF) : "memory");
}

template <typename T, typename R, int DERIV, bool NORM, bool LODD>
__global__ void __launch_bounds__(WK_MAX_THREADS, 1) sph_w_kernel(const WkParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int ROWS = wk_rows<DERIV>::n;
    constexpr int ES = (int)sizeof(T);
    using Stage = WkStage<ES, DERIV, LODD>;
    constexpr int AL = Stage::AL;
    constexpr int RS = Stage::RS;
    using RT = rec<R>;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const WkSmem lay(l_max, DERIV, ES, prm.nbuf);

    // ---- coefficient tables -> shared memory (once per CTA) -----------------------------------
    double* tabs = reinterpret_cast<double*>(smem);
    {
        const double* src[6] = {prm.tab->Np, prm.tab->G1, prm.tab->Gz, prm.tab->H2, prm.tab->Hxz, prm.tab->Hzz};
        for (int t = 0; t < lay.ntab; ++t)
            for (int i = threadIdx.x; i < lay.tsz; i += blockDim.x) tabs[t * lay.tsz + i] = src[t][i];
    }
    __syncthreads();
    const double* Np = tabs;
    WkTabView tv;
    tv.G1 = tabs + 1 * lay.tsz;
    tv.Gz = tabs + 2 * lay.tsz;
    tv.H2 = tabs + 3 * lay.tsz;   // only dereferenced when DERIV == 2
    tv.Hxz = tabs + 4 * lay.tsz;
    tv.Hzz = tabs + 5 * lay.tsz;

    unsigned char* my = smem + lay.tab_bytes + (size_t)warp * lay.warp_bytes;
    double* Qt = reinterpret_cast<double*>(my);
    double* cs = Qt + lay.tsz;
    unsigned char* stage = my + lay.scratch_bytes;
    const uint32_t stage_s = smem_u32(stage);
    // neighbour reads of assemble_pair may touch the padding behind cs (times a zero coefficient):
    // it only has to be finite
    for (int i = lane; i < (int)(lay.scratch_bytes / 8); i += 32) Qt[i] = 0.0;
    __syncwarp();

    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ out_base[3] = {static_cast<T*>(prm.sph), static_cast<T*>(prm.dsph), static_cast<T*>(prm.ddsph)};
    const uint64_t policy = policy_evict_first();

    int nbits = 0;
    while ((1 << nbits) <= (l_max < 31 ? l_max : 31)) ++nbits;

    // NOT persistent: CTA b owns the points [b W P, (b+1) W P) (W warps, P points per warp) and the
    // grid has many more CTAs than the machine holds, so the block scheduler balances SMs that
    // drain their stores at different rates (kernel_tpb.cuh has the measurement).
    const int64_t pt_begin = (int64_t)blockIdx.x * prm.warps_per_cta * prm.pts_per_warp;
    int64_t pt_end = pt_begin + (int64_t)prm.warps_per_cta * prm.pts_per_warp;
    if (pt_end > prm.n) pt_end = prm.n;
    int buf = 0;
    for (int64_t pt = pt_begin + warp; pt < pt_end; pt += prm.warps_per_cta) {
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
        const double xd = to_double(X), yd = to_double(Y), zd = to_double(Z);

        // ---- phase A: lane = m ---------------------------------------------------------------
        __syncwarp();  // the previous point's phase B has finished reading the scratch
        {
            const int m = lane;
            R c, s;
            cs_power<R>(m, X, Y, nbits, c, s);
            if (m <= l_max) {
                cs[2 * m] = to_double(c);
                cs[2 * m + 1] = to_double(s);
            }
            if (l_max == 32 && lane == 31) {  // the 33rd column: (c,s)_32 and Qt_32^32 = Np_32^32 * 1
                const R c32 = X * c - Y * s;
                const R s32 = X * s + Y * c;
                cs[64] = to_double(c32);
                cs[65] = to_double(s32);
                Qt[SPH_TRI(32, 32)] = Np[SPH_TRI(32, 32)];
            }
            R w = RT::make(0.0, 0.0), wp = RT::make(0.0, 0.0);
            for (int l = 0; l <= l_max; ++l) {
                const R wn = column_step_int<R, NORM>(l, m, Z, r2, w, wp);
                wp = w;
                w = wn;
                if (m <= l) Qt[SPH_TRI(l, m)] = to_double(w) * Np[SPH_TRI(l, m)];
            }
        }
        __syncwarp();

        // ---- phase B + store: chunks of whole l-rows ---------------------------------------------
        const uint32_t ptl = (uint32_t)pt;   // low 32 bits are enough modulo AL
        for (int ci = 0; ci < prm.n_chunks; ++ci) {
            const int l0 = prm.row0[ci], l1 = prm.row0[ci + 1];   // rows [l0, l1)
            const int k0 = l0 * l0;
            const int cnt = l1 * l1 - k0;
            const int tA = SPH_TRI(l0, 0), tB = SPH_TRI(l1, 0);   // this chunk's part of the triangle
            // the staging image we are about to fill must have been drained
            if (prm.nbuf == 1) bulk_wait_read<0>();
            else bulk_wait_read<1>();
            __syncwarp();
            // d_a = e(a, 0) mod AL, and the 32-bit shared address of row 0 of each array
            const uint32_t d0 = (ptl * (uint32_t)L + (uint32_t)k0) & (AL - 1);
            const uint32_t d1 = (ptl * 3u * (uint32_t)L + (uint32_t)k0) & (AL - 1);
            const uint32_t d2 = (ptl * 9u * (uint32_t)L + (uint32_t)k0) & (AL - 1);
            const uint32_t img_s = stage_s + (uint32_t)buf * Stage::bytes;
            const uint32_t b0 = img_s + d0 * ES;
            const uint32_t b1 = img_s + (Stage::A1 + d1) * ES;
            const uint32_t b2 = img_s + (Stage::A2 + d2) * ES;
            auto put = [&](int i, const double* o) {
                const uint32_t ib = (uint32_t)i * ES;
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

            auto lm_of = [](int t, int& l, int& m) {   // (l, m) of triangle index t
                l = (int)((sqrtf((float)(8 * t + 1)) - 1.0f) * 0.5f);
                l += (SPH_TRI(l + 1, 0) <= t);
                l -= (SPH_TRI(l, 0) > t);
                m = t - SPH_TRI(l, 0);
            };
            for (int t = tA + lane; t < tB; t += 32) {
                int l, m;
                lm_of(t, l, m);
                double oc[10], os[10];
                assemble_pair<DERIV, NORM>(l, m, t, Qt, cs, xd, yd, zd, rinv, tv, oc, os);
                const int ic = l * (l + 1) + m - k0;   // (l, +m) inside the chunk; (l, -m) sits 2m before it
                put(ic, oc);
                if (m > 0) put(ic - 2 * m, os);
            }
            fence_proxy_async_smem();
            __syncwarp();

            if (lane < ROWS) {
                const int j = lane;
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
                const T* srow = reinterpret_cast<const T*>(stage + (size_t)buf * Stage::bytes) + aoff + da + jj * RS;
                int head = (int)((AL - sg) & (AL - 1));   // elements before the first 16-byte boundary
                if (head > cnt) head = cnt;
                const int body = (cnt - head) & ~(AL - 1);
                for (int i = 0; i < head; ++i) st_cs(g + i, srow[i]);
                if (body > 0) bulk_store_hint(g + head, srow + head, (uint32_t)body * sizeof(T), policy);
                for (int i = head + body; i < cnt; ++i) st_cs(g + i, srow[i]);
                bulk_commit();
            }
            buf = (buf + 1 == prm.nbuf) ? 0 : buf + 1;
        }
    }
    bulk_wait_read<0>();   // shared memory must outlive the bulk stores' reads of it
}

// ---------------------------------------------------------------------------------------------
// generic VJP for rows too long to stage 32 points: one warp per point, lanes stride over k
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) sph_vjp_warp_kernel(const T* __restrict__ dsph, const T* __restrict__ gsph,
                                                           T* __restrict__ gxyz, int64_t n, int L) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    for (int64_t p = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); p < n; p += warps) {
        const T* g = gsph + p * L;
        const T* d = dsph + p * 3 * L;
        double ax = 0.0, ay = 0.0, az = 0.0;
        for (int k = lane; k < L; k += 32) {
            const double w = static_cast<double>(__ldcs(g + k));
            ax = fma(static_cast<double>(__ldcs(d + k)), w, ax);
            ay = fma(static_cast<double>(__ldcs(d + L + k)), w, ay);
            az = fma(static_cast<double>(__ldcs(d + 2 * L + k)), w, az);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            ax += __shfl_xor_sync(0xffffffffu, ax, o);
            ay += __shfl_xor_sync(0xffffffffu, ay, o);
            az += __shfl_xor_sync(0xffffffffu, az, o);
        }
        if (lane == 0) {
            gxyz[3 * p + 0] = static_cast<T>(ax);
            gxyz[3 * p + 1] = static_cast<T>(ay);
            gxyz[3 * p + 2] = static_cast<T>(az);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef void (*WkKernel)(const WkParams);

struct WkLaunch {
    const void* func;
    WkKernel kern;
    WkParams prm;
    int grid, threads;
    size_t smem;
};

template <typename T, typename R, bool LODD> static WkKernel wk_pick2(int deriv, int norm) {
    if (deriv == 0) return norm ? sph_w_kernel<T, R, 0, true, LODD> : sph_w_kernel<T, R, 0, false, LODD>;
    if (deriv == 1) return norm ? sph_w_kernel<T, R, 1, true, LODD> : sph_w_kernel<T, R, 1, false, LODD>;
    return norm ? sph_w_kernel<T, R, 2, true, LODD> : sph_w_kernel<T, R, 2, false, LODD>;
}
template <typename T, typename R> static WkKernel wk_pick(int deriv, int norm, bool lodd) {
    return lodd ? wk_pick2<T, R, true>(deriv, norm) : wk_pick2<T, R, false>(deriv, norm);
}


static inline int wk_plan(int sm_count, int smem_optin, int64_t n, int l_max, int normalized, int dtype,
                          void* sph, void* dsph, void* ddsph, const void* xyz, const SphTables* d_tab,
                          WkLaunch* out) {
    const int deriv = ddsph ? 2 : (dsph ? 1 : 0);
    const int esize = dtype == 0 ? 4 : 8;
    int nbuf = g_opt.w_nbuf;   // measured on C4: one image per warp and more warps beats two images
    if (nbuf < 1) nbuf = 1;
    if (nbuf > 2) nbuf = 2;
    const int budget = smem_optin - 1024;
    int warps = 0;
    for (;;) {
        WkSmem lay(l_max, deriv, esize, nbuf);
        warps = (int)(((size_t)budget - lay.tab_bytes) / lay.warp_bytes);
        if (warps >= 4 || nbuf == 1) break;
        nbuf = 1;
    }
    if (warps < 1) return 1;
    const int want = g_opt.w_warps > 0 ? g_opt.w_warps : WK_MAX_THREADS / 32;
    if (warps > want) warps = want;
    int64_t per_sm = (n + sm_count - 1) / sm_count;
    if (per_sm < warps) warps = (int)(per_sm < 1 ? 1 : per_sm);
    // points per warp: amortise the per-CTA table copy, but keep >= ~16 waves of CTAs
    int64_t ppw = g_opt.w_ppw;
    if (ppw <= 0) {
        ppw = n / ((int64_t)sm_count * warps * 16);
        if (ppw > 8) ppw = 8;
    }
    if (ppw < 1) ppw = 1;
    const int64_t ctas = (n + warps * ppw - 1) / (warps * ppw);
    if (ctas > 0x7fffffff) return 1;
    WkSmem lay(l_max, deriv, esize, nbuf);
    const bool lodd = (l_max & 1) == 0;
    out->kern = dtype == 0 ? wk_pick<float, double>(deriv, normalized, lodd) : wk_pick<double, dd>(deriv, normalized, lodd);
    out->func = (const void*)out->kern;
    out->prm.xyz = xyz;
    out->prm.sph = sph;
    out->prm.dsph = dsph;
    out->prm.ddsph = ddsph;
    out->prm.tab = d_tab;
    out->prm.n = n;
    out->prm.l_max = l_max;
    out->prm.warps_per_cta = warps;
    out->prm.nbuf = nbuf;
    out->prm.pts_per_warp = (int)ppw;
    // chunks of whole l-rows, at most WK_CH harmonics each: the partition that minimises
    // (32-pair assembly passes) x ~320 instructions + (chunks) x ~290 instructions, by dynamic programming
    int best[SPH_MAX_L + 2], from[SPH_MAX_L + 2];
    best[0] = 0;
    for (int e = 1; e <= l_max + 1; ++e) {   // rows [0, e) covered
        best[e] = 1 << 30;
        for (int b = e - 1; b >= 0 && e * e - b * b <= WK_CH; --b) {
            const int pairs = e * (e + 1) / 2 - b * (b + 1) / 2;
            const int c = best[b] + (pairs + 31) / 32 * 320 + 290;
            if (c < best[e]) best[e] = c, from[e] = b;
        }
    }
    int nc = 0;
    for (int e = l_max + 1; e > 0; e = from[e]) ++nc;
    out->prm.row0[nc] = (unsigned char)(l_max + 1);
    for (int e = l_max + 1, i = nc; e > 0; e = from[e]) out->prm.row0[--i] = (unsigned char)from[e];
    out->prm.n_chunks = nc;
    out->grid = (int)ctas;
    out->threads = warps * 32;
    out->smem = lay.tab_bytes + (size_t)warps * lay.warp_bytes;
    return 0;
}

static inline void wk_launch(const WkLaunch& lw, cudaStream_t stream) {
    lw.kern<<<lw.grid, lw.threads, lw.smem, stream>>>(lw.prm);
}

static inline int wk_launch_vjp(int sm_count, const void* dsph, const void* gsph, void* gxyz, int64_t n, int L,
                                int dtype, cudaStream_t stream) {
    int64_t blocks = (n + 7) / 8;
    if (blocks > (int64_t)sm_count * 8) blocks = (int64_t)sm_count * 8;
    if (dtype == 0)
        sph_vjp_warp_kernel<float><<<(int)blocks, 256, 0, stream>>>((const float*)dsph, (const float*)gsph,
                                                                     (float*)gxyz, n, L);
    else
        sph_vjp_warp_kernel<double><<<(int)blocks, 256, 0, stream>>>((const double*)dsph, (const double*)gsph,
                                                                      (double*)gxyz, n, L);
    return cudaGetLastError() == cudaSuccess ? 0 : 1;
}

}  // namespace sphb200
