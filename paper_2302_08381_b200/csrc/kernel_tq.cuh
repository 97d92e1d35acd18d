// "tq" kernel: two phases per batch of points, the whole CTA on both.  Any l_max, run-time l_max.
//   MODE 0  forward: values / + gradients / + Hessians (optionally in another axis / scale
//           convention, CONV: SURVEY 8(f) N4)
//   MODE 1  second-order VJP (double backward): the Hessians are
//           assembled as in MODE 0 and contracted on the fly, nothing but grad_grad rows is stored
//   MODE 2  recompute-in-backward VJP: the gradients are assembled as in
//           MODE 0 and contracted with grad_sph on the fly, nothing is staged at all
//
// Why (profiles/r2_*): the unrolled tpb kernels keep a point's whole Legendre
// column in registers and stage 16 points per warp, so from l_max ~ 11 (gradients) / 6 (Hessians)
// they run at 168-255 registers with 43-74 KB images: 3-8 warps per SM, latency-bound.  The
// run-time kernels that took over there (tpg, w) tie the recurrences and the assembly to the same
// lanes (lane = column class, or lane = m), so most lanes idle through one of the two.  Here the two
// are separate phases with their own mapping, and the image is sized by the store engine's needs
// (a contiguous byte range per output array, 16-byte aligned), not by the warp width:
//
//   phase A  lane = POINT (32-point batches; 2 / 4 lanes per point for batches of 16 / 8, which the
//            long rows need to fit shared memory).  The batch's points run Eq. 9 and the
//            folded Eq. 7 (tables.h) -- double for f32 I/O, double-double for f64 I/O -- with
//            coefficient loads from the constant bank; the columns m of the triangle are dealt to
//            the CTA's warps (and lane classes) in snake order (balanced lengths).  Qt_l^m, (c_m, s_m)
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
#include "tq_table.h"

namespace sphb200 {

// every translation unit that instantiates these kernels carries its own copy of the tables
static __constant__ SphTables c_tables_tq;

struct TqParams {
    const void* xyz;
    void* sph;                   // MODE 0: sph [n,L];  MODE 1: grad_grad_sph [n,L] (may be NULL)
    void* dsph;
    void* ddsph;
    const void* gsph;            // MODE 1, 2: grad_sph [n,L] (the upstream gradient w)
    const void* vvec;            // MODE 1: v [n,3] (the upstream gradient on grad_xyz)
    void* gxyz;                  // MODE 1: grad_grad_xyz [n,3];  MODE 2: grad_xyz [n,3]
    const SphTables* tab;        // global-memory copy of the tables (phase B: G1, Gz, H2, Hxz, Hzz)
    const unsigned short* lm;    // [(l_max+1)(l_max+2)/2]: l | m << 8 of triangle index t
    const double2* ab_hi;        // {A, B}[t] of the folded Eq. 7 (tables.h), high parts
    const double2* ab_lo;        // ... low parts (double-double recurrences)
    int64_t n;
    int l_max;
    int batch;                   // points per phase-A batch: 32, 16 or 8 (1, 2 or 4 lanes per point)
    int pts_tile;                // points per image; divides batch
    int batches_per_cta;         // consecutive batches one CTA works through
    int n_images;                // 2: a tile drains while the next is assembled; 1: the longest rows
    int cs_warps;                // f64 I/O: warps of phase A that run Eq. 9 only (1 or 2; the others run the columns)
    // CONV: the harmonics are evaluated at (x', y', z') = xyz[src[0..2]] and derivative axis a of the
    // evaluation frame is the caller's axis row[a]; every degree-l output is multiplied by lscale[l]
    int src[3], row[3];
    double lscale[SPH_MAX_L + 1];
};

constexpr int TQ_MAX_WARPS = 16;   // (one CTA per SM where the staging images leave room for no second one)
constexpr int TQ_RED_WARPS = 8;    // warps per CTA of the contracting modes (their reduction slots are sized for it)

// shared-memory carve-up (bytes), identical on host and device
struct TqSmem {
    int T, TP, CP, PTB;
    size_t gt_off, ht_off, lm_off, sl_off, red_off, q_off, cs_off, pt_off, img_off, img_bytes, total;
    size_t reg_g, reg_h;   // offsets of the dsph / ddsph regions inside an image
    // deriv: derivative order assembled; img_rows: rows per point staged (1 / 4 / 13 forward, 1 or 0
    // for the contracting modes); pt_bytes: per-point record (x, y, z, 1/r [, v])
    // direct: no staging image at all (phase B stores straight to global memory)
    __host__ __device__ TqSmem(int l_max, int deriv, int img_rows, int pt_bytes, int esize, int batch, int pts_tile,
                               int n_images, bool direct = false) {
        if (direct) img_rows = 0, n_images = 0;
        T = (l_max + 1) * (l_max + 2) / 2;
        TP = (T + 3) | 1;          // doubles per point: three finite pad entries, odd pitch (conflict-free lane = point stores)
        CP = (l_max + 3) | 1;      // (c, s) pairs per point behind two zero pad entries ((c,s)_{-1}, (c,s)_{-2}), odd pitch
        PTB = pt_bytes;
        size_t o = 0;
        gt_off = o;                // {G1, Gz}[t]
        o += deriv >= 1 ? (size_t)T * 16 : 0;
        ht_off = o;                // {H2, Hxz, Hzz, -}[t]
        o += deriv >= 2 ? (size_t)T * 32 : 0;
        sl_off = o;                // lscale[l] (CONV)
        o += (size_t)(SPH_MAX_L + 1) * 8 + 8;
        red_off = o;               // [warps][pairs of points of a tile][2][3] partial sums of the contracting modes
        const bool contracting = !direct && (img_rows == 0 || pt_bytes == 64);   // (modes 1 and 2)
        o += contracting ? (size_t)2 * TQ_RED_WARPS * ((pts_tile + 1) / 2) * 48 : 0;
        lm_off = o;                // l | m << 8
        o += ((size_t)T * 2 + 15) & ~(size_t)15;
        q_off = o;
        o += (size_t)batch * TP * 8;
        o = (o + 15) & ~(size_t)15;
        cs_off = o;
        o += (size_t)batch * CP * 16;
        pt_off = o;
        o += (size_t)batch * pt_bytes;
        img_off = (o + 127) & ~(size_t)127;
        // one region per output array, each with 16 bytes of slack: a region is staged at the offset
        // (0..15 bytes) its global address has from a 16-byte boundary, so that the aligned body of
        // the run can leave as one bulk store whatever the tile's first point is
        const size_t L = (size_t)(l_max + 1) * (l_max + 1);
        const size_t sb = (size_t)pts_tile * L * esize;
        reg_g = (sb + 16 + 15) & ~(size_t)15;
        reg_h = reg_g + ((3 * sb + 16 + 15) & ~(size_t)15);
        const size_t end = img_rows == 0 ? 0 : (img_rows == 1 ? reg_g : (img_rows == 4 ? reg_h : reg_h + ((9 * sb + 16 + 15) & ~(size_t)15)));
        img_bytes = (end + 127) & ~(size_t)127;
        total = img_off + (size_t)n_images * img_bytes;
    }
};
__host__ __device__ constexpr int tq_img_rows(int mode, int deriv) { return mode == 2 ? 0 : (mode == 1 ? 1 : (deriv == 0 ? 1 : (deriv == 1 ? 4 : 13))); }
__host__ __device__ constexpr int tq_pt_bytes(int mode) { return mode == 1 ? 64 : 32; }

// shared-memory accesses through 32-bit shared addresses (one IADD per address instead of the
// 64-bit generic arithmetic the compiler emits for pointers into a dynamic carve-up).  volatile:
// they keep their order against the barriers and fences, which are volatile too.
__device__ __forceinline__ double tq_lds(uint32_t a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double tq_lds8(uint32_t a) {   // [a + 8]
    double v;
    asm volatile("ld.shared.f64 %0, [%1+8];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double tq_lds16(uint32_t a) {  // [a + 16]
    double v;
    asm volatile("ld.shared.f64 %0, [%1+16];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void tq_lds2(uint32_t a, double& x, double& y) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a));
}
__device__ __forceinline__ unsigned tq_lds_u16(uint32_t a) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void tq_sts(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void tq_sts(uint32_t a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
// (DIRECT: the same call sites store to global memory, streaming)
__device__ __forceinline__ void tq_sts(unsigned char* a, float v) { __stcs(reinterpret_cast<float*>(a), v); }
__device__ __forceinline__ void tq_sts(unsigned char* a, double v) { __stcs(reinterpret_cast<double*>(a), v); }
__device__ __forceinline__ void tq_sts2(uint32_t a, double x, double y) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}

// DIRECT (forward mode only): no staging image; phase B stores every harmonic straight to global memory
// (lanes = consecutive (l, m) of one point: runs of consecutive words for +m, descending ones for -m).
// Where one tile image leaves room for a single CTA per SM (long rows), the shared memory this frees
// buys resident warps, and the kernel is latency-bound there.
template <typename T, typename R, int DERIV, bool NORM, int MODE, bool CONV, int DIRECT = 0>
__global__ void __launch_bounds__(TQ_MAX_WARPS * 32, 1) sph_tq_kernel(const TqParams prm) {
    using RT = rec<R>;
    constexpr int ES = (int)sizeof(T);
    constexpr int PTB = tq_pt_bytes(MODE);
    static_assert(MODE == 0 || (MODE == 1 && DERIV == 2) || (MODE == 2 && DERIV == 1), "mode / derivative order");
    static_assert(DIRECT == 0 || ((DIRECT == 2 || DIRECT == 4) && MODE == 0), "direct stores (2 or 4 points per lane): forward mode only");
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int W = blockDim.x >> 5;
    const int l_max = prm.l_max;
    const int L = (l_max + 1) * (l_max + 1);
    const int B = prm.batch, P = DIRECT ? prm.batch : prm.pts_tile;   // (DIRECT: the batch is the one tile)
    const TqSmem lay(l_max, DERIV, tq_img_rows(MODE, DERIV), PTB, ES, B, P, prm.n_images, DIRECT != 0);
    const int TT = lay.T, TP = lay.TP, CP = lay.CP;
    const uint32_t s0 = smem_u32(smem);
    const uint32_t sGT = s0 + (uint32_t)lay.gt_off, sHT = s0 + (uint32_t)lay.ht_off, sLM = s0 + (uint32_t)lay.lm_off;
    const uint32_t sSL = s0 + (uint32_t)lay.sl_off;
    const uint32_t sQ = s0 + (uint32_t)lay.q_off, sCS = s0 + (uint32_t)lay.cs_off, sPT = s0 + (uint32_t)lay.pt_off;
    unsigned char* img0 = smem + lay.img_off;
    const int64_t n = prm.n;
    const T* __restrict__ xyz = static_cast<const T*>(prm.xyz);
    T* __restrict__ sph = static_cast<T*>(prm.sph);
    T* __restrict__ dsph = static_cast<T*>(prm.dsph);
    T* __restrict__ ddsph = static_cast<T*>(prm.ddsph);
    const T* __restrict__ gsph = static_cast<const T*>(prm.gsph);
    T* __restrict__ gxyz = static_cast<T*>(prm.gxyz);
    const SphTables& TB = c_tables_tq;
    const uint64_t policy = policy_evict_first();

    // once per CTA: phase B's coefficient tables (times the degree's scale for CONV: every output of
    // degree l is linear in them and in Qt_l^m, which phase B scales as it reads it) and the (l, m)
    // of every triangle index -> shared memory; the pad entries behind every point's triangle and
    // in front of its (c, s) list, which phase B reads times a zero coefficient
    for (int t = threadIdx.x; t < TT; t += blockDim.x) {
        const unsigned short lmv = __ldg(prm.lm + t);
        const double sl = CONV ? prm.lscale[lmv & 0xff] : 1.0;
        if (DERIV >= 1) tq_sts2(sGT + t * 16, sl * __ldg(&prm.tab->G1[t]), sl * __ldg(&prm.tab->Gz[t]));
        if (DERIV >= 2) {
            tq_sts2(sHT + t * 32, sl * __ldg(&prm.tab->H2[t]), sl * __ldg(&prm.tab->Hxz[t]));
            tq_sts(sHT + t * 32 + 16, sl * __ldg(&prm.tab->Hzz[t]));
        }
        reinterpret_cast<unsigned short*>(smem + lay.lm_off)[t] = lmv;
    }
    if (CONV)
        for (int l = threadIdx.x; l <= l_max; l += blockDim.x) tq_sts(sSL + l * 8, prm.lscale[l]);
    for (int i = threadIdx.x; i < B * 3; i += blockDim.x) tq_sts(sQ + ((i / 3) * TP + TT + (i % 3)) * 8, 0.0);
    for (int i = threadIdx.x; i < B * 2; i += blockDim.x) tq_sts2(sCS + ((i >> 1) * CP + (i & 1)) * 16, 0.0, 0.0);

    const int NCH = (TT + 31) >> 5;                    // 32-pair chunks of one point's triangle
    const int d_pl = W / NCH, d_ch = W - d_pl * NCH;   // one step of a warp through the (point group, chunk) units
    const int w_pl0 = warp / NCH, w_ch0 = warp - w_pl0 * NCH;
    // points one lane takes through phase B with the same (l, m): 2, or DIRECT = 4 (the per-(l, m) decode and
    // table loads are then shared by four points; which of the two is faster depends on the cell: tq_table.h)
    constexpr int NPL = DIRECT == 4 ? 4 : 2;
    const int PP = (P + NPL - 1) / NPL;               // groups of NPL points per tile (the last one may hold fewer)
    const uint32_t row_b = (uint32_t)L * ES;          // bytes of one row of one point
    const uint32_t s_bytes = (uint32_t)P * row_b;     // bytes of the tile's sph image
    // derivative axis a of the evaluation frame is row `row[a]` of the caller's arrays
    const uint32_t rx = (CONV ? prm.row[0] : 0) * row_b, ry = (CONV ? prm.row[1] : 1) * row_b, rz = (CONV ? prm.row[2] : 2) * row_b;
    // Phase B for ONE (l, m >= 0) pair (triangle index t) and up to TWO points: the points pbb, pbb + 1
    // of the batch (global index pg0, pg0 + 1), staged as points plb, plb + 1 of the image whose
    // regions start at sS / sG / sH.  acc: this lane's partial sums of the contracting modes.
    // wv: the upstream gradient of the four harmonics {(l,+m), (l,-m)} x {point 0, 1} (contracting modes).
    // (sS / sG / sH: 32-bit shared addresses, or for DIRECT global byte pointers to the tile's first point)
    auto assemble = [&](int t, int plb, int pbb, int npt, const T* wv, auto sS, auto sG, auto sH, double* acc) {
        // ---- per (l, m): shared by the two points ----
        const unsigned lmv = tq_lds_u16(sLM + t * 2);
        const int l = (int)(lmv & 0xffu), m = (int)(lmv >> 8);
        const double dl = (double)l, dm = (double)m;
        // the (l, -m) outputs are stored FIRST and unconditionally: for m = 0 they land on the
        // (l, 0) slot and the cos-branch store that follows overwrites them (no branch)
        const int kc = l * (l + 1) + m;
        const uint32_t kc_b = (uint32_t)kc * ES, m2_b = (uint32_t)(2 * m) * ES;
        const uint32_t l8 = (uint32_t)l * 8;
        double G1 = 0.0, Gz = 0.0, H2 = 0.0, Hxz = 0.0, Hzz = 0.0, sl = 1.0;
        if constexpr (DERIV >= 1) tq_lds2(sGT + t * 16, G1, Gz);
        if constexpr (DERIV >= 2) {
            tq_lds2(sHT + t * 32, H2, Hxz);
            Hzz = tq_lds16(sHT + t * 32);
        }
        if constexpr (CONV) sl = tq_lds(sSL + l * 8);
        const double dmm = dm * (dm - 1.0);
#pragma unroll
        for (int j = 0; j < NPL; ++j) {
            if (j >= npt) break;
            const int pl = plb + j;   // point inside the image
            const int pb = pbb + j;   // ... inside the batch
            double x, y, z, ri;
            tq_lds2(sPT + pb * PTB, x, y);
            tq_lds2(sPT + pb * PTB + 16, z, ri);
            const uint32_t aQ = sQ + (pb * TP + t) * 8;
            const uint32_t aC = sCS + (pb * CP + m + 2) * 16;
            const double Q = CONV ? sl * tq_lds(aQ) : tq_lds(aQ);
            double c0, As;
            tq_lds2(aC, c0, As);
            const double Ac = (m == 0) ? SPH_INV_SQRT2 : c0;
            const auto aS = sS + pl * row_b + kc_b;
            if constexpr (MODE == 0) {
                tq_sts(aS - m2_b, static_cast<T>(Q * As));
                tq_sts(aS, static_cast<T>(Q * Ac));
            }
            double wc = 0.0, ws = 0.0;
            if constexpr (MODE != 0) {
                wc = static_cast<double>(wv[2 * j]);
                ws = static_cast<double>(wv[2 * j + 1]);
            }
            if constexpr (DERIV >= 1) {
                const uint32_t aQ1 = aQ - l8;   // Qt_{l-1}^m; Qt_{l-1}^{m+1} behind it
                const double q1 = G1 * tq_lds8(aQ1);   // F_l^m Q_{l-1}^{m+1}
                const double qz = Gz * tq_lds(aQ1);    // F_l^m (l+m) Q_{l-1}^m
                double c1, s1;
                tq_lds2(aC - 16, c1, s1);
                // Eq. 10: cos: A_x = m c_{m-1}, A_y = -m s_{m-1}; sin: A_x = m s_{m-1}, A_y = m c_{m-1}
                const double mc1 = dm * c1, ms1 = dm * s1;
                const double lQ = dl * Q;
                const double E1 = NORM ? q1 - lQ : q1;
                const double EZ = NORM ? SPH_FMA(-lQ, z, qz) : qz;
                const double sg = NORM ? ri : 1.0;
                const double E1g = E1 * sg;
                const double ax = x * E1g, ay = y * E1g, az = EZ * sg, Qg = Q * sg;
                const double Qc = Qg * mc1, Qs_ = Qg * ms1;
                const double gxs = SPH_FMA(ax, As, Qs_), gys = SPH_FMA(ay, As, Qc), gzs = az * As;
                const double gxc = SPH_FMA(ax, Ac, Qc), gyc = SPH_FMA(ay, Ac, -Qs_), gzc = az * Ac;
                if constexpr (MODE == 0) {
                    const auto aG = sG + pl * 3 * row_b + kc_b;
                    const auto aGs = aG - m2_b;
                    tq_sts(aGs + rx, static_cast<T>(gxs));
                    tq_sts(aGs + ry, static_cast<T>(gys));
                    tq_sts(aGs + rz, static_cast<T>(gzs));
                    tq_sts(aG + rx, static_cast<T>(gxc));
                    tq_sts(aG + ry, static_cast<T>(gyc));
                    tq_sts(aG + rz, static_cast<T>(gzc));
                } else if constexpr (MODE == 2) {   // grad_xyz[a] += dY/dx_a * grad_sph, both harmonics
                    acc[3 * j + 0] = SPH_FMA(gxc, wc, SPH_FMA(gxs, ws, acc[3 * j + 0]));
                    acc[3 * j + 1] = SPH_FMA(gyc, wc, SPH_FMA(gys, ws, acc[3 * j + 1]));
                    acc[3 * j + 2] = SPH_FMA(gzc, wc, SPH_FMA(gzs, ws, acc[3 * j + 2]));
                }
                if constexpr (DERIV >= 2) {
                    const uint32_t aQ2 = aQ1 - l8 + 8;   // Qt_{l-2}^m, then m+1, m+2
                    const double q2 = H2 * tq_lds16(aQ2);    // F_l^m Q_{l-2}^{m+2}
                    const double qxz = Hxz * tq_lds8(aQ2);   // F_l^m (l+m) Q_{l-2}^{m+1}
                    const double qzz = Hzz * tq_lds(aQ2);    // F_l^m (l+m)(l+m-1) Q_{l-2}^m
                    double c2, s2;
                    tq_lds2(aC - 32, c2, s2);
                    // Eq. 10 twice: cos: A_xx = m(m-1) c_{m-2}, A_xy = -m(m-1) s_{m-2}; sin: s_{m-2}, c_{m-2}
                    const double mmc2 = dmm * c2, mms2 = dmm * s2;
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
                    double vx = 0.0, vy = 0.0, vz = 0.0, pad_;
                    if constexpr (MODE == 1) {
                        tq_lds2(sPT + pb * PTB + 32, vx, vy);
                        tq_lds2(sPT + pb * PTB + 48, vz, pad_);
                    }
                    // one branch: its six second derivatives, stored (MODE 0) or contracted (MODE 1)
                    auto branch2 = [&](auto a, double A, double Ax, double Ay, double Axx, double Axy, double wk,
                                       double gx, double gy, double gz) {
                        const double QAxx = Qh * Axx;
                        const double hxx = SPH_FMA(cxx, A, SPH_FMA(bx2, Ax, QAxx));
                        const double hyy = SPH_FMA(cyy, A, SPH_FMA(by2, Ay, -QAxx));
                        const double hxy = SPH_FMA(cxy, A, SPH_FMA(bx, Ay, SPH_FMA(by, Ax, Qh * Axy)));
                        const double hxz = SPH_FMA(cxz, A, ezh * Ax);
                        const double hyz = SPH_FMA(cyz, A, ezh * Ay);
                        const double hzz = czz * A;
                        if constexpr (MODE == 0) {
                            const T txx = static_cast<T>(hxx), tyy = static_cast<T>(hyy), tzz = static_cast<T>(hzz);
                            const T txy = static_cast<T>(hxy), txz = static_cast<T>(hxz), tyz = static_cast<T>(hyz);
                            // row (a, b) of the caller's [3][3] block; both triangles stored, exactly equal
                            tq_sts(a + 3 * rx + rx, txx);
                            tq_sts(a + 3 * rx + ry, txy);
                            tq_sts(a + 3 * rx + rz, txz);
                            tq_sts(a + 3 * ry + rx, txy);
                            tq_sts(a + 3 * ry + ry, tyy);
                            tq_sts(a + 3 * ry + rz, tyz);
                            tq_sts(a + 3 * rz + rx, txz);
                            tq_sts(a + 3 * rz + ry, tyz);
                            tq_sts(a + 3 * rz + rz, tzz);
                        } else {
                            // grad_grad_sph[k] = sum_a dY_k/dx_a v_a;  grad_grad_xyz[b] += w_k sum_a d2Y_k/dx_a dx_b v_a
                            tq_sts(a, static_cast<T>(SPH_FMA(gx, vx, SPH_FMA(gy, vy, gz * vz))));
                            acc[3 * j + 0] = SPH_FMA(wk, SPH_FMA(hxx, vx, SPH_FMA(hxy, vy, hxz * vz)), acc[3 * j + 0]);
                            acc[3 * j + 1] = SPH_FMA(wk, SPH_FMA(hxy, vx, SPH_FMA(hyy, vy, hyz * vz)), acc[3 * j + 1]);
                            acc[3 * j + 2] = SPH_FMA(wk, SPH_FMA(hxz, vx, SPH_FMA(hyz, vy, hzz * vz)), acc[3 * j + 2]);
                        }
                    };
                    const auto aH = (MODE == 0 ? sH + pl * 9 * row_b : aS - kc_b) + kc_b;
                    branch2(aH - m2_b, As, ms1, mc1, mms2, mmc2, ws, gxs, gys, gzs);
                    branch2(aH, Ac, mc1, -ms1, mmc2, -mms2, wc, gxc, gyc, gzc);
                }
            }
        }
    };
    // The upstream gradient of pair t for the points pg0, pg0 + 1 (contracting modes), fetched one unit
    // ahead of its use so that the global-memory latency hides under the previous unit's arithmetic;
    // 0 for the absent (l, -0), for points past the end and for lanes past the triangle
    auto load_w = [&](int t, int npt, int64_t pg0, T* wv) {
        wv[0] = wv[1] = wv[2] = wv[3] = T(0);
        if (t < TT) {
            const unsigned lmv = tq_lds_u16(sLM + t * 2);
            const int l = (int)(lmv & 0xffu), m = (int)(lmv >> 8);
            const int kc = l * (l + 1) + m;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int64_t pg = pg0 + j;
                if (j < npt && pg < n) {
                    wv[2 * j] = __ldg(gsph + pg * L + kc);
                    if (m > 0) wv[2 * j + 1] = __ldg(gsph + pg * L + kc - 2 * m);
                }
            }
        }
    };
    // The image's runs (one per output array: np points' rows, contiguous in global memory) leave: the
    // 16-byte-aligned body by TMA, the few elements before and behind it by plain stores.  One thread.
    auto emit_runs = [&](int64_t p0, int np, const T* S0, const T* G0, const T* H0, uint32_t dS, uint32_t dG, uint32_t dH) {
        auto run = [&](T* g, const T* src, uint32_t d, uint32_t bytes) {
            uint32_t head = (16u - d) & 15u;
            if (head > bytes) head = bytes;
            const uint32_t body = (bytes - head) & ~15u;
            for (uint32_t i = 0; i < head / ES; ++i) st_cs(g + i, src[i]);
            if (body) bulk_store_hint(g + head / ES, src + head / ES, body, policy);
            for (uint32_t i = (head + body) / ES; i < bytes / ES; ++i) st_cs(g + i, src[i]);
        };
        const uint32_t sb = (uint32_t)np * row_b;
        run(sph + p0 * L, S0, dS, sb);
        if (MODE == 0 && DERIV >= 1) run(dsph + p0 * 3 * L, G0, dG, 3u * sb);
        if (MODE == 0 && DERIV >= 2) run(ddsph + p0 * 9 * L, H0, dH, 9u * sb);
        bulk_commit();
    };
    // ragged end of the batch: np (< the image's points) points by plain stores, threads tid of nthr
    auto emit_plain = [&](int64_t p0, int np, const T* S0, const T* G0, const T* H0, int tid, int nthr) {
        for (int i = tid; i < np * L; i += nthr) st_cs(sph + p0 * L + i, S0[i]);
        if (MODE == 0 && DERIV >= 1)
            for (int i = tid; i < np * 3 * L; i += nthr) st_cs(dsph + p0 * 3 * L + i, G0[i]);
        if (MODE == 0 && DERIV >= 2)
            for (int i = tid; i < np * 9 * L; i += nthr) st_cs(ddsph + p0 * 9 * L + i, H0[i]);
    };
    constexpr bool HAS_IMG = MODE != 2 && !DIRECT;

    // this lane's point of a batch; lanes past the end get a harmless point
    auto load_xyz = [&](int64_t b0, T& xa, T& ya, T& za) {
        const int64_t p = b0 + (lane & (B - 1));
        xa = T(0), ya = T(0), za = T(1);
        if (p < n) {
            xa = __ldg(xyz + 3 * p + (CONV ? prm.src[0] : 0));
            ya = __ldg(xyz + 3 * p + (CONV ? prm.src[1] : 1));
            za = __ldg(xyz + 3 * p + (CONV ? prm.src[2] : 2));
        }
    };
    T xn, yn, zn;   // the NEXT batch's point: fetched while the current batch is assembled
    load_xyz((int64_t)blockIdx.x * prm.batches_per_cta * B, xn, yn, zn);

    int tile_no = 0;   // tiles this CTA has issued: parity picks the image
    for (int bi = 0; bi < prm.batches_per_cta; ++bi) {
        const int64_t b0 = ((int64_t)blockIdx.x * prm.batches_per_cta + bi) * B;
        if (b0 >= n) break;

        // ---- phase A: lane = point --------------------------------------------------------------
        __syncthreads();   // the previous batch's phase B has finished reading the scratch
        {
            // B = 32: lane = point.  B = 16 / 8: 2 / 4 lanes per point, each its own share of the
            // columns (class `cls`), so that every lane of the warp works whatever the batch size
            const int pt_l = lane & (B - 1), cls = lane / B, NC = 32 / B;
            const int64_t p = b0 + pt_l;
            const double x = static_cast<double>(xn), y = static_cast<double>(yn), z = static_cast<double>(zn);
            if (bi + 1 < prm.batches_per_cta) load_xyz(b0 + B, xn, yn, zn);   // in flight through this batch
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
            // Eq. 9 and the point itself.  f32 I/O (plain double: 4 operations per power): the lanes
            // with the shortest columns do it on the side.  f64 I/O (double-double: ~50 per power, against
            // ~23 per Legendre entry): ONE chain over all m would be the critical path of the whole phase, so
            // `cs_warps` warps do nothing else, each lane class a SEGMENT of the powers, started from
            // (x + iy)^(segment start) by squarings (segment length a power of two).
            constexpr bool DD = sizeof(R) > sizeof(double);
            const int WC = DD ? prm.cs_warps : 0;          // warps that only run Eq. 9
            const int Wq = W - WC;                          // warps that run the Legendre columns
            const bool cs_lane = DD ? warp >= Wq : (warp == W - 1 && cls == NC - 1);
            if (cs_lane) {
                const int seg = DD ? (warp - Wq) * NC + cls : 0, nseg = DD ? WC * NC : 1;
                // segments of h = 2^sq powers, the largest power of two <= ceil((l_max + 1) / nseg); the
                // last segment takes what is left
                int h = 1, sq = 0;
                while (2 * h * nseg <= l_max + nseg) h <<= 1, ++sq;
                if (seg == 0) {
                    tq_sts2(sPT + pt_l * PTB, to_double(X), to_double(Y));
                    tq_sts2(sPT + pt_l * PTB + 16, to_double(Z), rinv);
                    if constexpr (MODE == 1) {
                        const T* __restrict__ vv = static_cast<const T*>(prm.vvec);
                        double vx = 0.0, vy = 0.0, vz = 0.0;
                        if (p < n) {
                            vx = static_cast<double>(__ldg(vv + 3 * p + 0));
                            vy = static_cast<double>(__ldg(vv + 3 * p + 1));
                            vz = static_cast<double>(__ldg(vv + 3 * p + 2));
                        }
                        tq_sts2(sPT + pt_l * PTB + 32, vx, vy);
                        tq_sts2(sPT + pt_l * PTB + 48, vz, 0.0);
                    }
                }
                R c = RT::make(1.0, 0.0), s = RT::make(0.0, 0.0);
                if (seg > 0) {
                    R pr = X, pi = Y;                       // (x + iy)^h by squarings ...
                    for (int i = 0; i < sq; ++i) {
                        const R prn = pr * pr - pi * pi;
                        const R pin = (pr * pi) * 2.0;
                        pr = prn;
                        pi = pin;
                    }
                    c = pr, s = pi;                         // ... to the power seg
                    for (int i = 1; i < seg; ++i) {
                        const R cn = c * pr - s * pi;
                        const R sn = c * pi + s * pr;
                        c = cn;
                        s = sn;
                    }
                }
                const int m0 = seg * h, m1 = seg == nseg - 1 ? l_max + 1 : min(m0 + h, l_max + 1);
                uint32_t a = sCS + (pt_l * CP + 2 + m0) * 16;
                for (int m = m0; m < m1; ++m, a += 16) {
                    tq_sts2(a, to_double(c), to_double(s));
                    const R cn = X * c - Y * s;
                    const R sn = X * s + Y * c;
                    c = cn;
                    s = sn;
                }
            }
            // Columns of the folded Eq. 7 in ADJACENT pairs (2k, 2k+1), the pairs dealt to the V column
            // classes in snake order (class v: k = v, 2V-1-v, 2V+v, ...: balanced step counts; the classes of
            // one warp sit on neighbouring pairs, so their loops run nearly in step).  Both chains of a pair
            // run over (nearly) the same rows: a lane has two independent recurrences in flight for its whole
            // loop -- the recurrence is one dependent chain per column, ~23 double-double operations per step
            // for f64 I/O.  The row loop is unrolled by two with the roles of (q, qp) exchanged, so that no
            // register is copied from one step to the next.  Coefficients {A, B}: f64 I/O from a packed
            // global table through the read-only path (indexed constant-bank loads were the top stall), f32
            // I/O from the constant bank (measured faster there).
            const uint32_t q_out = sQ + pt_l * TP * 8;
            const int V = Wq * NC, v = warp * NC + cls;   // (the cs warps of the double-double path run no columns)
            auto next = [&](int t, const R& q, const R& qp) -> R {   // Qt_l^m from (Qt_{l-1}^m, Qt_{l-2}^m), t = TRI(l, m)
                const R w = NORM ? qp : r2 * qp;
                R qn;
                if constexpr (sizeof(R) > sizeof(double)) {
                    const double2 hi = __ldg(prm.ab_hi + t);
                    const double2 lo = __ldg(prm.ab_lo + t);
                    qn = rec_step_u(hi.x, lo.x, hi.y, lo.y, Z, q, w);   // (B_{m+1}^m = 0)
                } else {
                    qn = RT::make(TB.A_hi[t], 0.0) * (Z * q) - RT::make(TB.B_hi[t], 0.0) * w;
                }
                tq_sts(q_out + t * 8, pair_value(qn));   // (unnormalised pair from rec_step_u)
                return qn;
            };
            const int n_pairs = l_max / 2 + 1;
            for (int i = 0; warp < Wq && i * V < n_pairs; ++i) {
                const int k = (i & 1) ? (i + 1) * V - 1 - v : i * V + v;
                if (k >= n_pairs) continue;
                const int ma = 2 * k, mb = ma + 1;
                R qa = RT::make(TB.D_hi[ma], TB.D_lo[ma]), qpa = RT::make(0.0, 0.0);
                int ta = SPH_TRI(ma, ma);
                tq_sts(q_out + ta * 8, to_double(qa));
                if (mb > l_max) continue;
                ta += mb;   // SPH_TRI(l, m) - SPH_TRI(l-1, m) = l
                int tb = SPH_TRI(mb, mb);
                qpa = next(ta, qa, qpa);                           // (column a: newest in qpa)
                R qb = RT::make(TB.D_hi[mb], TB.D_lo[mb]), qpb = RT::make(0.0, 0.0);
                tq_sts(q_out + tb * 8, to_double(qb));
                int l = mb + 1;
                if (l <= l_max) {   // one single step brings column a back to (newest in qa); b: newest in qpb
                    ta += l, tb += l;
                    qa = next(ta, qpa, qa);
                    qpb = next(tb, qb, qpb);
                    ++l;
                }
                for (; l + 1 <= l_max; l += 2) {
                    ta += l, tb += l;
                    qpa = next(ta, qa, qpa);
                    qb = next(tb, qpb, qb);
                    ta += l + 1, tb += l + 1;
                    qa = next(ta, qpa, qa);
                    qpb = next(tb, qb, qpb);
                }
                if (l <= l_max) {
                    ta += l, tb += l;
                    next(ta, qa, qpa);
                    next(tb, qpb, qb);
                }
            }
        }
        __syncthreads();

        // ---- phase B: lane = (point pair of the tile, (l, m) pair) ---------------------------------
        const int n_tiles = B / P;
        for (int ti = 0; ti < n_tiles; ++ti) {
            const int64_t p0 = b0 + (int64_t)ti * P;
            if (p0 >= n) break;
            unsigned char* img = img0 + (size_t)(tile_no & (prm.n_images - 1)) * lay.img_bytes;
            // each array's run is staged at the offset its global address has from a 16-byte boundary
            const uint32_t tile_b = (uint32_t)(p0 & 15) * row_b;   // (p0 L ES) mod 16, in 32 bits
            const uint32_t dS = tile_b & 15u, dG = (3u * tile_b) & 15u, dH = (9u * tile_b) & 15u;
            unsigned char* iS = img + dS;
            unsigned char* iG = img + lay.reg_g + dG;
            unsigned char* iH = img + lay.reg_h + dH;
            const uint32_t sS = smem_u32(iS), sG = smem_u32(iG), sH = smem_u32(iH);
            if (HAS_IMG && prm.n_images == 1 && tile_no > 0) {   // the one image: its last stores must have read it
                if (threadIdx.x == 0) bulk_wait_read<0>();
                __syncthreads();
            }
            // work units = (two points of the tile, 32 consecutive pairs of the triangle), dealt to the warps
            // round-robin; (pp, ch) of this warp's unit advances incrementally (warp-uniform, no division)
            double acc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            // (two sets of slots, alternating by tile: the threads that sum one tile's need no barrier
            // against the warps that fill the next one's)
            double* red_set = reinterpret_cast<double*>(smem + lay.red_off) + (tile_no & 1) * (TQ_RED_WARPS * PP * 6);
            double* red = red_set + warp * PP * 6;   // this warp's slots
            // contracting modes: a warp's units visit the pairs of points in ascending order, so its partial
            // sums of one pair are complete when the pair changes: over the lanes, then into the warp's slot
            auto flush = [&](int pair) {
#pragma unroll
                for (int q = 0; q < 6; ++q) {
                    double v = acc[q];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    if (lane == 0) red[pair * 6 + q] = v;
                    acc[q] = 0.0;
                }
            };
            if constexpr (MODE != 0) {
                for (int i = lane; i < PP * 6; i += 32) red[i] = 0.0;
                __syncwarp();
            }
            if constexpr (MODE == 0) {
                // work units = (group of NPL points of the tile, 32 consecutive (l, m) pairs of the triangle), dealt
                // to the warps round-robin; group and chunk advance incrementally (warp-uniform, no division), so
                // that everything derived from them stays in uniform registers.  The last chunk of every group is
                // partly empty (56 % of the lanes busy at l_max = 7, 69 % at 8 and 10, 82-86 % at 9, 11, 13, 15).
                // FLAT: the items (group, pair) flattened instead, i = group * TT + t in runs of 32 lanes -- every
                // lane busy, but group and pair are per-lane values then.  Measured over all cells: it pays for the
                // f32 Hessians through an image (l_max 7 / 8 / 10 / 13: 3.9 / 4.6 / 4.3 / 4.9 -> 4.7 / 5.0 / 4.7 /
                // 5.2 TB/s) and loses 3-15 % elsewhere (f64: at the HBM roof already; direct stores: more address
                // arithmetic per lane), so it is compiled in for those kernels only.  group = floor(i / TT) by a
                // float reciprocal, exact here: i < 16 * 561 and the fraction keeps 0.5 / TT clear of an integer.
                constexpr bool FLAT = sizeof(T) == 4 && DERIV == 2 && DIRECT == 0;
                if constexpr (FLAT) {
                    const int items = PP * TT;
                    const float rcp_tt = 1.0f / (float)TT;
                    for (int i = warp * 32 + lane; i < items; i += W * 32) {
                        const int pp = (int)(((float)i + 0.5f) * rcp_tt);
                        assemble(i - pp * TT, 2 * pp, ti * P + 2 * pp, P - 2 * pp, nullptr, sS, sG, sH, acc);
                    }
                } else {
                    int pp = w_pl0, ch = w_ch0;
                    while (pp < PP) {
                        const int t = ch * 32 + lane;
                        if constexpr (DIRECT) {   // straight to the caller's arrays; points past the end are skipped here
                            const int left = (int)min((int64_t)P, n - p0) - NPL * pp;
                            if (t < TT && left > 0)
                                assemble(t, NPL * pp, NPL * pp, left, nullptr, reinterpret_cast<unsigned char*>(sph + p0 * L),
                                         reinterpret_cast<unsigned char*>(dsph + (DERIV >= 1 ? p0 * 3 * L : 0)),
                                         reinterpret_cast<unsigned char*>(ddsph + (DERIV >= 2 ? p0 * 9 * L : 0)), acc);
                        } else if (t < TT) assemble(t, 2 * pp, ti * P + 2 * pp, P - 2 * pp, nullptr, sS, sG, sH, acc);
                        ch += d_ch;
                        pp += d_pl;
                        if (ch >= NCH) {
                            ch -= NCH;
                            ++pp;
                        }
                    }
                }
            } else {
                // contracting modes: the units are dealt in contiguous ranges instead, so that a warp stays
                // on one pair of points for as long as possible (a change of pair costs a reduction)
                const int U = PP * NCH, u0 = warp * U / W, u1 = (warp + 1) * U / W;
                int pp = u0 / NCH, ch = u0 - pp * NCH, cur = pp;
                T wn[4];
                if (u0 < u1) load_w(ch * 32 + lane, P - 2 * pp, p0 + 2 * pp, wn);
                for (int u = u0; u < u1; ++u) {
                    if (pp != cur) {
                        flush(cur);
                        cur = pp;
                    }
                    const T wv[4] = {wn[0], wn[1], wn[2], wn[3]};
                    const int t = ch * 32 + lane, pp_now = pp;
                    if (++ch == NCH) {
                        ch = 0;
                        ++pp;
                    }
                    if (u + 1 < u1) load_w(ch * 32 + lane, P - 2 * pp, p0 + 2 * pp, wn);   // the next unit's
                    if (t < TT) assemble(t, 2 * pp_now, ti * P + 2 * pp_now, P - 2 * pp_now, wv, sS, sG, sH, acc);
                }
                if (u1 > u0) flush(cur);
            }
            // this tile's image must be visible to the async proxy; with two images, the other one's
            // stores (issued one tile ago) must have read it before anyone writes there again
            if (HAS_IMG) fence_proxy_async_smem();
            if (HAS_IMG && prm.n_images == 2 && threadIdx.x == 0) bulk_wait_read<0>();
            if constexpr (!DIRECT) __syncthreads();   // (DIRECT: nothing staged; the barrier ahead of phase A orders the scratch)
            const T* S0 = reinterpret_cast<const T*>(iS);
            const T* G0 = reinterpret_cast<const T*>(iG);
            const T* H0 = reinterpret_cast<const T*>(iH);
            if constexpr (MODE != 0) {
                // the tile's points: 3 sums each, over the warps in a fixed order (deterministic)
                if (threadIdx.x < 3 * P && p0 + threadIdx.x / 3 < n) {
                    const double* all = red_set;
                    const int point = threadIdx.x / 3, comp = threadIdx.x - 3 * point;
                    const int slot = (point >> 1) * 6 + (point & 1) * 3 + comp;
                    double sum = 0.0;
                    for (int w = 0; w < W; ++w) sum += all[w * PP * 6 + slot];
                    gxyz[p0 * 3 + threadIdx.x] = static_cast<T>(sum);
                }
            }
            if (HAS_IMG && (MODE == 0 || sph != nullptr)) {
                if (n - p0 >= P) {
                    if (threadIdx.x == 0) emit_runs(p0, P, S0, G0, H0, dS, dG, dH);
                } else {   // ragged last tile: plain stores
                    emit_plain(p0, (int)(n - p0), S0, G0, H0, threadIdx.x, blockDim.x);
                    __syncthreads();   // the image is free again only when every thread has copied its share
                }
            }
            ++tile_no;
        }
    }
    // shared memory must outlive the bulk stores' reads of it
    if (HAS_IMG && threadIdx.x == 0) bulk_wait_read<0>();
}

}  // namespace sphb200
