/*
 * sphericart_cuda.h -- C ABI of the B200-native spherical-harmonics hot path.
 *
 * What is computed (arXiv 2302.08381, "Fast evaluation of spherical harmonics with sphericart";
 * P:n = line n of PAPER.md): for n Cartesian points, every real spherical harmonic with
 * l <= l_max -- either the solid harmonics Ytilde_l^m = r^l Y_l^m or the harmonics
 * normalised on the unit sphere, Y_l^m = Ytilde_l^m(x/r) -- by the Cartesian scheme
 *      Ytilde_l^m = F_l^|m| Q_l^|m|(z,r) * { s_|m| (m<0) | 1/sqrt2 (m=0) | c_m (m>0) }   Eq. 5
 * with Q from the modified Legendre recurrence Eq. 7, c_m/s_m from Eq. 9 and the
 * prefactors of Eq. 3 / Eq. C1; optionally the Cartesian gradients (Eq. 10,
 * P:89-92), the Hessians (Eq. 10 applied twice) and, for the normalised variant, the chain
 * rule through x/r.  sphericart_cuda_vjp is the backward pass of P:112.
 *
 * Conventions common to every entry point
 *   dtype        0 = float32, 1 = float64: element type of EVERY array of the call.
 *   L            (l_max+1)^2 harmonics per point; inside a row the index is k = l*(l+1)+m,
 *                l ascending, m = -l..l (m<0: sin branch, m>0: cos branch; no Condon-Shortley sign;
 *                orthonormal on the sphere, Y_0^0 = 1/(2 sqrt(pi))).
 *   layouts      dense row-major: xyz [n,3], sph [n,L], dsph [n,3,L] (axis order x,y,z),
 *                ddsph [n,3,3,L] (both triangles stored, exactly equal), grad_sph [n,L],
 *                grad_xyz [n,3].
 *   pointers     DEVICE pointers unless the function name ends in _host; owned by the caller;
 *                base addresses 16-byte aligned; buffers must not alias.  The library never
 *                returns memory.  It keeps small per-device coefficient tables for the process
 *                lifetime.
 *   stream       a cudaStream_t passed as void* (NULL = the legacy default stream).  Device entry
 *                points only enqueue work: no host synchronisation.  The first call on a device
 *                uploads the tables and sets kernel attributes, so time from the second.
 *   l_max        0 <= l_max <= SPHERICART_CUDA_MAX_L.
 *   return       0 on success; otherwise one of the SPHERICART_CUDA_E* codes, nothing is launched
 *                for argument errors, and sphericart_cuda_last_error() describes the failure.
 *                n == 0 succeeds without a launch.  No exception crosses this boundary.
 *   r = 0        normalized=1 at a point with r == 0 is mathematically undefined; that point's
 *                outputs are NaN (IEEE), other points are unaffected.  normalized=0 is defined
 *                there (Ytilde_0^0 = 1/(2 sqrt(pi)), the rest 0).
 */
#ifndef SPHERICART_CUDA_H
#define SPHERICART_CUDA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPHERICART_CUDA_MAX_L 32

#define SPHERICART_CUDA_F32 0
#define SPHERICART_CUDA_F64 1

#define SPHERICART_CUDA_OK 0
#define SPHERICART_CUDA_EINVAL 1   /* bad argument (NULL, negative n, l_max out of range, bad dtype ...) */
#define SPHERICART_CUDA_EALIGN 2   /* a base pointer is not 16-byte aligned */
#define SPHERICART_CUDA_ECUDA 3    /* a CUDA runtime call or the launch failed; see last_error */
#define SPHERICART_CUDA_ENOMEM 4   /* (_host entry points) device or host allocation failed */
#define SPHERICART_CUDA_ENOTSUP 5  /* valid arguments this build has no kernel for (sphericart_cuda_expand) */

/*
 * Forward pass ("takes a list of Cartesian coordinates and evaluates the scaled
 * Ytilde_l^m and, optionally, their derivatives"; P:108 for normalized=1).
 *   xyz    [n,3]      in
 *   sph    [n,L]      out
 *   dsph   [n,3,L]    out, or NULL: no gradients
 *   ddsph  [n,3,3,L]  out, or NULL: no Hessians; non-NULL requires dsph non-NULL
 *   normalized  0: solid harmonics r^l Y, derivatives of the polynomials (Eq. 10);
 *               1: Y on the unit sphere, derivatives of x -> Ytilde(x/|x|) w.r.t. x.
 */
int sphericart_cuda_compute(const void* xyz, int64_t n, int l_max, int normalized, int dtype,
                            void* sph, void* dsph, void* ddsph, void* stream);

/*
 * Backward pass ("custom backward function to compute gradients using the derivatives
 * evaluated in the forward pass"):  grad_xyz[i,a] = sum_k dsph[i,a,k] * grad_sph[i,k].
 *   xyz       [n,3]    accepted for symmetry with the forward call, not read; may be NULL
 *   dsph      [n,3,L]  in (as written by sphericart_cuda_compute)
 *   grad_sph  [n,L]    in
 *   grad_xyz  [n,3]    out
 * BASELINE.json writes the call as (xyz, dsph, grad_sph, grad_xyz, stream); raw pointers cannot
 * carry n, l_max and dtype, so they follow the pointers (reading B1).
 */
int sphericart_cuda_vjp(const void* xyz, const void* dsph, const void* grad_sph, void* grad_xyz,
                        int64_t n, int l_max, int dtype, void* stream);

/*
 * Backward pass WITHOUT stored derivatives (the paper's own backward, P:112,
 * contracts derivatives "evaluated in the forward pass"): the derivatives of Eq. 10 --
 * through x/r for normalized = 1 -- are evaluated again from xyz inside the kernel and
 * contracted on the fly:
 *     grad_xyz[i,a] = sum_k (d sph[i,k] / d xyz[i,a]) * grad_sph[i,k].
 * Same result as sphericart_cuda_compute(..., dsph, ...) followed by sphericart_cuda_vjp up to
 * rounding, reading 3 + L values per point instead of 4 L + 3, and the forward pass need not write
 * dsph.  Device pointers, caller-owned, 16-byte aligned; asynchronous on `stream`.
 *   xyz       [n,3]    in
 *   grad_sph  [n,L]    in
 *   grad_xyz  [n,3]    out
 * Any 0 <= l_max <= SPHERICART_CUDA_MAX_L (compile-time-specialised kernels for l_max <= 8, f32 <= 12;
 * the two-phase kernel above that).
 * Errors as for sphericart_cuda_compute; normalized = 1 at r = 0 gives NaN for that point only.
 */
int sphericart_cuda_vjp_recompute(const void* xyz, const void* grad_sph, void* grad_xyz, int64_t n,
                                  int l_max, int normalized, int dtype, void* stream);

/*
 * Forward pass in another convention (the paper compares with e3nn).
 *   axes   SPHERICART_CUDA_AXES_STANDARD  the paper's: the l = 1 row is proportional to (y, z, x)
 *          SPHERICART_CUDA_AXES_E3NN      the harmonics of the paper evaluated at the cyclically permuted
 *                                         point (x', y', z') = (z, x, y): the l = 1 row is proportional to
 *                                         (x, y, z); dsph / ddsph are derivatives w.r.t. the caller's x, y, z
 *   scale  what sum_m Y_lm^2 is on the unit sphere:
 *          SPHERICART_CUDA_SCALE_INTEGRAL   (2l+1)/4pi  (orthonormal; the paper's)
 *          SPHERICART_CUDA_SCALE_COMPONENT  2l+1        (every degree-l output times sqrt(4pi))
 *          SPHERICART_CUDA_SCALE_NORM       1           (... times sqrt(4pi/(2l+1)))
 * Everything else as sphericart_cuda_compute, which (axes, scale) = (0, 0) is.  The permutation is
 * applied where the point is loaded and where a derivative row is staged, the scale is folded into
 * the coefficient tables: no extra pass over the outputs.
 */
#define SPHERICART_CUDA_AXES_STANDARD 0
#define SPHERICART_CUDA_AXES_E3NN 1
#define SPHERICART_CUDA_SCALE_INTEGRAL 0
#define SPHERICART_CUDA_SCALE_COMPONENT 1
#define SPHERICART_CUDA_SCALE_NORM 2
int sphericart_cuda_compute_ex(const void* xyz, int64_t n, int l_max, int normalized, int dtype, int axes,
                               int scale, void* sph, void* dsph, void* ddsph, void* stream);

/*
 * Second-order VJP: the backward pass of the backward pass ("double backward";
 * P:112 for the backward pass, P:94 for derivatives beyond the first).  The backward pass is the map
 *     g(xyz, w)[i,a] = sum_k (d sph[i,k] / d xyz[i,a]) w[i,k],     w = grad_sph;
 * given an upstream gradient v [n,3] on its output, its own backward is
 *     grad_grad_xyz[i,b] = sum_{a,k} (d2 sph[i,k] / d xyz[i,a] d xyz[i,b]) v[i,a] w[i,k]
 *     grad_grad_sph[i,k] = sum_a     (d sph[i,k] / d xyz[i,a]) v[i,a]
 * Both derivative orders are evaluated from xyz inside the kernel (Eq. 10 once and twice, through
 * x/r for normalized = 1) and contracted as they are assembled: neither dsph nor ddsph is read or
 * written.
 *   xyz            [n,3]  in
 *   grad_sph       [n,L]  in
 *   v              [n,3]  in
 *   grad_grad_xyz  [n,3]  out
 *   grad_grad_sph  [n,L]  out, or NULL: not wanted
 * Device pointers, caller-owned, 16-byte aligned; asynchronous on `stream`; any l_max up to
 * SPHERICART_CUDA_MAX_L.  Errors as for sphericart_cuda_compute.
 */
int sphericart_cuda_vjp2(const void* xyz, const void* grad_sph, const void* v, void* grad_grad_xyz,
                         void* grad_grad_sph, int64_t n, int l_max, int normalized, int dtype, void* stream);

/*
 * Fused density expansion (the use the paper motivates, Eq. 1):
 *     coeff[s, n, lm] = sum over the points k of segment s of  radial[k, n, l] * Y_l^m(r_k / |r_k|),
 * lm = l(l+1)+m as everywhere, Y normalised (Eq. 1 evaluates Y at the direction of r_k).  The
 * harmonics are evaluated inside the kernel and never written to memory.
 *   xyz      [N,3]               in   the points r_k (e.g. neighbour vectors), N = seg_ptr[n_seg]
 *   radial   [N, n_rad, l_max+1] in   R_nl(r_k): the radial basis is the caller's (the paper fixes none)
 *                                     (xyz and radial may both be NULL when N = 0: every segment empty, coeff = 0)
 *   seg_ptr  [n_seg+1] int64     in   DEVICE array of ascending offsets into the points: segment s
 *                                     (e.g. the neighbours of centre s) is seg_ptr[s] .. seg_ptr[s+1]-1;
 *                                     an empty segment gives zeros
 *   coeff    [n_seg, n_rad, L]   out
 * Device pointers, caller-owned, 16-byte aligned (seg_ptr: 8); asynchronous on `stream`.
 * Any l_max <= SPHERICART_CUDA_MAX_L and any n_rad >= 1: a compile-time kernel (f64 tensor-core
 * contraction) for 4 <= l_max <= 8 with n_rad <= 16, a run-time-size kernel for everything else.
 * A point with r = 0 makes its segment's coefficients NaN.
 */
int sphericart_cuda_expand(const void* xyz, const void* radial, const int64_t* seg_ptr, int64_t n_seg,
                           int l_max, int n_rad, int dtype, void* coeff, void* stream);

/*
 * The same two operations on HOST buffers: the library copies xyz (and dsph/grad_sph) to the
 * device, runs the kernels above and copies the results back, in chunks on two streams so that
 * transfers overlap compute; returns after everything has landed (synchronises internally).
 * Pinned host memory gives full PCIe rate; pageable memory works.  Pointers need no alignment.
 */
int sphericart_cuda_compute_host(const void* xyz, int64_t n, int l_max, int normalized, int dtype,
                                 void* sph, void* dsph, void* ddsph);
int sphericart_cuda_vjp_host(const void* xyz, const void* dsph, const void* grad_sph,
                             void* grad_xyz, int64_t n, int l_max, int dtype);

/*
 * Backward pass (the same contraction as sphericart_cuda_vjp:
 * grad_xyz[i,a] = sum_k dsph[i,a,k] * grad_sph[i,k]) for callers that must not allocate: code under
 * CUDA graph capture, serving loops and harnesses that forbid cudaMalloc.  This call, its first
 * use on a device included, calls no cudaMalloc / cudaFree and no allocating library routine,
 * creates no stream or event, and does not synchronise: it enqueues two kernels on `stream`.
 *   dsph      [n,3,L]  in, DEVICE
 *   grad_sph  [n,L]    in, DEVICE
 *   grad_xyz  [n,3]    out, DEVICE
 * A row is cut into up to 8 slices, one warp per (point, slice) -- small batches of long rows fill
 * the GPU, which one warp per point does not -- and the slices' partial sums pass through a scratch
 * that is a file-scope `static __device__` array of the library:
 * SPHERICART_CUDA_NOALLOC_SCRATCH_BYTES (6 MiB) held by every GPU that loads the library until the
 * process exits.  Hence the limit: n <= SPHERICART_CUDA_NOALLOC_MAX_POINTS; a larger n returns
 * SPHERICART_CUDA_EINVAL with a message naming the limit (split the batch, or use
 * sphericart_cuda_vjp).  Sums are accumulated in f64 in a fixed order (deterministic); the result
 * differs from sphericart_cuda_vjp's only by the order of the additions.
 * Every call on a device shares the one scratch array: calls that may OVERLAP on the GPU (different
 * streams, or graph branches without a dependency between them) race on it and must be serialised
 * by the caller; calls in one stream are ordered and safe.  The array keeps the last call's
 * contents; every element a call reads it has written itself first, so nothing needs clearing.
 * Errors as for sphericart_cuda_vjp (EINVAL, EALIGN, ECUDA); n = 0 is a no-op.
 */
#define SPHERICART_CUDA_NOALLOC_MAX_POINTS 32768
#define SPHERICART_CUDA_NOALLOC_SCRATCH_BYTES (32768u * 8u * 3u * 8u)
int sphericart_cuda_vjp_noalloc(const void* dsph, const void* grad_sph, void* grad_xyz, int64_t n, int l_max,
                                int dtype, void* stream);

/* Message for the last non-zero return on the calling thread ("" if none).  Never NULL. */
const char* sphericart_cuda_last_error(void);

/* Number of kernels this library has launched in this process (all threads); for harnesses. */
int64_t sphericart_cuda_launch_count(void);

/* Name of the kernel family the calling thread's last launch used ("tpb", "tq", "tpg", "w", "wc",
 * "vjp", "vjp_warp", "vjpr", "tq_vjpr", "tq_vjp2", "vjpr_generic", "expand", ...; "" before the first launch).  Static
 * storage, never NULL.  For harnesses: bench.py records which kernel served each cell of its sweep. */
const char* sphericart_cuda_last_kernel(void);

/*
 * Launch options, for test harnesses and experiments only: the defaults are compiled in and
 * nothing on the call path reads the environment.  Process-wide, not synchronised with concurrent
 * calls.  Returns 0, or SPHERICART_CUDA_EINVAL for an unknown name or value.
 *   "force_kernel"      "" | "auto" (default dispatch) | "tpb" | "tq" | "tv" | "tpg" | "w" | "w1" | "wc" | "generic":
 *                       restrict the dispatch to one kernel family where it applies (results are
 *                       the same function; the tests compare every family with the oracle)
 *   "host_chunk_bytes"  bytes per chunk and stream of the _host entry points (default 256 MiB)
 *   "tpg_lp", "w_nbuf", "w_warps", "w_ppw", "wc_min_l", "vjp_warps", "tpb_tiles", "tpb_split",
 *   "pdl", "tq_points", "tq_warps", "tq_batch", "tq_images", "tq_cs_warps", "tq_direct"  integer launch-shape parameters (0 = the library's own rule)
 */
int sphericart_cuda_set_option(const char* name, const char* value);

#ifdef __cplusplus
}
#endif
#endif /* SPHERICART_CUDA_H */
