// Launch shapes of the tq kernel (kernel_tq.cuh), and where the default dispatch uses it.
//
// TQ_SHAPE[f64][deriv][l_max] = {B, P, W, N}: points per phase-A batch, points per tile, warps per
// CTA, staging images per CTA; {B, 0, W, 0 | 4}: the DIRECT variant (no staging image, phase B stores
// straight to global memory; two points per lane and (l, m), or four where the last field is 4); {0,0,0,0}: another kernel family is at least as fast there (tpb,
// tpg, w, wc), so the dispatch does not pick tq.  Measured on one B200 (1965 MHz): every cell of
// (f32 | f64) x (values | + gradients | + Hessians) x l_max = 5..32 was timed with the default
// dispatch's other kernels and with tq forced over B in {32,16,8} x P in {2,4,8} x W in {3..8} x N in {2,1}
// (normalised harmonics, xyz ~ N(0,1), ~1.5 GB of output per call, CUDA events over 4-5 calls); an
// entry is set where the best tq shape beat the default by more than 3 %.  Second pass (l_max >= 11):
// W in {8,10,12,14,16} for the staged shapes and B in {32,16,8} x W in {3..8,10,12,14,16} for DIRECT,
// an entry replaced where the new shape beat the first pass's by more than 3 %.
// Third pass: DIRECT with two and four points per lane over B in {32,16,8} x W in {2..6,8,10,12,16}, same rule.
// Fourth pass (f32 V+G+H through an image, after its work items were flattened): l_max 7 and 10 re-measured.
// f64 V+G+H from l_max = 23: left to the warp-per-point (23) and CTA-per-point (24-32) kernels (kernel_w.cuh,
// kernel_wc.cuh), which win there once a call has >= 256 points per SM (4.3-6.0 TB/s against 3.7-4.4; at 64 points
// per SM, the size of the first passes, they lost).
#pragma once

namespace sphb200 {

static const unsigned char TQ_SHAPE[2][3][33][4] = {
  {
    /* f32 V */ {{0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}},
    /* f32 V+G */ {{0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {16,0,4,0}, {16,0,4,4}, {16,0,4,4}, {32,0,4,0}, {16,0,4,0}, {32,0,6,0}, {32,0,6,0}, {32,0,4,0}, {32,0,8,0}, {32,0,8,0}, {32,0,4,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}, {32,0,8,0}},
    /* f32 V+G+H */ {{0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {16,8,2,1}, {32,8,3,1}, {32,8,4,1}, {16,8,4,1}, {16,8,5,1}, {8,4,3,1}, {16,4,3,1}, {8,4,4,1}, {16,4,4,1}, {8,2,3,1}, {16,4,6,1}, {8,2,3,1}, {16,4,6,1}, {8,2,4,1}, {8,2,4,1}, {16,2,8,1}, {16,2,5,1}, {32,2,10,2}, {16,2,12,2}, {16,2,12,2}, {16,2,12,2}, {32,0,4,0}, {32,0,4,0}, {32,0,4,0}, {32,0,4,0}, {32,0,4,0}, {32,0,3,0}},
  },
  {
    /* f64 V */ {{0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {16,0,4,4}, {0,0,0,0}, {0,0,0,0}, {32,0,8,0}, {32,0,8,4}, {0,0,0,0}, {16,0,5,0}, {0,0,0,0}, {16,0,5,0}, {0,0,0,0}, {8,0,4,0}},
    /* f64 V+G */ {{0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {32,8,4,1}, {32,8,4,1}, {16,8,3,1}, {16,4,3,1}, {32,4,4,1}, {16,4,4,1}, {16,4,4,1}, {16,2,3,1}, {16,4,4,1}, {16,4,4,1}, {8,2,3,1}, {8,2,4,1}, {8,2,4,1}, {16,2,4,1}, {16,4,6,1}, {8,2,4,1}, {8,2,4,1}, {8,2,4,1}, {16,2,6,1}, {32,2,8,2}, {8,2,7,1}, {8,2,8,1}, {8,2,8,1}, {16,0,8,0}, {16,0,8,0}},
    /* f64 V+G+H */ {{0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {16,8,2,1}, {32,8,4,1}, {16,4,2,1}, {32,4,4,1}, {8,2,2,1}, {16,2,3,1}, {8,2,3,1}, {16,2,3,1}, {8,2,4,1}, {16,2,4,1}, {8,2,5,1}, {16,2,6,1}, {16,2,6,1}, {16,2,6,1}, {8,2,7,1}, {8,2,8,2}, {32,2,8,1}, {32,2,12,2}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}, {0,0,0,0}},
  },
};

// Launch shapes of the values-only kernel (kernel_tv.cuh), and where the default dispatch uses it:
// TV_SHAPE[f64][l_max] = {B, W, C}: points per batch, warps per CTA, warps that run Eq. 9 only (f64);
// {0,0,0}: another family is at least as fast.  Same protocol as above, l_max = 10..32, over
// B in {32,16,8} x W in {4,6,8} x C in {1,2}; re-measured over W in {2..6,8,10,12} after the kernel's image became
// contiguous for odd L (one bulk store per batch).
static const unsigned char TV_SHAPE[2][33][3] = {
    /* f32 */ {{0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {16,3,1}, {16,4,1}, {8,2,1}, {16,5,1}, {16,4,1}, {16,5,1}, {8,3,1}, {8,3,1}, {8,3,1}, {16,5,1}, {8,3,1}, {8,3,1}, {8,3,1}, {8,3,1}},
    /* f64 */ {{0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {0,0,0}, {32,4,1}, {32,5,1}, {32,5,1}, {16,3,1}, {16,4,1}, {16,4,1}, {16,4,1}, {16,4,1}, {16,5,1}, {16,5,1}, {16,6,2}, {8,3,1}, {16,6,2}, {16,6,2}, {16,6,2}, {16,6,1}, {8,4,1}, {8,4,1}, {8,4,1}, {8,4,1}, {8,6,1}},
};

}  // namespace sphb200
