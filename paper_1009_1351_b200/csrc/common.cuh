// common.cuh -- shared declarations of libtnlm (CUDA, sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tnlm {

// Ray table entry, one per (phase, view, bin); built once in tnlm_create from the geometry in
// double precision.  Both projector kernels read the SAME entry and run the SAME fp32
// expressions on it (ray_cell below), so P^T is the exact transpose of P entry by entry.
//   steep ray (|dy| >= |dx|): column coordinate xi(eta) = p0 + m*eta   (grid units, pixel c = [c,c+1))
//   shallow ray             : row    coordinate eta(xi) = p0 + m*xi
//   plo  = p0 + min(m, 0): the smaller of the two coordinates at which the ray enters / leaves
//          row (column) q is lo(q) = m*q + plo; the larger one is lo + |m| <= lo + 1
//   len  = length of the ray inside one full row (steep, stored > 0) / column (shallow, stored < 0), mm
//   inva = 1/|m| (1e30 if m == 0)
struct __align__(16) RayEntry {
    float plo, m, len, inva;
};
struct __align__(8) RayRange {
    short lo, hi;      // inclusive range of rows (steep) / columns (shallow) to walk; empty if hi < lo
    short ilo, ihi;    // sub-range in which both touched cells are certainly inside the image (no bounds tests);
                       // empty if ihi < ilo
};

struct Geom {
    int nx, ny, n_phase, n_views, n_bins;
    float pix;                 // mm
    float sdd_over_pitch;      // bins per radian of fan angle
    float bin_centre;          // (B-1)/2 - bin_offset
    float hw_scale;            // 1.02 * (pix/sqrt(2)) * sdd_over_pitch: half-width of a pixel in bins x distance
};

// floor() of |x| < 2^22 without the conversion unit: round-down add of 1.5*2^23 leaves floor(x)
// in the low mantissa bits (FADD.RM on the FP32 pipe; FRND/F2I would go to the 16-lane XU pipe).
constexpr float FLOOR_MAGIC = 12582912.0f;
constexpr int FLOOR_MAGIC_BITS = 0x4B400000;

// One row (steep) or column (shallow) of one ray: the at most two cells it touches there and the
// lengths inside them.  qf = row index (steep) / column index (shallow) as a float.  Returns c0 (the
// cell holding the smaller coordinate; the other cell, if any, is c0+1) and w0, w1 (mm); w1 == 0
// when the ray stays in one cell.  The split is at the cell boundary b = c0+1: the fraction of the
// crossing below b is sat((b - lo)/|m|), which is 1 when the ray does not reach b.  Explicit
// intrinsics: no contraction differences between the two kernels that inline this.
__device__ __forceinline__ void ray_cell_f(const float plo, const float m, const float alen, const float inva,
                                           const float qf, float &f0r, float &f0, float &w0, float &w1)
{
    const float lo = __fmaf_rn(m, qf, plo);
    f0r = __fadd_rd(lo, FLOOR_MAGIC);                                  // bits: FLOOR_MAGIC_BITS + floor(lo)
    f0 = __fsub_rn(f0r, FLOOR_MAGIC);                                  // floor(lo) as a float, exactly
    const float t = __fsub_rn(f0, lo);                                 // floor(lo) - lo in (-1, 0]
    const float frac = __saturatef(__fmaf_rn(t, inva, inva));          // ((c0+1) - lo)/|m|, clamped
    w0 = __fmul_rn(alen, frac);
    w1 = __fsub_rn(alen, w0);
}
__device__ __forceinline__ void ray_cell(const float plo, const float m, const float alen, const float inva,
                                         const float qf, int &c0, float &w0, float &w1)
{
    float f0r, f0;
    ray_cell_f(plo, m, alen, inva, qf, f0r, f0, w0, w1);
    c0 = __float_as_int(f0r) - FLOOR_MAGIC_BITS;
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// FP32 (non-tensor) peak probe: 8 independent FFMA chains per thread, fully unrolled inner block, so the
// loop overhead is < 2 %.  The roofline denominator of the ALU-bound kernels is measured with this on the
// box the benchmark runs on (MEASURED_PEAKS.json has no FP32 figure).
__global__ void __launch_bounds__(256)
fp32_probe_kernel(float *out, float a, float b, int iters)
{
    float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    const float s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 1234.5678f) out[0] = s;       // never true for the arguments used; keeps the chains alive
}

}  // namespace tnlm
