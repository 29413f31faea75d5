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
//   len  = length of the ray inside one full row (steep) / column (shallow), in mm
//   inva = 1/|m| (0 if m == 0)
//   flag : bit0 = steep; lo/hi = inclusive range of rows (steep) / columns (shallow) to walk
struct __align__(16) RayEntry {
    float p0, m, len, inva;
};
struct __align__(8) RayRange {
    short lo, hi;      // empty if hi < lo
    int steep;
};

struct Geom {
    int nx, ny, n_phase, n_views, n_bins;
    float pix;                 // mm
    float sdd_over_pitch;      // bins per radian of fan angle
    float bin_centre;          // (B-1)/2 - bin_offset
    float half_diag;           // pix/sqrt(2) mm
};

// One row (steep) or column (shallow) of one ray: the at most two cells it touches there and
// the lengths inside them.  q = row index (steep) / column index (shallow).
// Returns c0,c1 (cell indices along the other axis; c1 >= c0) and w0,w1 (mm).  When the ray
// stays in one cell, c1 == c0 and w1 == 0.  Explicit intrinsics: no contraction differences
// between the two kernels that inline this.
__device__ __forceinline__ void ray_cell(const RayEntry e, int q, int &c0, int &c1, float &w0, float &w1)
{
    const float fq = (float)q;
    const float xa = __fmaf_rn(e.m, fq, e.p0);
    const float xb = __fmaf_rn(e.m, fq + 1.0f, e.p0);
    const float lo = fminf(xa, xb), hi = fmaxf(xa, xb);
    const float f0 = floorf(lo), f1 = floorf(hi);
    c0 = (int)f0;
    c1 = (int)f1;
    float frac = 1.0f;
    if (f1 > f0) frac = __saturatef(__fmul_rn(__fsub_rn(f1, lo), e.inva));
    w0 = __fmul_rn(e.len, frac);
    w1 = __fsub_rn(e.len, w0);
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace tnlm
