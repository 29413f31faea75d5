// common.cuh -- shared declarations of libtnlm (CUDA, sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tnlm {

// Ray table entry, one per (phase, view, bin); built once in tnlm_create from the geometry in
// double precision.  Both projector kernels read the SAME entry and run the SAME fp32
// expressions on it (ray_cum below), so P^T is the exact transpose of P entry by entry.
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
    float hw_scale;            // 1.02 * widening * pix * sdd_over_pitch (tnlm_create): candidate half-width of the backprojector per pixel of half-side
};

// floor() of |x| < 2^22 without the conversion unit: round-down add of 1.5*2^23 leaves floor(x)
// in the low mantissa bits (FADD.RM on the FP32 pipe; FRND/F2I would go to the 16-lane XU pipe).
constexpr float FLOOR_MAGIC = 12582912.0f;
constexpr int FLOOR_MAGIC_BITS = 0x4B400000;

// One row (steep) or column (shallow) q of one ray crosses the minor axis over [lo, lo + |m|], |m| <= 1,
// lo = m*q + plo, so it touches at most the two cells c0 = floor(lo) and c0 + 1.  With the cumulative
// fraction of the crossing that lies below coordinate b,
//     F(b) = sat( ((b - 1) - lo) * inva + inva ),          inva = 1/|m|   (1e30 for m = 0: a step function)
// the CANONICAL matrix entry both projectors produce is
//     P[ray, (q, c)] = fl( alen * fl( F(c+1) - F(c) ) ),    alen = length of the ray inside one full row (mm).
// F is exactly 0 for b <= c0 and exactly 1 for b >= c0 + 2, so only F(c0 + 1) is fractional: the forward
// projector evaluates just that one (ray_frac: F1 and U1 = 1 - F1 are the fractions of cells c0 and c0 + 1),
// the gather evaluates F at the three boundaries of its two pixels with the SAME expression (ray_cum), and
// every entry is bit-identical on the two sides: P^T is the exact transpose of P.
// Explicit intrinsics: no contraction differences between the two kernels that inline these.
__device__ __forceinline__ float ray_lo(const float plo, const float m, const float qf) { return __fmaf_rn(m, qf, plo); }
__device__ __forceinline__ float ray_cum(const float bm1, const float lo, const float inva)
{
    return __saturatef(__fmaf_rn(__fsub_rn(bm1, lo), inva, inva));
}
__device__ __forceinline__ void ray_frac(const float plo, const float m, const float inva, const float qf, int &c0,
                                         float &F1, float &U1)
{
    const float lo = ray_lo(plo, m, qf);
    const float f0r = __fadd_rd(lo, FLOOR_MAGIC);                      // bits: FLOOR_MAGIC_BITS + floor(lo)
    const float f0 = __fsub_rn(f0r, FLOOR_MAGIC);                      // floor(lo) as a float, exactly
    F1 = ray_cum(f0, lo, inva);                                        // F(c0 + 1)
    U1 = __fsub_rn(1.0f, F1);                                          // F(c0 + 2) - F(c0 + 1)
    c0 = __float_as_int(f0r) - FLOOR_MAGIC_BITS;
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// ---- cp.async (LDGSTS): global -> shared copies that hold no registers while in flight -----------------
// 4-byte copy; `valid` false writes 0.0f instead (src-size 0: nothing is read).
__device__ __forceinline__ void cp_async4_zfill(void *dst, const void *src, bool valid)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(valid ? 4 : 0) : "memory");
}
// 16-byte copy; `valid` false writes 16 zero bytes instead
__device__ __forceinline__ void cp_async16_zfill(void *dst, const void *src, bool valid)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(valid ? 16 : 0) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
// the same with a 32-bit shared-window address (no generic -> shared conversion per copy)
__device__ __forceinline__ void cp_async16_s(unsigned dst_s, const void *src, bool pred)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q cp.async.cg.shared.global [%0], [%1], 16;\n}" ::"r"(dst_s), "l"(src), "r"((int)pred) : "memory");
}
// L2 eviction-priority policies (createpolicy) and accesses that carry one: the part of a re-read stream that
// fits in L2 is marked evict_last and stays there between kernels, the rest is marked evict_first.
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void cp_async16_s_hint(unsigned dst_s, const void *src, bool pred, uint64_t pol)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %3;\n}" ::"r"(dst_s), "l"(src), "r"((int)pred), "l"(pol) : "memory");
}
__device__ __forceinline__ void stg128_hint(void *dst, const uint4 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(dst), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ uint4 lds128_s(unsigned addr_s)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr_s));
    return v;
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

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
