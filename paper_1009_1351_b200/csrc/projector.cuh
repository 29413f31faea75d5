// projector.cuh -- fan-beam forward projector P (ray-driven, one thread per (view,bin)) and its
// matched adjoint P^T (pixel-driven gather, one thread per 2 x 2 pixel block).  PAPER.md:L75, L79, L212.
// The slices of a batch share the ray geometry: up to 16 slices per thread in the adjoint, groups of 4 slices
// interleaved per pixel in the forward projector (project_il_kernel).
// Both kernels evaluate tnlm::ray_cum on the same RayEntry table, so every matrix entry
// len(ray ∩ pixel) is bit-identical on the two sides and P^T is the exact transpose of P (common.cuh).
#pragma once
#include <type_traits>

#include "common.cuh"

namespace tnlm {

#ifndef TNLM_BP_UNROLL
#define TNLM_BP_UNROLL 2
#endif
constexpr int BP_UNROLL = TNLM_BP_UNROLL;
#ifndef TNLM_FP_UNROLL
#define TNLM_FP_UNROLL 4
#endif
constexpr int FP_UNROLL = TNLM_FP_UNROLL;   // rows per unrolled body of the forward projector's interior loop   // candidates per unrolled body of the backprojector's inner loop

enum FwdMode {
    FWD_PLAIN = 0,  // out0 = P img
    FWD_RESID = 1,  // out0 = sw*(y - P img) = r ; out1 = sw*r            (CGLS init, L109)
    FWD_SCALE = 2   // out0 = sw*(P img) = q ; red += ||q||^2             (CGLS step 1, L112)
                    // sw = sqrt(w), the diagonal of Sigma^-1/2 (L103), precomputed (NULL = 1)
};

// atan on the fan-angle range: odd minimax polynomial on [-1, 1] (Abramowitz & Stegun 4.4.49,
// |error| <= 2e-8 rad, i.e. < 1e-4 bin); detectors wider than +-40 degrees use atanf (kernel
// template POLY = false).  Only the conservative candidate range of the backprojector depends on
// it; membership and lengths come from ray_cum.
__device__ __forceinline__ float fan_angle_poly(float t)
{
    const float z = t * t;
    float p = 0.0028662257f;
    p = fmaf(p, z, -0.0161657367f);
    p = fmaf(p, z, 0.0429096138f);
    p = fmaf(p, z, -0.0752896400f);
    p = fmaf(p, z, 0.1065626393f);
    p = fmaf(p, z, -0.1420889944f);
    p = fmaf(p, z, 0.1999355085f);
    p = fmaf(p, z, -0.3333314528f);
    return fmaf(p * z, t, t);
}

// ------------------------------------------------------------------------------ forward
// grid = (ceil(V*B/256), S*N); block = 256.  Adjacent threads = adjacent bins of a view, so a
// warp walks neighbouring pixels of the same image rows (coalesced, L1-resident gathers).
// imgT[prob][c][r] = img[prob][r][c]: shallow rays walk columns, and 32 neighbouring bins of a warp
// sit in ~18 different image rows there (18 cache lines per load); in the transposed copy they are
// neighbours again.  grid = (ceil(nx/32), ceil(ny/32), S*N), block = (32, 8).
__global__ void __launch_bounds__(256)
transpose_kernel(const float *__restrict__ img, float *__restrict__ imgT, int nx, int ny, int prob0)
{
    __shared__ float tile[32][33];
    const size_t base = (size_t)(blockIdx.z + prob0) * nx * ny;
    const int c = blockIdx.x * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int r = blockIdx.y * 32 + threadIdx.y + j;
        tile[threadIdx.y + j][threadIdx.x] = (r < ny && c < nx) ? __ldg(img + base + (size_t)r * nx + c) : 0.f;
    }
    __syncthreads();
    const int rT = blockIdx.y * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int cT = blockIdx.x * 32 + threadIdx.y + j;
        if (rT < ny && cT < nx) imgT[base + (size_t)cT * ny + rT] = tile[threadIdx.x][threadIdx.y + j];
    }
}

// NS slices of the batch share one thread: the slices of a batch have the same geometry (nothing
// couples them, and the gantry does not know about slices), so the walk of a ray -- ray_frac per row -- is done
// once and only the two loads and two FMAs per row are per slice (6 + 4 NS instructions per row instead of 10 NS,
// and 2 NS independent gathers in flight).  Per slice the arithmetic and its order are those of NS = 1.
// grid = (ceil(V*B/256), groups*N), group g = slices slice0 + g*NS .. + NS-1.
template <int MODE, int NS>
__global__ void __launch_bounds__(256)
project_kernel(Geom G, const RayEntry *__restrict__ tab, const RayRange *__restrict__ rng,
               const float *__restrict__ img, const float *__restrict__ imgT, const float *__restrict__ y,
               const float *__restrict__ sw_, float *__restrict__ out0, float *__restrict__ out1,
               double *__restrict__ red, int slice0)
{
    const int phase = blockIdx.y % G.n_phase;
    const int prob = (slice0 + (blockIdx.y / G.n_phase) * NS) * G.n_phase + phase;   // slice*N + phase of the group's first slice
    const int nray = G.n_views * G.n_bins;
    const size_t img_stride = (size_t)G.n_phase * G.nx * G.ny, sino_stride = (size_t)G.n_phase * nray;   // per slice
    const int ray = blockIdx.x * blockDim.x + threadIdx.x;
    float qq[NS];
#pragma unroll
    for (int s = 0; s < NS; ++s) qq[s] = 0.f;
    if (ray < nray) {
        const RayEntry e = tab[(size_t)phase * nray + ray];
        const RayRange rg = rng[(size_t)phase * nray + ray];
        const float alen = fabsf(e.len);
        float acc0[NS], acc1[NS];                              // sums of fraction x pixel value; x alen once at the end
#pragma unroll
        for (int s = 0; s < NS; ++s) { acc0[s] = 0.f; acc1[s] = 0.f; }
        // steep rays walk the rows of the image, shallow rays the rows of the transposed image
        const bool steep = e.len > 0.f;
        const int n_minor = steep ? G.nx : G.ny;             // length of a walked row
        const float *__restrict__ base = (steep ? img : imgT) + (size_t)prob * G.nx * G.ny;
        auto edge = [&](int q0, int q1) {                      // rows in which a touched cell may be outside
            float qf = (float)q0;
            const float *__restrict__ row = base + (size_t)q0 * n_minor;
            for (int q = q0; q <= q1; ++q, qf += 1.0f, row += n_minor) {
                int c0; float F1, U1;
                ray_frac(e.plo, e.m, e.inva, qf, c0, F1, U1);
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    if ((unsigned)c0 < (unsigned)n_minor) acc0[s] = fmaf(F1, __ldg(row + s * img_stride + c0), acc0[s]);
                    if ((unsigned)(c0 + 1) < (unsigned)n_minor) acc1[s] = fmaf(U1, __ldg(row + s * img_stride + c0 + 1), acc1[s]);
                }
            }
        };
        if (rg.ihi >= rg.ilo) {
            edge(rg.lo, rg.ilo - 1);
            float qf = (float)rg.ilo;
            const float *__restrict__ row = base + (size_t)rg.ilo * n_minor;
#pragma unroll (NS == 1 ? FP_UNROLL : (NS == 2 ? 2 : 1))
            for (int q = rg.ilo; q <= rg.ihi; ++q, qf += 1.0f, row += n_minor) {
                int c0; float F1, U1;
                ray_frac(e.plo, e.m, e.inva, qf, c0, F1, U1);
                const float *__restrict__ cell = row + c0;
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    acc0[s] = fmaf(F1, __ldg(cell + s * img_stride), acc0[s]);
                    acc1[s] = fmaf(U1, __ldg(cell + s * img_stride + 1), acc1[s]);
                }
            }
            edge(rg.ihi + 1, rg.hi);
        } else {
            edge(rg.lo, rg.hi);
        }
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const float p = __fmul_rn(alen, acc0[s] + acc1[s]);
            const size_t o = (size_t)prob * nray + s * sino_stride + ray;
            if (MODE == FWD_PLAIN) {
                out0[o] = p;
            } else {
                const float sw = sw_ ? sw_[o] : 1.0f;
                if (MODE == FWD_RESID) {
                    const float r = sw * (y[o] - p);
                    out0[o] = r;
                    out1[o] = sw * r;
                } else {
                    const float q = sw * p;
                    out0[o] = q;
                    qq[s] = q * q;
                }
            }
        }
    }
    if (MODE == FWD_SCALE) {
        __shared__ float part[NS][8];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const float v = warp_sum(qq[s]);
            if ((threadIdx.x & 31) == 0) part[s][threadIdx.x >> 5] = v;
        }
        __syncthreads();
        // warp w sums slices w, w + warps, ...: a CTA of 64 threads (project_block = 64) has fewer warps than NS = 4 slices
        const int nwarp = (int)(blockDim.x >> 5), l = threadIdx.x & 31;
        for (int s = threadIdx.x >> 5; s < NS; s += nwarp) {
            float v = l < nwarp ? part[s][l] : 0.f;
            v = warp_sum(v);
            if (l == 0) atomicAdd(red + prob + s * G.n_phase, (double)v);
        }
    }
}

// ---- four slices interleaved per pixel -------------------------------------------------------------------------
// project_kernel is bound by the load/store unit: two 32-lane gathers per (ray, row), ~1.8 cycles of LSU issue each
// per SM whatever the width of the load.  For a batch the projector therefore reads copies of the image in which
// the four slices of a group sit side by side per pixel, imI[group][phase][r][c] = (slice 4g .. 4g+3) as one float4
// and the same transposed (imTI[group][phase][c][r]): one LDG.128 per cell serves four slices, i.e. half a gather
// per (ray, row, slice) instead of two, and the ray walk (ray_frac) is shared as in project_kernel<., NS>.  Per
// slice the arithmetic and its order are unchanged (bit-identical results).  The copies are made by
// interleave4_kernel for the first P of a call and by cgls_update_us_il afterwards.
// grid = (ceil(nx/32), ceil(ny/32), groups*N), block = (32, 8).
__global__ void __launch_bounds__(256)
interleave4_kernel(const float *__restrict__ img, float4 *__restrict__ imI, float4 *__restrict__ imTI, int nx, int ny,
                   int n_phase)
{
    __shared__ float4 tile[32][33];
    const int group = blockIdx.z / n_phase, phase = blockIdx.z - group * n_phase;
    const size_t npix = (size_t)nx * ny, sl = (size_t)n_phase * npix;                 // slice stride
    const float *__restrict__ src = img + ((size_t)group * 4 * n_phase + phase) * npix;
    const size_t base4 = ((size_t)group * n_phase + phase) * npix;
    const int c = blockIdx.x * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int r = blockIdx.y * 32 + threadIdx.y + j;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (r < ny && c < nx) {
            const size_t o = (size_t)r * nx + c;
            v = make_float4(__ldg(src + o), __ldg(src + sl + o), __ldg(src + 2 * sl + o), __ldg(src + 3 * sl + o));
            imI[base4 + o] = v;
        }
        tile[threadIdx.y + j][threadIdx.x] = v;
    }
    __syncthreads();
    const int rT = blockIdx.y * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int cT = blockIdx.x * 32 + threadIdx.y + j;
        if (rT < ny && cT < nx) imTI[base4 + (size_t)cT * ny + rT] = tile[threadIdx.x][threadIdx.y + j];
    }
}

// grid = (ceil(V*B/256), groups*N); group g = slices 4g .. 4g+3 (the groups start at slice 0).
template <int MODE>
__global__ void __launch_bounds__(256)
project_il_kernel(Geom G, const RayEntry *__restrict__ tab, const RayRange *__restrict__ rng,
                  const float4 *__restrict__ imI, const float4 *__restrict__ imTI, const float *__restrict__ y,
                  const float *__restrict__ sw_, float *__restrict__ out0, float *__restrict__ out1,
                  double *__restrict__ red)
{
    constexpr int NS = 4;
    const int group = blockIdx.y / G.n_phase, phase = blockIdx.y - group * G.n_phase;
    const int prob = group * NS * G.n_phase + phase;         // slice*N + phase of the group's first slice
    const int nray = G.n_views * G.n_bins;
    const size_t sino_stride = (size_t)G.n_phase * nray;     // per slice
    const int ray = blockIdx.x * blockDim.x + threadIdx.x;
    float qq[NS] = {0.f, 0.f, 0.f, 0.f};
    if (ray < nray) {
        const RayEntry e = tab[(size_t)phase * nray + ray];
        const RayRange rg = rng[(size_t)phase * nray + ray];
        const float alen = fabsf(e.len);
        float acc0[NS] = {0.f, 0.f, 0.f, 0.f}, acc1[NS] = {0.f, 0.f, 0.f, 0.f};
        const bool steep = e.len > 0.f;
        const int n_minor = steep ? G.nx : G.ny;
        const float4 *__restrict__ base = (steep ? imI : imTI) + ((size_t)group * G.n_phase + phase) * G.nx * G.ny;
        auto edge = [&](int q0, int q1) {                      // rows in which a touched cell may be outside
            float qf = (float)q0;
            const float4 *__restrict__ row = base + (size_t)q0 * n_minor;
            for (int q = q0; q <= q1; ++q, qf += 1.0f, row += n_minor) {
                int c0; float F1, U1;
                ray_frac(e.plo, e.m, e.inva, qf, c0, F1, U1);
                if ((unsigned)c0 < (unsigned)n_minor) {
                    const float4 v = __ldg(row + c0);
                    acc0[0] = fmaf(F1, v.x, acc0[0]); acc0[1] = fmaf(F1, v.y, acc0[1]);
                    acc0[2] = fmaf(F1, v.z, acc0[2]); acc0[3] = fmaf(F1, v.w, acc0[3]);
                }
                if ((unsigned)(c0 + 1) < (unsigned)n_minor) {
                    const float4 v = __ldg(row + c0 + 1);
                    acc1[0] = fmaf(U1, v.x, acc1[0]); acc1[1] = fmaf(U1, v.y, acc1[1]);
                    acc1[2] = fmaf(U1, v.z, acc1[2]); acc1[3] = fmaf(U1, v.w, acc1[3]);
                }
            }
        };
        if (rg.ihi >= rg.ilo) {
            edge(rg.lo, rg.ilo - 1);
            float qf = (float)rg.ilo;
            const float4 *__restrict__ row = base + (size_t)rg.ilo * n_minor;
#pragma unroll 2
            for (int q = rg.ilo; q <= rg.ihi; ++q, qf += 1.0f, row += n_minor) {
                int c0; float F1, U1;
                ray_frac(e.plo, e.m, e.inva, qf, c0, F1, U1);
                const float4 v0 = __ldg(row + c0), v1 = __ldg(row + c0 + 1);
                acc0[0] = fmaf(F1, v0.x, acc0[0]); acc0[1] = fmaf(F1, v0.y, acc0[1]);
                acc0[2] = fmaf(F1, v0.z, acc0[2]); acc0[3] = fmaf(F1, v0.w, acc0[3]);
                acc1[0] = fmaf(U1, v1.x, acc1[0]); acc1[1] = fmaf(U1, v1.y, acc1[1]);
                acc1[2] = fmaf(U1, v1.z, acc1[2]); acc1[3] = fmaf(U1, v1.w, acc1[3]);
            }
            edge(rg.ihi + 1, rg.hi);
        } else {
            edge(rg.lo, rg.hi);
        }
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const float p = __fmul_rn(alen, acc0[s] + acc1[s]);
            const size_t o = (size_t)prob * nray + s * sino_stride + ray;
            if (MODE == FWD_PLAIN) {
                out0[o] = p;
            } else {
                const float sw = sw_ ? sw_[o] : 1.0f;
                if (MODE == FWD_RESID) {
                    const float r = sw * (y[o] - p);
                    out0[o] = r;
                    out1[o] = sw * r;
                } else {
                    const float q = sw * p;
                    out0[o] = q;
                    qq[s] = q * q;
                }
            }
        }
    }
    if (MODE == FWD_SCALE) {
        __shared__ float part[NS][8];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const float v = warp_sum(qq[s]);
            if ((threadIdx.x & 31) == 0) part[s][threadIdx.x >> 5] = v;
        }
        __syncthreads();
        // warp w sums slices w, w + warps, ...: a CTA of 64 threads (project_block = 64) has fewer warps than NS = 4 slices
        const int nwarp = (int)(blockDim.x >> 5), l = threadIdx.x & 31;
        for (int s = threadIdx.x >> 5; s < NS; s += nwarp) {
            float v = l < nwarp ? part[s][l] : 0.f;
            v = warp_sum(v);
            if (l == 0) atomicAdd(red + prob + s * G.n_phase, (double)v);
        }
    }
}

// The same projector with the gathers served from shared memory.  ncu on project_kernel: 51 % issue-active,
// 19 long-scoreboard stall cycles per issue, L1TEX 60-88 % busy: two 32-lane gathers per row, each touching two or
// three sectors of one or two lines, are what it waits for.  Here a WARP owns 32 neighbouring bins of one view and
// walks its rows in chunks of PS_R: for a chunk it works out the columns its rays touch (lo is linear in the row,
// so the extremes are at the chunk's ends), stages that strip (<= PS_W columns, 16-byte cp.async, zero-filled
// outside the image so that no bounds test is left in the inner loop) in its private shared-memory slot and reads
// both cells of every row with conflict-free LDS.  The arithmetic and its order are those of project_kernel, so
// the result is bit-identical and P^T stays the exact transpose.  A warp whose rays are not all steep or all
// shallow (one per view at most), an image whose rows are not 16-byte aligned, or a chunk wider than PS_W
// columns takes the gather path.  grid = (ceil(V * ceil(B/32) / PS_WARPS), S*N); block = 32 * PS_WARPS.
constexpr int PS_R = 16;        // rows per staged chunk
constexpr int PS_W = 64;        // columns per strip row
constexpr int PS_WARPS = 8;

template <int MODE>
__global__ void __launch_bounds__(32 * PS_WARPS)
project_strip_kernel(Geom G, const RayEntry *__restrict__ tab, const RayRange *__restrict__ rng,
                     const float *__restrict__ img, const float *__restrict__ imgT, const float *__restrict__ y,
                     const float *__restrict__ sw_, float *__restrict__ out0, float *__restrict__ out1,
                     double *__restrict__ red)
{
    __shared__ __align__(16) float strip_all[PS_WARPS][PS_R * PS_W];
    const int prob = blockIdx.y;                 // slice*N + phase
    const int phase = prob % G.n_phase;
    const int V = G.n_views, B = G.n_bins, nray = V * B;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WB = (B + 31) >> 5;                // warp tasks per view
    const int task = blockIdx.x * PS_WARPS + warp;
    const int v = task / WB, k = (task - v * WB) * 32 + lane;
    const bool valid = (v < V) && (k < B);
    const int ray = v * B + k;
    float *__restrict__ strip = strip_all[warp];
    float qq = 0.f;
    RayEntry e = {0.f, 0.f, 1.f, 1.f};
    RayRange rg = {1, 0, 1, 0};
    if (valid) {
        e = tab[(size_t)phase * nray + ray];
        rg = rng[(size_t)phase * nray + ray];
    }
    const bool active = valid && rg.hi >= rg.lo;
    const bool steep = e.len > 0.f;
    const unsigned m_act = __ballot_sync(0xffffffffu, active), m_steep = __ballot_sync(0xffffffffu, active && steep);
    const bool uniform = (m_steep == m_act) || (m_steep == 0u);
    const bool steep_w = m_steep != 0u;
    const int n_minor_w = steep_w ? G.nx : G.ny, n_major_w = steep_w ? G.ny : G.nx;
    const float *__restrict__ base_w = (steep_w ? img : imgT) + (size_t)prob * G.nx * G.ny;
    const bool can_stage = uniform && ((n_minor_w & 3) == 0) && ((reinterpret_cast<uintptr_t>(base_w) & 15) == 0);
    float acc0 = 0.f, acc1 = 0.f;                // sums of fraction x pixel value; x alen once at the end
    // rows [q0, q1] of this lane's ray by gathers from global memory (bounds-tested)
    auto gather = [&](int q0, int q1) {
        const int n_minor = steep ? G.nx : G.ny;
        const float *__restrict__ row = (steep ? img : imgT) + (size_t)prob * G.nx * G.ny + (size_t)q0 * n_minor;
        float qf = (float)q0;
        for (int q = q0; q <= q1; ++q, qf += 1.0f, row += n_minor) {
            int c0; float F1, U1;
            ray_frac(e.plo, e.m, e.inva, qf, c0, F1, U1);
            if ((unsigned)c0 < (unsigned)n_minor) acc0 = fmaf(F1, __ldg(row + c0), acc0);
            if ((unsigned)(c0 + 1) < (unsigned)n_minor) acc1 = fmaf(U1, __ldg(row + c0 + 1), acc1);
        }
    };
    if (!can_stage) {
        if (active) gather(rg.lo, rg.hi);
    } else if (m_act) {
        const int q_begin = __reduce_min_sync(0xffffffffu, active ? (int)rg.lo : 0x7fffffff);
        const int q_end = __reduce_max_sync(0xffffffffu, active ? (int)rg.hi : -1);
        for (int qa = q_begin; qa <= q_end; qa += PS_R) {
            const int qb = min(qa + PS_R - 1, q_end);
            const int my_a = max(qa, (int)rg.lo), my_b = min(qb, (int)rg.hi);
            const bool has = active && my_a <= my_b;
            // columns this lane touches in the chunk: lo is linear in the row, extremes at its two ends
            const float la = ray_lo(e.plo, e.m, (float)my_a), lb = ray_lo(e.plo, e.m, (float)my_b);
            const int cl = __float_as_int(__fadd_rd(fminf(la, lb), FLOOR_MAGIC)) - FLOOR_MAGIC_BITS;
            const int ch = __float_as_int(__fadd_rd(fmaxf(la, lb), FLOOR_MAGIC)) - FLOOR_MAGIC_BITS + 1;
            const int cmin = __reduce_min_sync(0xffffffffu, has ? cl : 0x7fffffff);
            const int cmax = __reduce_max_sync(0xffffffffu, has ? ch : (int)0x80000000);
            if (cmin > cmax) continue;                       // no lane has a row in this chunk
            const int c_al = cmin & ~3;                      // (two's complement: rounds towards -inf)
            const int ngrp = ((cmax - c_al) >> 2) + 1;       // 16-byte groups per strip row
            if (ngrp * 4 > PS_W) {                           // too wide for the slot (a very oblique geometry)
                if (has) gather(my_a, my_b);
                continue;
            }
            __syncwarp();                                    // the previous chunk is no longer read
            {   // lanes 0-15 stage the groups of one row, lanes 16-31 those of the next
                const int gi = lane & 15, c = c_al + 4 * gi;
                const bool cin = gi < ngrp && (unsigned)c < (unsigned)n_minor_w;
                for (int rr = lane >> 4; qa + rr <= qb; rr += 2) {
                    const int q = qa + rr;
                    const bool in = cin && (unsigned)q < (unsigned)n_major_w;
                    if (gi < ngrp)
                        cp_async16_zfill(strip + rr * PS_W + 4 * gi, base_w + (in ? (size_t)q * n_minor_w + c : 0), in);
                }
            }
            cp_async_commit();
            cp_async_wait<0>();
            __syncwarp();
            if (has) {
                const float *__restrict__ srow = strip + (my_a - qa) * PS_W - c_al;
                float qf = (float)my_a;
#pragma unroll 4
                for (int q = my_a; q <= my_b; ++q, qf += 1.0f, srow += PS_W) {
                    int c0; float F1, U1;
                    ray_frac(e.plo, e.m, e.inva, qf, c0, F1, U1);
                    acc0 = fmaf(F1, srow[c0], acc0);
                    acc1 = fmaf(U1, srow[c0 + 1], acc1);
                }
            }
        }
    }
    if (valid) {
        const float p = __fmul_rn(fabsf(e.len), acc0 + acc1);
        const size_t o = (size_t)prob * nray + ray;
        if (MODE == FWD_PLAIN) {
            out0[o] = p;
        } else {
            const float sw = sw_ ? sw_[o] : 1.0f;
            if (MODE == FWD_RESID) {
                const float r = sw * (y[o] - p);
                out0[o] = r;
                out1[o] = sw * r;
            } else {
                const float q = sw * p;
                out0[o] = q;
                qq = q * q;
            }
        }
    }
    if (MODE == FWD_SCALE) {
        __shared__ float part[PS_WARPS];
        qq = warp_sum(qq);
        if (lane == 0) part[warp] = qq;
        __syncthreads();
        if (threadIdx.x < 32) {
            float vv = threadIdx.x < PS_WARPS ? part[threadIdx.x] : 0.f;
            vv = warp_sum(vv);
            if (threadIdx.x == 0) atomicAdd(red + prob, (double)vv);
        }
    }
}

// ----------------------------------------------------------------------------- adjoint
// One thread per BR x BC pixel block (rows r0 .. r0+BR-1, columns c0 .. c0+BC-1; a warp covers 4 x 8 blocks, a CTA
// of 4 warps 16 x 8 blocks), loop over the views of its phase.  Per view the candidate bins are those whose fan angle
// is within the block's angular footprint (conservative superset).  A steep candidate is evaluated in the block's
// BR rows, a shallow one in its BC columns: one evaluation of a line serves all block pixels of that line with the
// cumulative fraction F (ray_cum) at their cell boundaries, so the same expressions as the forward projector decide
// membership and give the lengths (exact transpose), and the per-view work (fan angle, candidate range, the runs of
// ray classes) is shared by BR*BC pixels.
// NS slices of the batch share one thread (same geometry, see project_kernel): the candidate's ray_cum values are
// computed once, each slice adds one sinogram load, one multiply and BR*BC FMAs.
// (Accumulating slice pairs with packed f32x2 FMAs was measured and dropped: 8.3 instead of 9.2 ms for NS = 4, but
// 6.75 instead of 6.55 ms for NS = 8 on 64 slices: the FMA pipe does the same lane work either way.)
// grid = (ceil(nx/(8 BC)), ceil(ny/(16 BR)), groups*N), group g = slices slice0 + g*NS .. + NS-1; block = 128.
// red (optional) += ||out||^2 of every problem.
template <bool POLY, int NS, int BR, int BC>
__global__ void __launch_bounds__(128)
backproject_kernel(Geom G, const RayEntry *__restrict__ tab, const float4 *__restrict__ views,
                   const int4 *__restrict__ split, const float *__restrict__ sino, float *__restrict__ out,
                   double *__restrict__ red, int slice0)
{
    const int phase = blockIdx.z % G.n_phase;
    const int prob = (slice0 + (blockIdx.z / G.n_phase) * NS) * G.n_phase + phase;   // of the group's first slice
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c0 = (blockIdx.x * 8 + (lane & 7)) * BC;
    const int r0 = (blockIdx.y * 16 + warp * 4 + (lane >> 3)) * BR;
    const int V = G.n_views, B = G.n_bins;
    const size_t img_stride = (size_t)G.n_phase * G.nx * G.ny, sino_stride = (size_t)G.n_phase * V * B;   // per slice
    const bool inside = (c0 < G.nx) && (r0 < G.ny);
    float acc[NS][BR][BC];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int j = 0; j < BR; ++j)
#pragma unroll
            for (int k = 0; k < BC; ++k) acc[s][j][k] = 0.f;
    if (inside) {
        // block centre
        const float X = ((float)c0 + 0.5f * (float)(BC - 1) - 0.5f * (float)(G.nx - 1)) * G.pix;
        const float Y = ((float)r0 + 0.5f * (float)(BR - 1) - 0.5f * (float)(G.ny - 1)) * G.pix;
        const float rf = (float)r0, cf = (float)c0;
        const float4 *__restrict__ vt = views + (size_t)phase * V;
        const int4 *__restrict__ spl = split + (size_t)phase * V;
        const float4 *__restrict__ tb0 = reinterpret_cast<const float4 *>(tab + (size_t)phase * V * B);
        const float *__restrict__ sg0 = sino + (size_t)prob * V * B;
        // Candidates kb0..kb1 (offsets into the phase's table / the sinogram) of ONE class: steep rays are evaluated
        // in the block's rows, where its pixels sit at minor-axis indices c0 .. c0+BC-1; shallow rays in its columns
        // with minor-axis indices r0 .. r0+BR-1.  Pixel n of a line gets alen * (F(cA+n+1) - F(cA+n)), F = ray_cum
        // (common.cuh): zero for cells the ray misses, and bit for bit the forward projector's entry for the cells
        // it touches -- no membership test anywhere.
        auto run = [&](auto steep_c, int kb0, int kb1) {
            constexpr bool STEEP = decltype(steep_c)::value;
            constexpr int NL = STEEP ? BR : BC, NP = STEEP ? BC : BR;      // lines, pixels per line
            const float q0 = STEEP ? rf : cf, m0 = (STEEP ? cf : rf) - 1.0f;
            const float4 *__restrict__ tp = tb0 + kb0;
            const float *__restrict__ sp = sg0 + kb0;
#pragma unroll (NS == 1 && BR * BC == 4 ? BP_UNROLL : 1)
            for (int n = kb1 - kb0; n >= 0; --n, ++tp, ++sp) {
                const float4 e4 = __ldg(tp);                 // plo, m, len (sign = steep), inva
                const float alen = fabsf(e4.z);
                float d[NL][NP];
#pragma unroll
                for (int l = 0; l < NL; ++l) {
                    const float lo = ray_lo(e4.x, e4.y, q0 + (float)l);
                    float Gp = ray_cum(m0, lo, e4.w);
#pragma unroll
                    for (int n2 = 0; n2 < NP; ++n2) {
                        const float Gn = ray_cum(m0 + (float)(n2 + 1), lo, e4.w);
                        d[l][n2] = __fsub_rn(Gn, Gp);
                        Gp = Gn;
                    }
                }
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    const float asv = __fmul_rn(alen, __ldg(sp + s * sino_stride));
#pragma unroll
                    for (int j = 0; j < BR; ++j)
#pragma unroll
                        for (int k = 0; k < BC; ++k)
                            acc[s][j][k] = __fmaf_rn(asv, STEEP ? d[j][k] : d[k][j], acc[s][j][k]);
                }
            }
        };
        int vB = 0;                                          // v * B
        for (int v = 0; v < V; ++v, vB += B) {
            const float4 vw = __ldg(vt + v);                 // sx, sy, cos th, sin th
            const int4 sp = __ldg(spl + v);                  // bins [0, sp.x) and [sp.y, B) are of class sp.z (1 = steep), [sp.x, sp.y) of the other
            const float px = X - vw.x, py = Y - vw.y;
            const float dot = -(vw.z * px + vw.w * py);      // along the central ray (> 0)
            const float crs = vw.w * px - vw.z * py;         // ccw from the central ray
            float rdot;
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rdot) : "f"(dot));
            const float t = crs * rdot;
            const float kc = fmaf(POLY ? fan_angle_poly(t) : atanf(t), G.sdd_over_pitch, G.bin_centre);
            // a ray at angle D from the direction of the block centre (distance d) crosses the block (half-sides
            // hx = BC/2, hy = BR/2 pixels, half-diagonal hd) iff d*|sin D| <= h(n) = pix*(hx*|nx| + hy*|ny|), n the
            // ray's unit normal; n turns with D, |h(n) - h(n0)| <= hd*|D| with n0 = (-py, px)/d, so
            // |D| <= (h(n0)/d) / (1 - hd/d) up to the sinc term: h(n0)/d = pix*(hx*|py| + hy*|px|)/d^2 <= .../dot^2.
            // hw_scale carries pix, bins per radian, 2 % for the second-order terms and the factor 1/(1 - hd/d) at
            // the smallest d of the geometry (tnlm_create: without it a source ~15 pixels from the image lost matrix
            // entries; found by random-geometry fuzzing), + 0.05 bin of rounding
            const float hw = fmaf(G.hw_scale * (0.5f * (float)BC * fabsf(py) + 0.5f * (float)BR * fabsf(px)), rdot * rdot, 0.05f);
            const int k_lo = max(0, __float_as_int(__fadd_ru(kc - hw, FLOOR_MAGIC)) - FLOOR_MAGIC_BITS);
            const int k_hi = min(B - 1, __float_as_int(__fadd_rd(kc + hw, FLOOR_MAGIC)) - FLOOR_MAGIC_BITS);
            // the steep / shallow classes are contiguous runs of the bin index (a fan narrower than 90 degrees crosses a
            // 45-degree direction at most once, one narrower than 180 degrees at most twice): one specialised loop per
            // run, nearly always only one of them is non-empty
            const int a1 = min(k_hi, sp.x - 1), b0 = max(k_lo, sp.x), b1 = min(k_hi, sp.y - 1), c0k = max(k_lo, sp.y);
            if (sp.z) {
                run(std::true_type{}, vB + k_lo, vB + a1);
                run(std::false_type{}, vB + b0, vB + b1);
                run(std::true_type{}, vB + c0k, vB + k_hi);
            } else {
                run(std::false_type{}, vB + k_lo, vB + a1);
                run(std::true_type{}, vB + b0, vB + b1);
                run(std::false_type{}, vB + c0k, vB + k_hi);
            }
        }
        const bool full = (c0 + BC <= G.nx);
        const bool vec = full && ((G.nx & (BC - 1)) == 0) && ((reinterpret_cast<uintptr_t>(out) & (4 * BC - 1)) == 0);
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            float *__restrict__ o = out + (size_t)prob * G.nx * G.ny + s * img_stride + (size_t)r0 * G.nx + c0;
#pragma unroll
            for (int j = 0; j < BR; ++j) {
                const bool rin = r0 + j < G.ny;
                if (rin && vec) {
                    if (BC == 4) *reinterpret_cast<float4 *>(o + (size_t)j * G.nx) = make_float4(acc[s][j][0], acc[s][j][1], acc[s][j][BC > 2 ? 2 : 0], acc[s][j][BC > 3 ? 3 : 0]);
                    else *reinterpret_cast<float2 *>(o + (size_t)j * G.nx) = make_float2(acc[s][j][0], acc[s][j][1]);
                }
#pragma unroll
                for (int k = 0; k < BC; ++k) {
                    const bool in = rin && (c0 + k < G.nx);
                    if (in && !vec) o[(size_t)j * G.nx + k] = acc[s][j][k];
                    if (!in) acc[s][j][k] = 0.f;             // (not part of the image: keep it out of the norm)
                }
            }
        }
    }
    if (red) {
        __shared__ float part[NS][4];
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            float v = 0.f;
#pragma unroll
            for (int j = 0; j < BR; ++j)
#pragma unroll
                for (int k = 0; k < BC; ++k) v = fmaf(acc[s][j][k], acc[s][j][k], v);
            v = warp_sum(v);
            if (lane == 0) part[s][warp] = v;
        }
        __syncthreads();
        if (threadIdx.x < NS) {
            const int s = threadIdx.x;
            atomicAdd(red + prob + s * G.n_phase, (double)(part[s][0] + part[s][1] + part[s][2] + part[s][3]));
        }
    }
}

}  // namespace tnlm
