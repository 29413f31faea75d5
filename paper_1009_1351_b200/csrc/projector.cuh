// projector.cuh -- fan-beam forward projector P (ray-driven, one thread per (view,bin)) and its
// matched adjoint P^T (pixel-driven gather, one thread per pixel).  PAPER.md:L75, L79, L212.
// Both kernels evaluate tnlm::ray_cell on the same RayEntry table, so every matrix entry
// len(ray ∩ pixel) is bit-identical on the two sides and P^T is the exact transpose of P.
#pragma once
#include "common.cuh"

namespace tnlm {

enum FwdMode {
    FWD_PLAIN = 0,  // out0 = P img
    FWD_RESID = 1,  // out0 = sw*(y - P img) = r ; out1 = sw*r            (CGLS init, L109)
    FWD_SCALE = 2   // out0 = sw*(P img) = q ; red += ||q||^2             (CGLS step 1, L112)
};

// ------------------------------------------------------------------------------ forward
// grid = (ceil(V*B/256), S*N); block = 256.  Adjacent threads = adjacent bins of a view, so a
// warp walks neighbouring pixels of the same image rows (coalesced, L1-resident gathers).
template <int MODE>
__global__ void __launch_bounds__(256)
project_kernel(Geom G, const RayEntry *__restrict__ tab, const RayRange *__restrict__ rng,
               const float *__restrict__ img, const float *__restrict__ y,
               const float *__restrict__ w, float *__restrict__ out0, float *__restrict__ out1,
               double *__restrict__ red)
{
    const int prob = blockIdx.y;                 // slice*N + phase
    const int phase = prob % G.n_phase;
    const int nray = G.n_views * G.n_bins;
    const int ray = blockIdx.x * blockDim.x + threadIdx.x;
    float qq = 0.f;
    if (ray < nray) {
        const RayEntry e = tab[(size_t)phase * nray + ray];
        const RayRange rg = rng[(size_t)phase * nray + ray];
        const float *__restrict__ im = img + (size_t)prob * G.nx * G.ny;
        float acc0 = 0.f, acc1 = 0.f;
        if (rg.steep) {
            const int nx = G.nx;
            for (int q = rg.lo; q <= rg.hi; ++q) {
                int c0, c1; float w0, w1;
                ray_cell(e, q, c0, c1, w0, w1);
                const float *row = im + (size_t)q * nx;
                if ((unsigned)c0 < (unsigned)nx) acc0 = fmaf(w0, __ldg(row + c0), acc0);
                if (c1 != c0 && (unsigned)c1 < (unsigned)nx) acc1 = fmaf(w1, __ldg(row + c1), acc1);
            }
        } else {
            const int nx = G.nx, ny = G.ny;
            for (int q = rg.lo; q <= rg.hi; ++q) {
                int c0, c1; float w0, w1;
                ray_cell(e, q, c0, c1, w0, w1);
                if ((unsigned)c0 < (unsigned)ny) acc0 = fmaf(w0, __ldg(im + (size_t)c0 * nx + q), acc0);
                if (c1 != c0 && (unsigned)c1 < (unsigned)ny) acc1 = fmaf(w1, __ldg(im + (size_t)c1 * nx + q), acc1);
            }
        }
        const float p = acc0 + acc1;
        const size_t o = (size_t)prob * nray + ray;
        if (MODE == FWD_PLAIN) {
            out0[o] = p;
        } else {
            const float sw = w ? sqrtf(w[o]) : 1.0f;
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
        __shared__ float part[8];
        qq = warp_sum(qq);
        if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = qq;
        __syncthreads();
        if (threadIdx.x < 32) {
            float v = threadIdx.x < 8 ? part[threadIdx.x] : 0.f;
            v = warp_sum(v);
            if (threadIdx.x == 0) atomicAdd(red + prob, (double)v);
        }
    }
}

// ----------------------------------------------------------------------------- adjoint
// grid = (ceil(nx/32), ceil(ny/BP_ROWS), S*N); block = (32, BP_ROWS).  One thread per pixel,
// loop over the views of its phase; per view the candidate bins are those whose fan angle is
// within the pixel's angular footprint (conservative superset); each candidate's ray_cell for
// this pixel's row (steep ray) or column (shallow ray) decides membership and gives the length.
// red (optional) += ||out||^2 of this problem.
#define BP_ROWS 4
__global__ void __launch_bounds__(32 * BP_ROWS)
backproject_kernel(Geom G, const RayEntry *__restrict__ tab, const RayRange *__restrict__ rng,
                   const float4 *__restrict__ views, const float *__restrict__ sino,
                   float *__restrict__ out, double *__restrict__ red)
{
    const int prob = blockIdx.z;
    const int phase = prob % G.n_phase;
    const int c = blockIdx.x * 32 + threadIdx.x;
    const int r = blockIdx.y * BP_ROWS + threadIdx.y;
    const int V = G.n_views, B = G.n_bins;
    const bool inside = (c < G.nx) && (r < G.ny);
    float acc = 0.f;
    if (inside) {
        const float X = ((float)c - 0.5f * (float)(G.nx - 1)) * G.pix;
        const float Y = ((float)r - 0.5f * (float)(G.ny - 1)) * G.pix;
        const float4 *__restrict__ vt = views + (size_t)phase * V;
        const RayEntry *__restrict__ tb = tab + (size_t)phase * V * B;
        const RayRange *__restrict__ rb = rng + (size_t)phase * V * B;
        const float *__restrict__ sg = sino + (size_t)prob * V * B;
        for (int v = 0; v < V; ++v) {
            const float4 vw = __ldg(vt + v);                 // sx, sy, cos th, sin th
            const float px = X - vw.x, py = Y - vw.y;
            const float dot = -(vw.z * px + vw.w * py);      // along the central ray (> 0)
            const float crs = vw.w * px - vw.z * py;         // ccw from the central ray
            const float gam = atanf(__fdividef(crs, dot));
            const float kc = fmaf(gam, G.sdd_over_pitch, G.bin_centre);
            const float hw = fmaf(G.half_diag * rsqrtf(px * px + py * py), G.sdd_over_pitch * 1.02f, 0.05f);
            const int k_lo = max(0, (int)ceilf(kc - hw));
            const int k_hi = min(B - 1, (int)floorf(kc + hw));
            for (int k = k_lo; k <= k_hi; ++k) {
                const float4 e4 = __ldg(reinterpret_cast<const float4 *>(tb + (size_t)v * B + k));
                RayEntry e; e.p0 = e4.x; e.m = e4.y; e.len = e4.z; e.inva = e4.w;
                const int steep = __ldg(&rb[(size_t)v * B + k].steep);
                int c0, c1; float w0, w1;
                ray_cell(e, steep ? r : c, c0, c1, w0, w1);
                const int me = steep ? c : r;
                float wgt = 0.f;
                if (c0 == me) wgt = w0;
                else if (c1 == me) wgt = w1;
                acc = fmaf(wgt, __ldg(sg + (size_t)v * B + k), acc);
            }
        }
        out[(size_t)prob * G.nx * G.ny + (size_t)r * G.nx + c] = acc;
    }
    if (red) {
        __shared__ float part[BP_ROWS];
        float v = inside ? acc * acc : 0.f;
        v = warp_sum(v);
        if (threadIdx.x == 0) part[threadIdx.y] = v;
        __syncthreads();
        if (threadIdx.y == 0 && threadIdx.x == 0) {
            float s = 0.f;
#pragma unroll
            for (int i = 0; i < BP_ROWS; ++i) s += part[i];
            atomicAdd(red + prob, (double)s);
        }
    }
}

}  // namespace tnlm
