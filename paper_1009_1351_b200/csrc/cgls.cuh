// cgls.cuh -- vector updates of the "CGLS Algorithm".  All scalars
// (gamma_m = ||P_n^T r^(m)||^2, qq_m = ||P_n s^(m)||^2) live on the device as doubles, one per
// (slice, phase) problem and inner step; kernels derive a_m and b_m from them on the fly, so
// nothing synchronises with the host.
//
// Launches per inner step m (tnlm_api.cu, cgls_device):
//   project_kernel<FWD_SCALE>   q = sqrt(w) P s_m, qq_m                      (reads s_m and its transpose)
//   cgls_update_r               r -= a_m q ; rw = sqrt(w) r                   (sinogram pass)
//   backproject_kernel          t = P^T rw, gamma_{m+1}
//   cgls_update_us              u += a_m s_m ; s_{m+1} = t + b_m s_m ; sT = s_{m+1}^T   (one image pass)
// The last step only needs u += a_m s_m (cgls_update_us<true>): r, t, s of step M1 feed nothing (L127).
// In a call with four or more slices the groups of four slices run project_il_kernel / cgls_update_us_il instead:
// their s lives only in the interleaved copies the batch projector reads (projector.cuh).
#pragma once
#include "common.cuh"

namespace tnlm {

// Scalars of problem `prob`: gam[m*nprob + prob] for m = 0..m1, qq[m*nprob + prob] for m < m1.
// A phase that breaks down (gamma or qq not > 0) stops for good: a = b = 0 from then on.
__device__ __forceinline__ bool cgls_alive(const double *gam, const double *qq, int nprob, int prob, int m)
{
    for (int i = 0; i <= m; ++i)
        if (!(gam[(size_t)i * nprob + prob] > 0.0) || !(qq[(size_t)i * nprob + prob] > 0.0)) return false;
    return true;
}
__device__ __forceinline__ float cgls_a(const double *gam, const double *qq, int nprob, int prob, int m)
{
    if (!cgls_alive(gam, qq, nprob, prob, m)) return 0.f;
    return (float)(gam[(size_t)m * nprob + prob] / qq[(size_t)m * nprob + prob]);      // step 1 (L112)
}
__device__ __forceinline__ float cgls_b(const double *gam, const double *qq, int nprob, int prob, int m)
{
    if (!cgls_alive(gam, qq, nprob, prob, m)) return 0.f;
    return (float)(gam[(size_t)(m + 1) * nprob + prob] / gam[(size_t)m * nprob + prob]); // step 4 (L125)
}

// sw = sqrt(w): the diagonal of Sigma^-1/2 (L103), computed once per call instead of once per use.
__global__ void sqrt_weights_kernel(const float *__restrict__ w, float *__restrict__ sw, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) sw[i] = sqrtf(w[i]);
}

// r -= a q (step 3, L115);  rw = sqrt(w) r (the sinogram P_n^T gathers);  grid = (ceil(nray/256), nprob)
__global__ void __launch_bounds__(256)
cgls_update_r(float *__restrict__ r, float *__restrict__ rw, const float *__restrict__ q,
              const float *__restrict__ sw, int nray, const double *gam, const double *qq, int nprob, int m)
{
    __shared__ float a_sh;
    const int prob = blockIdx.y;
    if (threadIdx.x == 0) a_sh = cgls_a(gam, qq, nprob, prob, m);
    __syncthreads();
    const float a = a_sh;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nray) {
        const size_t o = (size_t)prob * nray + i;
        const float rn = fmaf(-a, q[o], r[o]);
        r[o] = rn;
        rw[o] = (sw ? sw[o] : 1.0f) * rn;
    }
}

// u += a_m s (step 2, L114) and, unless LAST, s = t + b_m s (step 5, L126) with the transposed copy sT
// the forward projector reads for its shallow rays, in one pass over 32 x 32 image tiles.
// A broken-down phase has a = b = 0: u stays, s = t (never used again).
// grid = (ceil(nx/32), ceil(ny/32), problems prob0 .. ); block = (32, 8).
template <bool LAST>
__global__ void __launch_bounds__(256)
cgls_update_us(float *__restrict__ u, float *__restrict__ s, const float *__restrict__ t, float *__restrict__ sT,
               int nx, int ny, const double *gam, const double *qq, int nprob, int m, int prob0)
{
    __shared__ float tile[32][33];
    __shared__ float ab[2];
    const int prob = blockIdx.z + prob0;
    if (threadIdx.x == 0 && threadIdx.y == 0) {
        ab[0] = cgls_a(gam, qq, nprob, prob, m);
        ab[1] = LAST ? 0.f : cgls_b(gam, qq, nprob, prob, m);
    }
    __syncthreads();
    const float a = ab[0], b = ab[1];
    const size_t base = (size_t)prob * nx * ny;
    const int c = blockIdx.x * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int r = blockIdx.y * 32 + threadIdx.y + j;
        float sn = 0.f;
        if (r < ny && c < nx) {
            const size_t o = base + (size_t)r * nx + c;
            const float so = s[o];
            u[o] = fmaf(a, so, u[o]);
            if (!LAST) {
                sn = fmaf(b, so, t[o]);
                s[o] = sn;
            }
        }
        if (!LAST) tile[threadIdx.y + j][threadIdx.x] = sn;
    }
    if (LAST) return;
    __syncthreads();
    const int rT = blockIdx.y * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int cT = blockIdx.x * 32 + threadIdx.y + j;
        if (rT < ny && cT < nx) sT[base + (size_t)cT * ny + rT] = tile[threadIdx.x][threadIdx.y + j];
    }
}

// The same for a group of four slices whose search direction s lives only in the interleaved copies the batch
// projector reads (project_il_kernel): sI[group][phase][r][c] = s of slices 4g .. 4g+3, updated in place, and its
// transpose sTI; u and t stay in the caller's layout.  Per slice the arithmetic is that of cgls_update_us.
// grid = (ceil(nx/32), ceil(ny/32), groups*N); block = (32, 8).
template <bool LAST>
__global__ void __launch_bounds__(256)
cgls_update_us_il(float *__restrict__ u, float4 *__restrict__ sI, const float *__restrict__ t, float4 *__restrict__ sTI,
                  int nx, int ny, int n_phase, const double *gam, const double *qq, int nprob, int m)
{
    __shared__ float4 tile[32][33];
    __shared__ float ab[2][4];
    const int group = blockIdx.z / n_phase, phase = blockIdx.z - group * n_phase;
    const int prob = group * 4 * n_phase + phase;            // of the group's first slice
    if (threadIdx.y == 0 && threadIdx.x < 4) {
        ab[0][threadIdx.x] = cgls_a(gam, qq, nprob, prob + threadIdx.x * n_phase, m);
        ab[1][threadIdx.x] = LAST ? 0.f : cgls_b(gam, qq, nprob, prob + threadIdx.x * n_phase, m);
    }
    __syncthreads();
    const float a[4] = {ab[0][0], ab[0][1], ab[0][2], ab[0][3]}, b[4] = {ab[1][0], ab[1][1], ab[1][2], ab[1][3]};
    const size_t npix = (size_t)nx * ny, sl = (size_t)n_phase * npix;
    const size_t base = (size_t)prob * npix, base4 = ((size_t)group * n_phase + phase) * npix;
    const int c = blockIdx.x * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int r = blockIdx.y * 32 + threadIdx.y + j;
        float4 sn = make_float4(0.f, 0.f, 0.f, 0.f);
        if (r < ny && c < nx) {
            const size_t o = (size_t)r * nx + c;
            const float4 so4 = sI[base4 + o];
            const float so[4] = {so4.x, so4.y, so4.z, so4.w};
            float snv[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const size_t oq = base + q * sl + o;
                u[oq] = fmaf(a[q], so[q], u[oq]);
                if (!LAST) snv[q] = fmaf(b[q], so[q], t[oq]);
            }
            if (!LAST) {
                sn = make_float4(snv[0], snv[1], snv[2], snv[3]);
                sI[base4 + o] = sn;
            }
        }
        if (!LAST) tile[threadIdx.y + j][threadIdx.x] = sn;
    }
    if (LAST) return;
    __syncthreads();
    const int rT = blockIdx.y * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int cT = blockIdx.x * 32 + threadIdx.y + j;
        if (rT < ny && cT < nx) sTI[base4 + (size_t)cT * ny + rT] = tile[threadIdx.x][threadIdx.y + j];
    }
}

}  // namespace tnlm
