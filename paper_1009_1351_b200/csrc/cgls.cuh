// cgls.cuh -- vector updates of the "CGLS Algorithm".  All scalars
// (gamma_m = ||P_n^T r^(m)||^2, qq_m = ||P_n s^(m)||^2) live on the device as doubles, one per
// (slice, phase) problem and inner step; kernels derive a_m and b_m from them on the fly, so
// nothing synchronises with the host.
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

// u += a s (step 2, L114);  grid = (ceil(npix/256), nprob)
__global__ void cgls_update_u(float *__restrict__ u, const float *__restrict__ s, int npix,
                              const double *gam, const double *qq, int nprob, int m)
{
    const int prob = blockIdx.y;
    const float a = cgls_a(gam, qq, nprob, prob, m);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < npix) {
        const size_t o = (size_t)prob * npix + i;
        u[o] = fmaf(a, s[o], u[o]);
    }
}

// r -= a q (step 3, L115);  rw = sqrt(w) r (the sinogram P_n^T gathers);  grid = (ceil(nray/256), nprob)
__global__ void cgls_update_r(float *__restrict__ r, float *__restrict__ rw, const float *__restrict__ q,
                              const float *__restrict__ w, int nray, const double *gam,
                              const double *qq, int nprob, int m)
{
    const int prob = blockIdx.y;
    const float a = cgls_a(gam, qq, nprob, prob, m);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nray) {
        const size_t o = (size_t)prob * nray + i;
        const float rn = fmaf(-a, q[o], r[o]);
        r[o] = rn;
        rw[o] = (w ? sqrtf(w[o]) : 1.0f) * rn;
    }
}

// s = t + b s (step 5, L126);  a broken-down phase keeps s (it is never used again)
__global__ void cgls_update_s(float *__restrict__ s, const float *__restrict__ t, int npix,
                              const double *gam, const double *qq, int nprob, int m)
{
    const int prob = blockIdx.y;
    const float b = cgls_b(gam, qq, nprob, prob, m);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < npix) {
        const size_t o = (size_t)prob * npix + i;
        s[o] = fmaf(b, s[o], t[o]);
    }
}

}  // namespace tnlm
