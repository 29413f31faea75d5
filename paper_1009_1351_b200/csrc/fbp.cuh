// fbp.cuh -- step 1 of the "TNLM Algorithm": f_i^(0) = the image reconstructed by
// filtered backprojection from ALL projections of ALL N phases, the same for every i.  The paper
// names the method only; this is the textbook equiangular fan-beam FBP (Kak & Slaney 3.4.1,
// DESIGN.md reading 24):
//   R'_j(n) = y_j(n) * SID * cos(gamma_n)                                   (fbp_filter_kernel)
//   Q_j(n)  = dgamma * sum_m R'_j(m) g((n-m) dgamma),  g(0) = 1/(8 dgamma^2), g(even) = 0,
//             g(odd k) = -1/(2 pi^2 sin^2(k dgamma))      (ramp filter; its 1/2 is the full-scan 1/2)
//   f(x)    = sum_j dbeta_j * Q_j(gamma'(x)) / L_j(x)^2                      (fbp_backproject_kernel)
// with dbeta_j the trapezoid weight of view j in the sorted cyclic union of all N*V source angles,
// gamma' the fan angle of the pixel centre (Q linearly interpolated between bins, 0 outside the
// detector) and L the source-pixel distance.  The filter table g, the cosine weights and dbeta are
// built in double precision at tnlm_create; the convolution accumulates in double (the ramp kernel
// alternates in sign over three orders of magnitude), the backprojection in fp32.
#pragma once
#include "common.cuh"

namespace tnlm {

// grid = (N*V, S); block = 256; dynamic shared memory = B floats.
// y [S][N*V][B] -> q [S][N*V][B];  cosw[n] = SID*cos(gamma_n);  gk[k] = dgamma * g(k dgamma), k = 0..B-1.
__global__ void __launch_bounds__(256)
fbp_filter_kernel(const float *__restrict__ y, float *__restrict__ q, const float *__restrict__ cosw,
                  const double *__restrict__ gk, int B)
{
    extern __shared__ float rp[];
    const size_t row = ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * B;
    for (int n = threadIdx.x; n < B; n += blockDim.x) rp[n] = __ldg(y + row + n) * __ldg(cosw + n);
    __syncthreads();
    for (int n = threadIdx.x; n < B; n += blockDim.x) {
        double acc = (double)rp[n] * gk[0];
        for (int m = (n + 1) & 1; m < B; m += 2) {           // only odd n - m carry weight
            const int k = n > m ? n - m : m - n;
            acc = fma((double)rp[m], gk[k], acc);
        }
        q[row + n] = (float)acc;
    }
}

// grid = (ceil(nx/32), ceil(ny/8), S); block = (32, 8).  One thread per pixel, loop over all N*V views.
// views[j] = (sx, sy, cos beta, sin beta); wv[j] = dbeta_j.  Writes the same value to all N phase images.
__global__ void __launch_bounds__(256)
fbp_backproject_kernel(Geom G, const float4 *__restrict__ views, const float *__restrict__ wv,
                       const float *__restrict__ q, float *__restrict__ out)
{
    const int c = blockIdx.x * 32 + threadIdx.x, r = blockIdx.y * 8 + threadIdx.y;
    if (c >= G.nx || r >= G.ny) return;
    const int M = G.n_phase * G.n_views, B = G.n_bins;
    const float X = ((float)c - 0.5f * (float)(G.nx - 1)) * G.pix;
    const float Y = ((float)r - 0.5f * (float)(G.ny - 1)) * G.pix;
    const float *__restrict__ qs = q + (size_t)blockIdx.z * M * B;
    float acc = 0.f;
    for (int j = 0; j < M; ++j, qs += B) {
        const float4 vw = __ldg(views + j);
        const float px = X - vw.x, py = Y - vw.y;
        const float dot = -(vw.z * px + vw.w * py);          // L cos(gamma') > 0
        const float crs = vw.w * px - vw.z * py;             // L sin(gamma')
        const float k = fmaf(atan2f(crs, dot), G.sdd_over_pitch, G.bin_centre);
        const float kf = floorf(k);
        const int k0 = (int)kf;
        const float fr = k - kf;
        const float qa = ((unsigned)k0 < (unsigned)B) ? __ldg(qs + k0) : 0.f;
        const float qb = ((unsigned)(k0 + 1) < (unsigned)B) ? __ldg(qs + k0 + 1) : 0.f;
        acc = fmaf(__ldg(wv + j) * fmaf(fr, qb - qa, qa), __fdividef(1.0f, fmaf(px, px, py * py)), acc);
    }
    float *__restrict__ o = out + (size_t)blockIdx.z * G.n_phase * G.nx * G.ny + (size_t)r * G.nx + c;
    for (int i = 0; i < G.n_phase; ++i) o[(size_t)i * G.nx * G.ny] = acc;
}

}  // namespace tnlm
