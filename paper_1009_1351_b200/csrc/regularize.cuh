// regularize.cuh -- the TNLM half of one outer iteration: patch-distance weights to the two
// cyclic neighbour phases (Eq. 3/8) inside a W x W search window
// (L204), one Gauss-Jacobi sweep of Eq. (7) (L143-L158), optional positivity clip (L167).
//
// Formulation.  For one search offset delta the patch distance of every pixel is a d x d box
// sum of ONE shifted squared-difference image SD_delta(y) = (g_i(y) - g_j(y+delta))^2.  Each
// thread owns a 4 x 4 pixel tile and, per offset, builds the (4+2b) x (4+2b) differences from
// registers (g_i, loaded once) and shared memory (g_j), box-sums them separably with running
// sums (rows first, then columns), and folds the 16 distances into per-pixel softmax
// accumulators (m, Z, A) that stay in registers for the whole window:
//     t = -D*log2(e)/h^2 - m ;  e = 2^t ;  Z += e ;  A += e*u_j(x+delta)
// m is a lazily updated reference exponent (raised only when some t exceeds TAU), so the
// quotient A/Z is the softmax-weighted mean of Eq. (7) without overflow or underflow.
// Weights are never stored (recomputing beats 2*W^2 floats per pixel of HBM traffic).
#pragma once
#include "common.cuh"

namespace tnlm {

constexpr int TQ = 4;           // thread tile: TQ x TQ pixels
constexpr float TAU = 16.0f;    // lazy-rescale threshold in log2 units

struct RegParams {
    int nx, ny, n_phase;
    int a;                  // (window-1)/2
    float neg_c;            // -log2(e)/h^2
    float c_self;           // 1/(1+mu)
    float c_nb;             // mu/(2mu+2)
    float big_d;            // distance given to out-of-image candidates (finite)
    float m_init;           // initial reference exponent: neg_c*big_d/10
    int clip;               // apply max(.,0) to the output
};

// Shared-memory tile layout ("planar-4"): element (row, col) of a tile lives at
//   row*4*P + (col & 3)*P + (col >> 2),   P odd.
// A thread reads columns 4*tx + e for several e; for a fixed e the lanes of a warp touch
// consecutive words of one plane (and the second half-warp, four rows further down, lands 16
// banks away because 16*P = 16 mod 32), so every LDS.32 of the inner loop is conflict-free.
__device__ __forceinline__ int planar(int row, int col, int P) { return row * 4 * P + (col & 3) * P + (col >> 2); }

template <int TX, int TY>
__host__ __device__ constexpr int reg_tile_w() { return TX * TQ; }

// PB = (patch-1)/2.  BORDER: the tile has candidates outside the image (or is partial).
template <int PB, int TX, int TY, bool BORDER>
__global__ void __launch_bounds__(TX * TY)
gj_sweep_kernel(RegParams p, const float *__restrict__ g, const float *__restrict__ u,
                float *__restrict__ out, const int2 *__restrict__ tiles, int tiles_per_image)
{
    constexpr int RW = TQ + 2 * PB;           // region side per thread
    constexpr int TW = TX * TQ, TH = TY * TQ; // CTA pixel tile
    const int a = p.a, halo = a + PB;
    const int gw = TW + 2 * halo, gh = TH + 2 * halo;   // g_j tile
    const int uw = TW + 2 * a, uh = TH + 2 * a;         // u_j tile
    const int P = (((gw + 3) >> 2) | 1);                // odd plane stride
    extern __shared__ float smem[];
    float *sG = smem;                                   // gh rows
    float *sU = smem + gh * 4 * P;                      // uh rows (same P)

    const int img = blockIdx.x / tiles_per_image;       // slice*N + phase
    const int2 tile = tiles[blockIdx.x % tiles_per_image];
    const int slice = img / p.n_phase, phase = img % p.n_phase;
    const int nx = p.nx, ny = p.ny;
    const size_t npix = (size_t)nx * ny;
    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
    const int r0 = tile.y + ty * TQ, c0 = tile.x + tx * TQ;    // thread's first pixel

    // g_i region of this thread: (r0-PB .. r0+TQ-1+PB) x (c0-PB .. c0+TQ-1+PB), zero outside.
    const float *__restrict__ gi = g + ((size_t)slice * p.n_phase + phase) * npix;
    float Gi[RW][RW];
#pragma unroll
    for (int rr = 0; rr < RW; ++rr)
#pragma unroll
        for (int cc = 0; cc < RW; ++cc) {
            const int r = r0 - PB + rr, c = c0 - PB + cc;
            Gi[rr][cc] = ((unsigned)r < (unsigned)ny && (unsigned)c < (unsigned)nx) ? __ldg(gi + (size_t)r * nx + c) : 0.f;
        }

    float nbsum[TQ][TQ];
#pragma unroll
    for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
        for (int q = 0; q < TQ; ++q) nbsum[rr][q] = 0.f;

    // per-thread smem base offsets (tile row 4*ty, column 4*tx => plane 0, index tx)
    const int rowstride = 4 * P;
    const int tbase = (ty * TQ) * rowstride + tx;

    for (int side = 0; side < 2; ++side) {
        const int j = (phase + (side == 0 ? p.n_phase - 1 : 1)) % p.n_phase;   // cyclic (L81)
        const float *__restrict__ gj = g + ((size_t)slice * p.n_phase + j) * npix;
        const float *__restrict__ uj = u + ((size_t)slice * p.n_phase + j) * npix;
        __syncthreads();                                   // previous side's readers are done
        for (int idx = threadIdx.x; idx < gh * gw; idx += TX * TY) {
            const int rr = idx / gw, cc = idx - rr * gw;
            const int r = tile.y - halo + rr, c = tile.x - halo + cc;
            sG[planar(rr, cc, P)] = ((unsigned)r < (unsigned)ny && (unsigned)c < (unsigned)nx) ? __ldg(gj + (size_t)r * nx + c) : 0.f;
        }
        for (int idx = threadIdx.x; idx < uh * uw; idx += TX * TY) {
            const int rr = idx / uw, cc = idx - rr * uw;
            const int r = tile.y - a + rr, c = tile.x - a + cc;
            sU[planar(rr, cc, P)] = ((unsigned)r < (unsigned)ny && (unsigned)c < (unsigned)nx) ? __ldg(uj + (size_t)r * nx + c) : 0.f;
        }
        __syncthreads();

        float m[TQ][TQ], Z[TQ][TQ], A[TQ][TQ];
#pragma unroll
        for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
            for (int q = 0; q < TQ; ++q) { m[rr][q] = p.m_init; Z[rr][q] = 0.f; A[rr][q] = 0.f; }

        for (int dr = -a; dr <= a; ++dr) {
            float rowpen[TQ];
            if (BORDER) {
#pragma unroll
                for (int rr = 0; rr < TQ; ++rr) rowpen[rr] = ((unsigned)(r0 + rr + dr) < (unsigned)ny) ? 0.f : p.big_d;
            }
            const int gbase = tbase + (dr + a) * rowstride;   // g_j tile row (4ty + rr' + dr + a)
            for (int dc = -a; dc <= a; ++dc) {
                // column offsets inside a tile row for e = j + dc + a, j = 0..RW-1
                int off[RW];
#pragma unroll
                for (int jj = 0; jj < RW; ++jj) {
                    const int e = jj + dc + a;
                    off[jj] = (e & 3) * P + (e >> 2);
                }
                // ---- rows of the region: differences, horizontal running box sums
                float H[RW][TQ];
#pragma unroll
                for (int rr = 0; rr < RW; ++rr) {
                    float df[RW];
#pragma unroll
                    for (int jj = 0; jj < RW; ++jj) df[jj] = Gi[rr][jj] - sG[gbase + rr * rowstride + off[jj]];
                    float h0 = df[0] * df[0];
#pragma unroll
                    for (int jj = 1; jj <= 2 * PB; ++jj) h0 = fmaf(df[jj], df[jj], h0);
                    H[rr][0] = h0;
#pragma unroll
                    for (int q = 1; q < TQ; ++q) {
                        h0 = fmaf(df[q + 2 * PB], df[q + 2 * PB], h0);
                        h0 = fmaf(-df[q - 1], df[q - 1], h0);
                        H[rr][q] = h0;
                    }
                }
                // ---- vertical running box sums -> D, then exponent relative to m
                float t[TQ][TQ], Dd[TQ][TQ];
#pragma unroll
                for (int q = 0; q < TQ; ++q) {
                    float colpen = 0.f;
                    if (BORDER) colpen = ((unsigned)(c0 + q + dc) < (unsigned)nx) ? 0.f : p.big_d;
                    float d0 = H[0][q];
#pragma unroll
                    for (int rr = 1; rr <= 2 * PB; ++rr) d0 += H[rr][q];
#pragma unroll
                    for (int rr = 0; rr < TQ; ++rr) {
                        if (rr > 0) d0 = (d0 + H[rr + 2 * PB][q]) - H[rr - 1][q];
                        float dv = d0;
                        if (BORDER) dv = fmaxf(fmaxf(dv, rowpen[rr]), colpen);
                        Dd[rr][q] = dv;
                        t[rr][q] = fmaf(dv, p.neg_c, -m[rr][q]);
                    }
                }
                // ---- lazy rescale: rare once the window's best matches have been seen
                float tmax = t[0][0];
#pragma unroll
                for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
                    for (int q = 0; q < TQ; ++q) tmax = fmaxf(tmax, t[rr][q]);
                if (tmax > TAU) {
#pragma unroll
                    for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
                        for (int q = 0; q < TQ; ++q)
                            if (t[rr][q] > TAU) {
                                const float s = Dd[rr][q] * p.neg_c;
                                const float corr = exp2f(m[rr][q] - s);
                                Z[rr][q] *= corr;
                                A[rr][q] *= corr;
                                m[rr][q] = s;
                                t[rr][q] = 0.f;
                            }
                }
                // ---- accumulate
                const int ubase = tbase + (dr + a) * rowstride;   // u_j tile row (4ty + rr + dr + a)
#pragma unroll
                for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
                    for (int q = 0; q < TQ; ++q) {
                        float e;
                        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(t[rr][q]));
                        Z[rr][q] += e;
                        A[rr][q] = fmaf(e, sU[ubase + rr * rowstride + off[q]], A[rr][q]);
                    }
            }
        }
#pragma unroll
        for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
            for (int q = 0; q < TQ; ++q) nbsum[rr][q] += __fdividef(A[rr][q], Z[rr][q]);
    }

    float *__restrict__ o = out + ((size_t)slice * p.n_phase + phase) * npix;
#pragma unroll
    for (int rr = 0; rr < TQ; ++rr)
#pragma unroll
        for (int q = 0; q < TQ; ++q) {
            const int r = r0 + rr, c = c0 + q;
            if (r < ny && c < nx) {
                float v = fmaf(p.c_nb, nbsum[rr][q], p.c_self * Gi[rr + PB][q + PB]);
                if (p.clip) v = fmaxf(v, 0.f);
                o[(size_t)r * nx + c] = v;
            }
        }
}

// f = max(g, 0): the m2 = 0 case of steps 3-5.
__global__ void clip_kernel(const float *__restrict__ g, float *__restrict__ out, size_t n)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = fmaxf(g[i], 0.f);
}

}  // namespace tnlm
