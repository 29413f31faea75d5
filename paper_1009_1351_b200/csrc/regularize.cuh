// regularize.cuh -- the TNLM half of one outer iteration: patch-distance weights to the two
// cyclic neighbour phases (Eq. 3/8) inside a W x W search window
// (L204), one Gauss-Jacobi sweep of Eq. (7) (L143-L158), optional positivity clip (L167).
//
// Formulation (v2, "row march").  For one search offset delta = (dr, dc) the patch distance of
// every pixel is the d x d box sum of ONE shifted squared-difference image
//     SD_delta(y) = (g_i(y) - g_j(y + delta))^2 ,   D(x, delta) = sum_{p in [-b,b]^2} SD_delta(x + p).
// A warp owns a band of RB rows x 128 columns of phase i and ONE neighbour phase j ("side");
// lane l owns the C = 4 columns 4l..4l+3.  An "item" is one dr and G = 4 consecutive dc.  For an
// item the lane marches down the RB + 2b rows of its band: per row it loads 4+2b values of g_i
// and 4+2b+3 values of g_j (aligned LDS.128), forms the squared differences, slides the
// horizontal box sum over its 4 columns (2 FMA per step), adds the row into a vertical running
// sum D[g][c] and retires the row that left the window from a 2b-deep register ring.  Every
// D is then one FMA (exponent), one ex2.approx, one FADD (Z) and one FMA (numerator A) away from
// the accumulators Z[row][c], A[row][c], which stay in registers for the whole window.
// Per weight evaluation this costs 2 FSUB-slots + 2.75 FMA (box rows, x 1+2b/RB for the warm-up
// rows) + 2 FADD (vertical) + 4: about 12 FP32 instructions against 2d+4 = 14 algorithmic flops.
//
// Softmax reference.  w = exp(-D/h^2)/Z is evaluated as 2^(c*(D0(x) - D(x,delta)) - 100),
// c = log2(e)/h^2, D0 = the distance at delta = 0 (always a valid candidate), so the delta = 0
// term is 2^-100 and Z can never underflow to 0; a pixel whose weight sum reaches 2^100 (a candidate
// about 200/c better than delta = 0) or whose numerator is not below 2^120 is flagged, and flagged
// pixels are recomputed by the warp with the minimum-subtracted two-pass form (exact_side_ratio)
// straight from the shared tiles.  With Z < 2^100 the numerator sum_delta e u_j stays finite for
// |u| < 2^17 (documented in tnlm.h), here and in gj_apply3_kernel, which re-reads the same weights.
// The value is always the softmax of Eq. (3); the reference only picks the fp32 range.
//
// Borders.  Tiles are zero-filled outside the image (patches are zero-extended, DESIGN.md
// reading 7).  A candidate column outside the image (or a dc beyond the window in the last
// item of a row) gets its running sum D initialised to a huge finite value, which no sliding
// update can change, so its weight is exactly 0 at no per-evaluation cost; candidate rows
// outside the image are skipped warp-uniformly.
//
// Stored weights ("reusing this factor ... instead of recomputing").  The weights
// belong to g^(k) and stay fixed for all M2 sweeps (L162), so when M2 > 1 and the caller has opted in
// (option weight_cache_mb > 0; by default every sweep computes its weights) the first sweep
// (STORE_W = true) also writes every unnormalised weight as bf16 into
// wts[image][band][tile_x][side][delta][RB/2 row pairs][32 lanes][2 rows][4 columns] -- one
// contiguous chunk per warp band, written and later read as a sequential stream (DRAM-page
// friendly; a plane-per-offset layout scatters 256-byte pieces and ran 3x slower); inside a plane
// the two rows of a pair are interleaved per lane so that the applying sweeps read 16 bytes per
// lane (plane_off below).  bf16 keeps the fp32 exponent range, so the
// stored values are the very 2^(c(D0-D)-100) of the fast path (an fp16 version needed its own
// reference and sent every moving edge through the slow exact route: 2.6x slower); the quotient
// A/Z of Eq. (7) does not depend on the per-pixel scale, and the 2^-9 rounding of each weight
// moves it by < 1e-6 relative.  Pixels on the exact route store their
// minimum-subtracted weights instead.  Sweeps 2..M2 are gj_apply3_kernel: a streaming pass
// over the chunks, bound by HBM (2 bytes per weight) instead of by the FP32 pipes.  With M2 = 1
// nothing is stored.
#pragma once
#include <cuda_bf16.h>

#include "common.cuh"

namespace tnlm {

constexpr int SW_C = 4;        // columns per lane
constexpr int SW_G = 4;        // search offsets (consecutive dc) per item
constexpr int SW_TW = 128;     // tile width = 32 lanes x SW_C
// Keeps ptxas from hoisting the next row's shared-memory loads over a whole march step (the
// hoisted values push the kernel over 255 registers and spill); the other warp of the scheduler
// covers the exposed load latency.
#ifndef SW_STEP_FENCE
#define SW_STEP_FENCE() asm volatile("" ::: "memory")
#endif

struct SweepParams {
    int nx, ny, n_phase;
    int a;                  // (window-1)/2
    int ngroups;            // ceil(window / SW_G)
    int nb;                 // row bands per CTA; a CTA has 2*nb warps (band x side)
    int tiles_x, tiles_y;   // tiles per image
    int rb;                 // rows per band (= RB of the sweep kernel that stored the weights)
    int nbands;             // row bands per image in the stored-weight layout (tiles_y * nb of that sweep)
    float neg_c;            // -log2(e)/h^2
    float pos_c;            // +log2(e)/h^2
    float c_self;           // 1/(1+mu)
    float c_nb;             // mu/(2mu+2)
    float big_d;            // distance given to excluded candidates (finite, big_d*pos_c finite)
    float margin;           // the delta = 0 weight is 2^-margin (100)
    float z_limit;          // a side whose weight sum is not below this (2^100) is recomputed exactly
    float a_limit;          // ... or whose numerator magnitude is not below this (2^120)
    int clip;               // apply max(.,0) to the output
    int n_img;              // gj_apply3_kernel: S*N images in this launch
    int ap_reverse;         // gj_apply3_kernel: take the stored bands from the last one down (snake order over the sweeps)
    long long res_tasks;    // stored-weight tasks (row pairs, in layout order) below this index are kept in L2
                            // (evict_last) by the storing sweep and the applying sweeps; the rest streams (evict_first)
};

// Shared-memory tile geometry (words), shared by host (sizing) and device.
template <int PB>
struct SweepGeom {
    static constexpr int NGI = (SW_C + 2 * PB + 3) / 4;               // float4 loads of g_i per row
    static constexpr int NGJ = (SW_C + 2 * PB + SW_G - 1 + 3) / 4;    // float4 loads of g_j per row
    static constexpr int NUJ = (SW_C + SW_G - 1 + 3) / 4;             // float4 loads of u_j per row
    static constexpr int GIW = 124 + 4 * NGI;                         // g_i tile row stride
    __host__ __device__ static int gjw(int ngroups) { return 124 + 4 * (ngroups - 1) + 4 * NGJ; }
    __host__ __device__ static int ujw(int ngroups) { return 124 + 4 * (ngroups - 1) + 4 * NUJ; }
    __host__ __device__ static size_t smem_words(int a, int ngroups, int nb, int rb)
    {
        const int th = nb * rb;
        return (size_t)(th + 2 * PB) * GIW + 2 * (size_t)(th + 2 * PB + 2 * a) * gjw(ngroups) +
               2 * (size_t)(th + 2 * a) * ujw(ngroups) + 2 * (size_t)nb * rb * SW_TW;
    }
};

// Position (in halves) of pixel (band row rr, tile column cc) inside one stored-weight plane of RB x 128.
__host__ __device__ __forceinline__ int plane_off(int rr, int cc)
{
    return ((((rr >> 1) << 5) + (cc >> 2)) << 3) + ((rr & 1) << 2) + (cc & 3);
}

__device__ __forceinline__ float fast_ex2(float t)
{
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(t));
    return e;
}

// Zero-filled copy of the image window rows [r_org, r_org+rows) x cols [c_org, c_org+width) into
// dst[rows][width]; warps take rows, lanes take columns (coalesced).  Asynchronous: every element is its
// own cp.async, so all of a tile's loads are in flight together (a load-then-store loop exposed one L2
// round trip per row and lane: 13 us per CTA of the sweep, 7-14 us per CTA of the stored-weight sweep).
// The caller commits the group, waits for it and synchronises the threads that read the tile.
__device__ __forceinline__ void stage_tile_async(float *__restrict__ dst, int rows, int width,
                                                 const float *__restrict__ img, int r_org, int c_org, int ny, int nx,
                                                 int warp, int nwarps, int lane)
{
    for (int rr = warp; rr < rows; rr += nwarps) {
        const int r = r_org + rr;
        const bool rin = (unsigned)r < (unsigned)ny;
        const float *__restrict__ src = img + (size_t)(rin ? r : 0) * nx;
        float *__restrict__ d = dst + rr * width;
        for (int cc = lane; cc < width; cc += 32) {
            const int c = c_org + cc;
            const bool in = rin && (unsigned)c < (unsigned)nx;
            cp_async4_zfill(d + cc, src + (in ? c : 0), in);
        }
    }
}

// Exact (minimum-subtracted, two-pass) softmax-weighted mean of u_j over the window of ONE pixel
// and one side, computed by the whole warp from the shared tiles: the fallback for pixels whose
// fast-path sums overflowed.  (pr, pc) = pixel position inside the CTA tile; (r, c) = in the image.
template <int PB>
__device__ __noinline__ float exact_side_ratio(const float *__restrict__ sGi, const float *__restrict__ sGj,
                                               const float *__restrict__ sUj, int GJW, int UJW, int pr, int pc,
                                               int r, int c, int a, int ny, int nx, float neg_c, int lane,
                                               __nv_bfloat16 *__restrict__ wpix, size_t wstride)
{
    // wpix (optional): slot of this pixel in offset 0 of its stored-weight chunk; offset stride wstride
    constexpr int GIW = SweepGeom<PB>::GIW;
    const int W = 2 * a + 1;
    float dmin = 3.0e38f;
    for (int pass = 0; pass < 2; ++pass) {
        float z = 0.f, aa = 0.f, dm = 3.0e38f;
        for (int idx = lane; idx < W * W; idx += 32) {
            const int dr = idx / W - a, dc = idx % W - a;
            if ((unsigned)(r + dr) >= (unsigned)ny || (unsigned)(c + dc) >= (unsigned)nx) {
                if (pass == 1 && wpix) wpix[(size_t)idx * wstride] = __float2bfloat16_rn(0.f);
                continue;
            }
            float D = 0.f;
            for (int y = 0; y <= 2 * PB; ++y)
                for (int x = 0; x <= 2 * PB; ++x) {
                    const float df = sGi[(pr + y) * GIW + pc + x] - sGj[(pr + dr + a + y) * GJW + pc + dc + a + x];
                    D = fmaf(df, df, D);
                }
            if (pass == 0) {
                dm = fminf(dm, D);
            } else {
                float e = exp2f(neg_c * (D - dmin));
                if (wpix) {                        // the sweeps that follow see exactly the stored value
                    const __nv_bfloat16 eh = __float2bfloat16_rn(e);
                    wpix[(size_t)idx * wstride] = eh;
                    e = __bfloat162float(eh);
                }
                z += e;
                aa = fmaf(e, sUj[(pr + dr + a) * UJW + pc + dc + a], aa);
            }
        }
        if (pass == 0) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) dm = fminf(dm, __shfl_xor_sync(0xffffffffu, dm, o));
            dmin = dm;
        } else {
            z = warp_sum(z);
            aa = warp_sum(aa);
            return aa / z;
        }
    }
    return 0.f;
}

// One Gauss-Jacobi sweep of Eq. (7) for every pixel of every phase of every slice.
// grid.x = (S*N) * tiles_y * tiles_x; block = 64 * nb threads; warp w: band = w >> 1, side = w & 1.
template <int PB, int RB, bool STORE_W>
__global__ void __launch_bounds__(256, 1)
gj_sweep_kernel(SweepParams p, const float *__restrict__ g, const float *__restrict__ u, float *__restrict__ out,
                __nv_bfloat16 *__restrict__ wts)
{
    using GEO = SweepGeom<PB>;
    constexpr int C = SW_C, G = SW_G, NGI = GEO::NGI, NGJ = GEO::NGJ, NUJ = GEO::NUJ, GIW = GEO::GIW;
    constexpr int NQ = C + 2 * PB;             // squared differences per offset and row
    constexpr int RING = (PB > 0) ? 2 * PB : 1;
    const int a = p.a, ng = p.ngroups, nb = p.nb, nx = p.nx, ny = p.ny;
    const int TH = nb * RB;
    const int GJW = GEO::gjw(ng), UJW = GEO::ujw(ng);
    const int gi_rows = TH + 2 * PB, gj_rows = TH + 2 * PB + 2 * a, uj_rows = TH + 2 * a;

    extern __shared__ float4 smem4[];
    float *sGi = reinterpret_cast<float *>(smem4);
    float *sGj = sGi + gi_rows * GIW;              // [2][gj_rows][GJW]
    float *sUj = sGj + 2 * gj_rows * GJW;          // [2][uj_rows][UJW]
    float *sK = sUj + 2 * uj_rows * UJW;           // [2*nb][RB][128]

    const int tiles_per_img = p.tiles_x * p.tiles_y;
    const int img = blockIdx.x / tiles_per_img;    // slice*N + phase
    const int tl = blockIdx.x - img * tiles_per_img;
    const int tile_r0 = (tl / p.tiles_x) * TH, tile_c0 = (tl % p.tiles_x) * SW_TW;
    const int slice = img / p.n_phase, phase = img - slice * p.n_phase;
    const size_t npix = (size_t)nx * ny;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = 2 * nb;

    {   // stage g_i, and g_j / u_j of both cyclic neighbours (L81), zero-filled outside the image
        const float *__restrict__ gi = g + (size_t)img * npix;
        stage_tile_async(sGi, gi_rows, GIW, gi, tile_r0 - PB, tile_c0 - PB, ny, nx, warp, nwarps, lane);
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int j = (phase + (s == 0 ? p.n_phase - 1 : 1)) % p.n_phase;
            const size_t jo = ((size_t)slice * p.n_phase + j) * npix;
            stage_tile_async(sGj + s * gj_rows * GJW, gj_rows, GJW, g + jo, tile_r0 - PB - a, tile_c0 - PB - a, ny, nx,
                             warp, nwarps, lane);
            stage_tile_async(sUj + s * uj_rows * UJW, uj_rows, UJW, u + jo, tile_r0 - a, tile_c0 - a, ny, nx, warp,
                             nwarps, lane);
        }
        cp_async_commit();
        cp_async_wait<0>();
    }
    __syncthreads();

    const int side = warp & 1, band = warp >> 1;
    const int lr0 = band * RB;                     // first pixel row of the band inside the tile
    const int r0 = tile_r0 + lr0, c0 = tile_c0 + C * lane;
    const float *__restrict__ myGj = sGj + side * gj_rows * GJW;
    const float *__restrict__ myUj = sUj + side * uj_rows * UJW;
    float *__restrict__ myK = sK + warp * RB * SW_TW;

    // ---- reference exponents K(x) = c*D0(x) - margin, D0 = distance at delta = 0 (same march, one offset)
    {
        float D0[C], ring[C][RING];
#pragma unroll
        for (int c = 0; c < C; ++c) D0[c] = 0.f;
        const float *__restrict__ gip = sGi + lr0 * GIW + C * lane;
        const float *__restrict__ gjp = myGj + (lr0 + a) * GJW + C * lane + a;
#pragma unroll
        for (int s = 0; s < RB + 2 * PB; ++s) {
            float sd[NQ], H[C];
#pragma unroll
            for (int q = 0; q < NQ; ++q) sd[q] = gip[s * GIW + q] - gjp[s * GJW + q];
            float h = sd[0] * sd[0];
#pragma unroll
            for (int q = 1; q <= 2 * PB; ++q) h = fmaf(sd[q], sd[q], h);
            H[0] = h;
#pragma unroll
            for (int c = 1; c < C; ++c) {
                h = fmaf(sd[c + 2 * PB], sd[c + 2 * PB], h);
                h = fmaf(-sd[c - 1], sd[c - 1], h);
                H[c] = h;
            }
#pragma unroll
            for (int c = 0; c < C; ++c) {
                D0[c] += H[c];
                if (s >= 2 * PB) {
                    myK[(s - 2 * PB) * SW_TW + C * lane + c] = fmaf(D0[c], p.pos_c, -p.margin);
                    D0[c] -= (PB > 0) ? ring[c][s % RING] : H[c];
                }
                ring[c][s % RING] = H[c];
            }
        }
    }
    __syncwarp();

    // ---- the window: items (dr, 4 consecutive dc), accumulators in registers
    // (column pairs: the vertical sums, exponents and accumulations issue as packed f32x2 instructions,
    // which halves their issue slots; the FP32 pipe does the same lane work either way)
    float2 Z[RB][C / 2], A[RB][C / 2];
#pragma unroll
    for (int rr = 0; rr < RB; ++rr)
#pragma unroll
        for (int cp = 0; cp < C / 2; ++cp) { Z[rr][cp] = make_float2(0.f, 0.f); A[rr][cp] = make_float2(0.f, 0.f); }
    const float2 negc2 = make_float2(p.neg_c, p.neg_c), neg1 = make_float2(-1.f, -1.f);

    // stored-weight chunk of this warp: [W*W][RB][128] halves
    constexpr size_t WSTRIDE = (size_t)RB * SW_TW;         // halves per offset
    __nv_bfloat16 *__restrict__ wchunk = nullptr;
    uint64_t wpol = 0;                                     // L2 policy of this chunk's stores (see SweepParams::res_tasks)
    if (STORE_W) {
        const size_t gband = (size_t)(tile_r0 / RB) + band, tx = tile_c0 / SW_TW;
        // (chosen per CTA, from its first band: uniform, so the policy lives in a uniform register)
        const long long chunk = ((long long)img * ((ny + RB - 1) / RB) + (long long)(tile_r0 / RB)) * p.tiles_x + (long long)tx;
        wpol = (chunk * (RB / 2) < p.res_tasks) ? l2_policy_evict_last() : l2_policy_evict_first();
        wchunk = wts + ((((size_t)img * p.nbands + gband) * p.tiles_x + tx) * 2 + side) *
                           (size_t)((2 * a + 1) * (2 * a + 1)) * WSTRIDE;
    }

    for (int dr = -a; dr <= a; ++dr) {
        unsigned okmask = 0;                       // pixel row and candidate row inside the image
#pragma unroll
        for (int rr = 0; rr < RB; ++rr)
            if (r0 + rr < ny && (unsigned)(r0 + rr + dr) < (unsigned)ny) okmask |= 1u << rr;
        if (!STORE_W && okmask == 0) continue;     // (stored planes must be written even when all-zero)
        for (int dcg = 0; dcg < ng; ++dcg) {
            const int dc0 = -a + G * dcg;
            float2 D[G][C / 2], ring[G][C / 2][RING];
#pragma unroll
            for (int gg = 0; gg < G; ++gg)
#pragma unroll
                for (int cp = 0; cp < C / 2; ++cp) {
                    const int col = c0 + 2 * cp + dc0 + gg;
                    const bool in_win = dc0 + gg <= a;
                    D[gg][cp].x = (in_win && (unsigned)col < (unsigned)nx) ? 0.f : p.big_d;
                    D[gg][cp].y = (in_win && (unsigned)(col + 1) < (unsigned)nx) ? 0.f : p.big_d;
                }
            const float4 *__restrict__ gip = reinterpret_cast<const float4 *>(sGi + lr0 * GIW) + lane;
            const float4 *__restrict__ gjp = reinterpret_cast<const float4 *>(myGj + (lr0 + dr + a) * GJW) + lane + dcg;
            const float4 *__restrict__ ujp = reinterpret_cast<const float4 *>(myUj + (lr0 + dr + a) * UJW) + lane + dcg;
            const float4 *__restrict__ kp = reinterpret_cast<const float4 *>(myK) + lane;
            uint2 held[G];                         // STORE_W: packed weights of the even row of a pair
            __nv_bfloat16 *__restrict__ witem =
                STORE_W ? wchunk + ((size_t)(dr + a) * (2 * a + 1) + (dc0 + a)) * WSTRIDE + 8 * lane : nullptr;
#pragma unroll
            for (int s = 0; s < RB + 2 * PB; ++s) {
                float gi_[4 * NGI], gj_[4 * NGJ];
#pragma unroll
                for (int k = 0; k < NGI; ++k) {
                    const float4 v = gip[s * (GIW / 4) + k];
                    gi_[4 * k] = v.x; gi_[4 * k + 1] = v.y; gi_[4 * k + 2] = v.z; gi_[4 * k + 3] = v.w;
                }
#pragma unroll
                for (int k = 0; k < NGJ; ++k) {
                    const float4 v = gjp[s * (GJW / 4) + k];
                    gj_[4 * k] = v.x; gj_[4 * k + 1] = v.y; gj_[4 * k + 2] = v.z; gj_[4 * k + 3] = v.w;
                }
                float uj_[4 * NUJ];
                float2 K_[C / 2];
                if (s >= 2 * PB) {                 // this step completes the window of pixel row rr
                    const int rr = s - 2 * PB;
                    // rows whose pixel or candidate row is outside the image get K = -huge: weight 0
                    const bool ok = (okmask >> rr) & 1u;
#pragma unroll
                    for (int k = 0; k < NUJ; ++k) {
                        const float4 v = ujp[rr * (UJW / 4) + k];
                        uj_[4 * k] = v.x; uj_[4 * k + 1] = v.y; uj_[4 * k + 2] = v.z; uj_[4 * k + 3] = v.w;
                    }
                    const float4 kv = kp[rr * (SW_TW / 4)];
                    K_[0].x = ok ? kv.x : -1.0e30f; K_[0].y = ok ? kv.y : -1.0e30f;
                    K_[1].x = ok ? kv.z : -1.0e30f; K_[1].y = ok ? kv.w : -1.0e30f;
                }
#pragma unroll
                for (int gg = 0; gg < G; ++gg) {
                    // squared differences and the horizontal box sums of this row for offset gg
                    float sd[NQ], H[C];
#pragma unroll
                    for (int q = 0; q < NQ; ++q) sd[q] = gi_[q] - gj_[q + gg];
                    float h = sd[0] * sd[0];
#pragma unroll
                    for (int q = 1; q <= 2 * PB; ++q) h = fmaf(sd[q], sd[q], h);
                    H[0] = h;
#pragma unroll
                    for (int c = 1; c < C; ++c) {
                        h = fmaf(sd[c + 2 * PB], sd[c + 2 * PB], h);
                        h = fmaf(-sd[c - 1], sd[c - 1], h);
                        H[c] = h;
                    }
                    float2 e_[C / 2];
#pragma unroll
                    for (int cp = 0; cp < C / 2; ++cp) {
                        const float2 H2 = make_float2(H[2 * cp], H[2 * cp + 1]);
                        D[gg][cp] = __fadd2_rn(D[gg][cp], H2);
                        if (s >= 2 * PB) {
                            const int rr = s - 2 * PB;
                            const float2 t2 = __ffma2_rn(D[gg][cp], negc2, K_[cp]);
                            const float2 e2 = make_float2(fast_ex2(t2.x), fast_ex2(t2.y));
                            if (STORE_W) e_[cp] = e2;
                            Z[rr][cp] = __fadd2_rn(Z[rr][cp], e2);
                            A[rr][cp] = __ffma2_rn(e2, make_float2(uj_[2 * cp + gg], uj_[2 * cp + gg + 1]), A[rr][cp]);
                            D[gg][cp] = __ffma2_rn((PB > 0) ? ring[gg][cp][s % RING] : H2, neg1, D[gg][cp]);
                        }
                        ring[gg][cp][s % RING] = H2;
                    }
                    if (STORE_W && s >= 2 * PB) {  // 4 bf16 weights of row rr, offset gg
                        const int rr = s - 2 * PB;
                        const __nv_bfloat162 lo = __floats2bfloat162_rn(e_[0].x, e_[0].y), hi = __floats2bfloat162_rn(e_[1].x, e_[1].y);
                        uint2 pk;
                        pk.x = *reinterpret_cast<const unsigned *>(&lo);
                        pk.y = *reinterpret_cast<const unsigned *>(&hi);
                        // rows 2q and 2q+1 share one 16-byte slot per lane (plane_off): the even row waits in
                        // registers for one step, then one STG.128 per offset and row pair (8-byte stores at a
                        // 16-byte stride cost 20 us more per cfg-2 sweep)
                        if (rr & 1) {
                            if (dc0 + gg <= a)     // (rows / columns past the image edge land in chunk padding)
                                stg128_hint(witem + gg * WSTRIDE + (rr >> 1) * 256, make_uint4(held[gg].x, held[gg].y, pk.x, pk.y), wpol);
                        } else {
                            held[gg] = pk;
                        }
                    }
                }
                SW_STEP_FENCE();
            }
        }
    }

    // ---- softmax-weighted mean per pixel; overflowed pixels take the exact two-pass route
#pragma unroll
    for (int rr = 0; rr < RB; ++rr)
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const bool valid = (r0 + rr < ny) && (c0 + c < nx);
            float &Arc = (c & 1) ? A[rr][c >> 1].y : A[rr][c >> 1].x;
            const float Zrc = (c & 1) ? Z[rr][c >> 1].y : Z[rr][c >> 1].x;
            const bool bad = valid && (!(Zrc < p.z_limit) || !(fabsf(Arc) < p.a_limit));
            Arc = Arc / Zrc;
            unsigned m = __ballot_sync(0xffffffffu, bad);
            while (m) {
                const int L = __ffs(m) - 1;
                m &= m - 1;
                __nv_bfloat16 *wpix = STORE_W ? wchunk + plane_off(rr, C * L + c) : nullptr;
                __syncwarp();                      // the fast path's stores to this pixel come first
                const float v = exact_side_ratio<PB>(sGi, myGj, myUj, GJW, UJW, lr0 + rr, C * L + c, r0 + rr,
                                                     tile_c0 + C * L + c, a, ny, nx, p.neg_c, lane, wpix, WSTRIDE);
                if (lane == L) Arc = v;
            }
        }

    // ---- combine the two sides (Eq. 7): side-1 warps hand their means to the side-0 warp of the band
    if (side == 1) {
#pragma unroll
        for (int rr = 0; rr < RB; ++rr)
            reinterpret_cast<float4 *>(myK)[rr * (SW_TW / 4) + lane] = make_float4(A[rr][0].x, A[rr][0].y, A[rr][1].x, A[rr][1].y);
    }
    __syncthreads();
    if (side == 0) {
        const float *__restrict__ other = sK + (warp + 1) * RB * SW_TW;
        float *__restrict__ o = out + (size_t)img * npix;
        const bool vec = ((nx & 3) == 0) && ((reinterpret_cast<uintptr_t>(out) & 15) == 0) && (c0 + C <= nx);
#pragma unroll
        for (int rr = 0; rr < RB; ++rr) {
            const int r = r0 + rr;
            if (r >= ny) break;
            const float4 ov = reinterpret_cast<const float4 *>(other)[rr * (SW_TW / 4) + lane];
            const float on[C] = {ov.x, ov.y, ov.z, ov.w};
            float v[C];
#pragma unroll
            for (int c = 0; c < C; ++c) {
                const float gc = sGi[(lr0 + rr + PB) * GIW + C * lane + PB + c];
                v[c] = fmaf(p.c_nb, ((c & 1) ? A[rr][c >> 1].y : A[rr][c >> 1].x) + on[c], p.c_self * gc);
                if (p.clip) v[c] = fmaxf(v[c], 0.f);
            }
            if (vec) {
                *reinterpret_cast<float4 *>(o + (size_t)r * nx + c0) = make_float4(v[0], v[1], v[2], v[3]);
            } else {
#pragma unroll
                for (int c = 0; c < C; ++c)
                    if (c0 + c < nx) o[(size_t)r * nx + c0 + c] = v[c];
            }
        }
    }
}

// ---- sweeps 2..M2 from the stored weights (opt-in, option weight_cache_mb > 0) ---------------------------------
// u_i'(x) = g_i(x)/(1+mu) + mu/(2mu+2) * sum over the two sides of (sum_delta w u_j(x+delta)) / (sum_delta w), with w
// read back as bf16: 2 bytes per weight, HBM bound.  One CTA per stored band (chunk) of rb rows x 128 columns; warp k
// owns the ROW PAIR 2k, 2k+1 (lane l: columns 4l..4l+3 of both rows).  The row-pair interleave of the stored layout
// (plane_off) makes a warp's share of one offset plane a contiguous piece of 512 bytes, 16 bytes per lane, so the
// 2 W^2 pieces of a warp (both sides) are one uninterrupted stream with a constant stride, kept DEPTH pieces deep
// in a private cp.async ring (LDGSTS: no registers held by loads in flight, no mbarriers, no producer warp).  The
// u_j windows of BOTH sides (rb + 2a rows each, zero-filled outside the image; excluded candidates carry weight 0
// in the chunks) are staged once by all threads of the CTA.  Measured on the box: a 322 MB
// read-only stream of this shape runs at 6.2 TB/s; this kernel reaches 5.7-5.8 TB/s (0.87-0.89 of the copy peak).
// Two earlier formulations were measured and removed in round 3: one CTA per band fed by a producer warp through a
// cp.async.bulk (TMA) ring with mbarriers (72 us per cfg-2 sweep: bulk copies alone, no arithmetic, streamed the same
// bytes at 4.9 TB/s for any stage size and depth) and persistent warp tasks with private windows (62 us: two ring
// restarts per task and 3x the window bytes from L2); this one takes 56-57 us.  All three were bit-identical.
// grid.x = chunks = (S*N) * bands that hold image rows * tiles_x; block = 32 * rb/2; dynamic smem = apply3_smem_bytes.
__host__ __device__ inline int apply_uw(int window) { return 124 + 4 * ((window + 3) / 4 + 1); }
__host__ __device__ inline size_t apply3_smem_bytes(int window, int rb, int depth)
{
    const int a = (window - 1) / 2;
    return (size_t)2 * (rb + 2 * a) * apply_uw(window) * sizeof(float) + (size_t)(rb / 2) * depth * 512;
}

// (Writing the weight sums Z in the first applying sweep and reading them back in the later ones -- 8 fewer
// instructions per piece -- was measured here too and left the sweep at 55.7 us: dropped.)
template <int DEPTH>             // pieces in flight per warp (a power of two)
__global__ void __launch_bounds__(160, 4)
gj_apply3_kernel(SweepParams p, const float *__restrict__ g, const float *__restrict__ u, float *__restrict__ out,
                 const __nv_bfloat16 *__restrict__ wts)
{
    constexpr int C = SW_C;
    const int a = p.a, nx = p.nx, ny = p.ny, W = 2 * a + 1, WW = W * W;
    const int rb = p.rb, npairs = rb >> 1, urows = rb + 2 * a, UW = apply_uw(W);
    const size_t pstride = (size_t)rb * (SW_TW / 8);     // uint4 per offset plane
    const size_t npix = (size_t)nx * ny;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    extern __shared__ float4 smem4[];
    float *sU = reinterpret_cast<float *>(smem4);                                            // [2][urows][UW]
    const unsigned ring_s = smem_u32(sU + 2 * urows * UW) + warp * (DEPTH * 512) + 16 * lane; // [npairs][DEPTH][32] x 16 B

    const int tiles_per_img = p.tiles_x * p.tiles_y;       // tiles_y = bands that hold image rows
    const long long n_chunks = (long long)p.n_img * tiles_per_img;
    const long long chunk = p.ap_reverse ? n_chunks - 1 - (long long)blockIdx.x : (long long)blockIdx.x;
    const int img = (int)(chunk / tiles_per_img);
    const int tl = (int)(chunk - (long long)img * tiles_per_img);
    const int gband = tl / p.tiles_x, tx = tl - gband * p.tiles_x;
    const int tile_r0 = gband * rb, tile_c0 = tx * SW_TW, c0 = tile_c0 + C * lane;
    const int r = tile_r0 + 2 * warp;
    const int slice = img / p.n_phase, phase = img - slice * p.n_phase;
    const uint64_t pol = chunk * npairs < p.res_tasks ? l2_policy_evict_last() : l2_policy_evict_first();

    // oldest group: both windows (all threads of the CTA)
#pragma unroll
    for (int sd = 0; sd < 2; ++sd) {
        const int j = (phase + (sd == 0 ? p.n_phase - 1 : 1)) % p.n_phase;
        stage_tile_async(sU + sd * urows * UW, urows, UW, u + ((size_t)slice * p.n_phase + j) * npix, tile_r0 - a, tile_c0 - a,
                         ny, nx, warp, npairs, lane);
    }
    cp_async_commit();
    // this warp's pieces: 0 .. WW-1 of side 0, then WW .. 2 WW-1 of side 1: one stream at a constant stride (the two
    // sides of a band are contiguous in the stored layout)
    const uint4 *__restrict__ nextp = reinterpret_cast<const uint4 *>(wts) +
                                      ((((size_t)img * p.nbands + gband) * p.tiles_x + tx) * 2) * (size_t)WW * pstride + warp * 32 + lane;
    unsigned issued = 0, wr = ring_s;
    const unsigned total = 2u * (unsigned)WW;
#pragma unroll 1
    for (; issued < DEPTH - 1; ++issued) {
        cp_async16_s_hint(wr, nextp, issued < total, pol);
        cp_async_commit();
        wr += 512;
        nextp += pstride;
    }
    cp_async_wait<DEPTH - 1>();                               // this thread's window copies have landed
    __syncthreads();                                          // ... and everybody else's
    float nbsum[2][C] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    unsigned rd = 0;                                          // ring offset of the piece consumed next
    const int wfull = W & ~3, wtail = W & 3;                  // offsets of a window row in groups of four, and the rest
#pragma unroll 1
    for (int sd = 0; sd < 2; ++sd) {
        float Z[2][C] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}}, A[2][C] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
        const float *__restrict__ uwin = sU + (sd * urows + 2 * warp) * UW + C * lane;
        // one piece: issue the piece DEPTH-1 ahead, wait for the oldest, accumulate its 2 x 4 weights
        auto piece = [&](const float (&uw0)[8], const float (&uw1)[8], int jj) {
            cp_async16_s_hint(wr, nextp, issued < total, pol);
            cp_async_commit();                                // (empty groups keep the wait count uniform)
            ++issued;
            nextp += pstride;
            wr = (wr == ring_s + (DEPTH - 1) * 512) ? ring_s : wr + 512;
            cp_async_wait<DEPTH - 1>();                       // the oldest piece has landed (this lane's own 16 bytes)
            const uint4 wv = lds128_s(ring_s + rd);
            rd = (rd + 512) & ((DEPTH - 1) << 9);
            // bf16 -> fp32 is a 16-bit shift: low half << 16, high half masked
            const float w0[C] = {__uint_as_float(wv.x << 16), __uint_as_float(wv.x & 0xffff0000u),
                                 __uint_as_float(wv.y << 16), __uint_as_float(wv.y & 0xffff0000u)};
            const float w1[C] = {__uint_as_float(wv.z << 16), __uint_as_float(wv.z & 0xffff0000u),
                                 __uint_as_float(wv.w << 16), __uint_as_float(wv.w & 0xffff0000u)};
#pragma unroll
            for (int c = 0; c < C; ++c) {
                Z[0][c] += w0[c];
                A[0][c] = fmaf(w0[c], uw0[c + jj], A[0][c]);
                Z[1][c] += w1[c];
                A[1][c] = fmaf(w1[c], uw1[c + jj], A[1][c]);
            }
        };
#pragma unroll 1
        for (int dr = 0; dr < W; ++dr) {
            const float *__restrict__ urow0 = uwin + dr * UW;
#pragma unroll 1
            for (int k = 0; k <= W - 1; k += 4) {
                const float4 ua = *reinterpret_cast<const float4 *>(urow0 + k), ub = *reinterpret_cast<const float4 *>(urow0 + k + 4);
                const float4 uc = *reinterpret_cast<const float4 *>(urow0 + UW + k), ud = *reinterpret_cast<const float4 *>(urow0 + UW + k + 4);
                const float uw0[8] = {ua.x, ua.y, ua.z, ua.w, ub.x, ub.y, ub.z, ub.w};
                const float uw1[8] = {uc.x, uc.y, uc.z, uc.w, ud.x, ud.y, ud.z, ud.w};
                if (k < wfull) {                              // a full group of four offsets: no per-piece test
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) piece(uw0, uw1, jj);
                } else {
#pragma unroll
                    for (int jj = 0; jj < 3; ++jj)
                        if (jj < wtail) piece(uw0, uw1, jj);
                }
            }
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {
            nbsum[0][c] += A[0][c] / Z[0][c];
            nbsum[1][c] += A[1][c] / Z[1][c];
        }
    }
    if (c0 < nx) {
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            if (r + q < ny) {
                const float *__restrict__ gi = g + (size_t)img * npix + (size_t)(r + q) * nx + c0;
                float *__restrict__ o = out + (size_t)img * npix + (size_t)(r + q) * nx + c0;
#pragma unroll
                for (int c = 0; c < C; ++c)
                    if (c0 + c < nx) {
                        float v = fmaf(p.c_nb, nbsum[q][c], p.c_self * __ldg(gi + c));
                        if (p.clip) v = fmaxf(v, 0.f);
                        o[c] = v;
                    }
            }
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
