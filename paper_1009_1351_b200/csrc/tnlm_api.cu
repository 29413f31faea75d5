// tnlm_api.cu -- C ABI of libtnlm (see include/tnlm.h): handle, argument checks, workspace,
// and the launch sequences of the five operations.  Host code only orchestrates; every step
// of the path runs in the kernels of projector.cuh, cgls.cuh and regularize.cuh.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "../../include/tnlm.h"
#include "cgls.cuh"
#include "common.cuh"
#include "fbp.cuh"
#include "projector.cuh"
#include "regularize.cuh"

using namespace tnlm;

static constexpr int MAX_PATCH = 9, MAX_WINDOW = 31;

// One compiled shape of gj_sweep_kernel<PB, RB> with nb row bands per CTA (regularize.cuh).
struct SweepShape {
    const void *fn = nullptr;       // compute only
    const void *fn_store = nullptr; // compute and store the weights (first of several sweeps)
    int rb = 0, nb = 0, occ = 0;    // rows per band, bands per CTA, resident CTAs per SM
    size_t smem = 0;
};

struct tnlm_handle {
    int nx = 0, ny = 0, n_phase = 0, window = 0, patch = 0;
    float h = 0.f, mu = 0.f;
    bool has_geom = false;
    bool fan_poly = true;   // every pixel is seen within +-45 degrees of the central ray: polynomial atan
    Geom G{};
    SweepParams R{};
    std::vector<SweepShape> shapes;   // launchable sweep shapes for this (window, patch)
    int device = 0;         // the CUDA device the handle was created on; every entry point runs there
    int n_sm = 148;
    size_t smem_per_sm = 233472;
    // tuning knobs, read once from the environment at tnlm_create (tnlm_set_option changes them later)
    long long opt_cache_mb = 0;   // 0 (default): every sweep computes the weights in fp32; > 0: sweeps 2..m2 read stored bf16 weights
    int opt_rb = 0, opt_nb = 0;
    int opt_project = -1;   // 1: project_strip_kernel (shared-memory strips per warp); 0: project_kernel (L1 gathers); -1: by size
    int opt_depth = 0;      // gj_apply3_kernel ring depth override (0 = the deepest of 8, 4 that fits)
    int opt_project_il = 1;         // forward projector: groups of four slices read interleaved copies (project_il_kernel)
    int opt_project_block = 128;    // project_kernel / project_il_kernel: threads per CTA (256, 128, 64; 128 measured 2-3 % faster than 256: tail balance)
    int opt_backproject_group = 16; // backproject_kernel: at most this many slices of a batch per thread (16, 8, 4, 2 or 1)
    int opt_snake = 1;      // gj_apply3_kernel: successive sweeps take the stored bands in opposite orders
    long long opt_resident_mb = 32;   // MB of stored weights marked evict_last in L2 (the rest evict_first); 0 = none
    // geometry tables (device)
    RayEntry *d_tab = nullptr;
    RayRange *d_rng = nullptr;
    float4 *d_views = nullptr;
    int4 *d_split = nullptr;         // per (phase, view): the runs of steep / shallow bins (backproject_kernel)
    // FBP initialisation (fbp.cuh): ramp filter table, cosine weights, view weights; filtered sinograms
    double *d_fbp_g = nullptr;
    float *d_fbp_cosw = nullptr, *d_fbp_wv = nullptr;
    float *d_fbp_q = nullptr;
    // workspace, sized for ws_slices
    int ws_slices = 0;
    float *d_s = nullptr, *d_t = nullptr, *d_g = nullptr, *d_f = nullptr;  // images
    float *d_ua = nullptr, *d_ub = nullptr;                                  // sweep ping-pong
    float *d_imT = nullptr;                                                  // transposed image of the forward projector
    float *d_imI = nullptr;                                                  // its interleaved copy (groups of four slices)
    float *d_r = nullptr, *d_rw = nullptr, *d_q = nullptr, *d_sw = nullptr;  // sinograms (d_sw = sqrt(w))
    float *d_yh = nullptr, *d_wh = nullptr;                                  // host-API staging
    __nv_bfloat16 *d_wts = nullptr;          // stored weights of the sweeps (layout: regularize.cuh)
    size_t wts_cap = 0;               // in halves
    size_t apply_smem = 0;
    double *d_scal = nullptr;
    int scal_cap = 0;
    long long launches = 0;
    // optional per-launch timing of every kernel of the path (tnlm_profile_kernels / tnlm_kernel_times)
    bool prof = false;
    std::vector<cudaEvent_t> prof_ev;     // 2 events per timed launch
    std::vector<int> prof_kind;
    std::string err;
};

static thread_local std::string g_create_error;     // message of the last failed tnlm_create of this thread

// NVTX range around a C-ABI call (visible in nsys / ncu --nvtx; free when no tool is attached).
struct NvtxRange {
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

// Makes the handle's device current for the duration of a call and restores the caller's.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) {
            err = cudaSetDevice(dev);
            switched = (err == cudaSuccess);
        }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

static int fail(tnlm_handle *h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}
static int cuda_fail(tnlm_handle *h, cudaError_t e, const char *what)
{
    return fail(h, TNLM_CUDA_ERROR, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(h, call)                                                    \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return cuda_fail(h, e__, #call);       \
    } while (0)
#define LAUNCHED(h)                                                    \
    do {                                                               \
        (h)->launches++;                                               \
        cudaError_t e__ = cudaGetLastError();                          \
        if (e__ != cudaSuccess) return cuda_fail(h, e__, "kernel launch"); \
    } while (0)

extern "C" const char *tnlm_version(void) { return "tnlm-b200 0.3 (sm_100a)"; }

extern "C" const char *tnlm_last_error(const tnlm_handle *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

extern "C" long long tnlm_launch_count(const tnlm_handle *h) { return h ? h->launches : 0; }

// ------------------------------------------------------------------------------ tables
// Ray (phase i, view v, bin k) in grid units (pixel c covers [c, c+1) in xi, row r in eta):
// source (xs, es), unit direction (dx, dy).  Steep (|dy| >= |dx|): xi(eta) = p0 + m*eta with
// m = dx/dy, p0 = xs - m*es, length per full row = pix/|dy|.  Shallow: roles swapped.
// Returns false if some view has more than three runs of steep / shallow bins (a fan of 180 degrees or more).
static bool build_tables(const tnlm_geometry &g, int nx, int ny, int n_phase, std::vector<RayEntry> &tab,
                         std::vector<RayRange> &rng, std::vector<float4> &views, std::vector<int4> &split)
{
    const int V = g.n_views, B = g.n_bins;
    tab.resize((size_t)n_phase * V * B);
    rng.resize(tab.size());
    views.resize((size_t)n_phase * V);
    split.resize((size_t)n_phase * V);
    bool ok = true;
    for (int i = 0; i < n_phase; ++i)
        for (int v = 0; v < V; ++v) {
            const double th = g.angles_rad[(size_t)i * V + v];
            const double sx = g.sid_mm * std::cos(th), sy = g.sid_mm * std::sin(th);
            views[(size_t)i * V + v] = make_float4((float)sx, (float)sy, (float)std::cos(th), (float)std::sin(th));
            const double xs = sx / g.pixel_mm + 0.5 * nx, es = sy / g.pixel_mm + 0.5 * ny;
            for (int k = 0; k < B; ++k) {
                const double gam = ((double)k - 0.5 * (B - 1) + g.bin_offset) * g.bin_pitch_mm / g.sdd_mm;
                const double dx = -std::cos(th + gam), dy = -std::sin(th + gam);
                const bool steep = std::fabs(dy) >= std::fabs(dx);
                const double m = steep ? dx / dy : dy / dx;
                const double p0 = steep ? xs - m * es : es - m * xs;
                const double len = g.pixel_mm / (steep ? std::fabs(dy) : std::fabs(dx));
                RayEntry e;
                e.m = (float)m;
                e.plo = (float)(p0 + std::fmin((double)e.m, 0.0));
                e.len = (float)(steep ? len : -len);
                e.inva = (e.m != 0.f) ? 1.0f / std::fabs(e.m) : 1e30f;
                // walk range along the major axis: where the minor coordinate is within [-1, n+1]
                const int n_major = steep ? ny : nx, n_minor = steep ? nx : ny;
                int lo = 0, hi = n_major - 1;
                if (e.m != 0.f) {
                    double q0 = (-1.0 - p0) / m, q1 = ((double)n_minor + 1.0 - p0) / m;
                    if (q0 > q1) std::swap(q0, q1);
                    lo = (int)std::fmax(0.0, std::floor(q0) - 1.0);
                    hi = (int)std::fmin((double)(n_major - 1), std::floor(q1) + 1.0);
                } else if (p0 < 0.0 || p0 >= (double)n_minor) {
                    hi = -1;
                }
                RayRange r;
                r.lo = (short)lo; r.hi = (short)hi;
                // interior: lo(q) = m*q + plo within [0.5, n_minor - 2.5], so that the fp32 floor c0 and c0+1
                // are inside whatever the rounding; lo(q) is linear in q, so the rows form one interval
                r.ilo = 0; r.ihi = -1;
                if (hi >= lo) {
                    const double plo = p0 + std::fmin(m, 0.0), a0 = 0.5, a1 = (double)n_minor - 2.5;
                    double q0 = (double)lo, q1 = (double)hi;
                    if (e.m != 0.f) {
                        double t0 = (a0 - plo) / m, t1 = (a1 - plo) / m;
                        if (t0 > t1) std::swap(t0, t1);
                        q0 = std::fmax(q0, std::ceil(t0) + 1.0);
                        q1 = std::fmin(q1, std::floor(t1) - 1.0);
                    } else if (!(plo >= a0 && plo <= a1)) {
                        q1 = q0 - 1.0;
                    }
                    if (q1 >= q0) { r.ilo = (short)q0; r.ihi = (short)q1; }
                }
                tab[((size_t)i * V + v) * B + k] = e;
                rng[((size_t)i * V + v) * B + k] = r;
            }
            // runs of steep (len > 0) / shallow bins of this view: [0, s1) and [s2, B) of class c0, [s1, s2) of the other
            const RayEntry *row = &tab[((size_t)i * V + v) * B];
            const int c0 = row[0].len > 0.f ? 1 : 0;
            int s1 = B, s2 = B, runs = 1;
            for (int k = 1; k < B; ++k)
                if ((row[k].len > 0.f) != (row[k - 1].len > 0.f)) {
                    ++runs;
                    if (runs == 2) s1 = k; else if (runs == 3) s2 = k;
                }
            if (runs > 3) ok = false;
            split[(size_t)i * V + v] = make_int4(s1, s2, c0, 0);
        }
    return ok;
}

// Every compiled (PB, RB) of gj_sweep_kernel, with nb in {4, 2, 1}, that fits one CTA's shared
// memory becomes a SweepShape; the launcher picks the cheapest one for the image count at hand.
template <int PB, int RB>
static cudaError_t add_sweep_shapes(tnlm_handle *H, size_t smem_limit)
{
    const void *fn = (const void *)gj_sweep_kernel<PB, RB, false>;
    const void *fn_store = (const void *)gj_sweep_kernel<PB, RB, true>;
    std::vector<SweepShape> mine;
    for (int nb = 4; nb >= 1; nb >>= 1) {
        SweepShape sh;
        sh.fn = fn; sh.fn_store = fn_store; sh.rb = RB; sh.nb = nb;
        sh.smem = SweepGeom<PB>::smem_words(H->R.a, H->R.ngroups, nb, RB) * sizeof(float);
        if (sh.smem > smem_limit) continue;
        mine.push_back(sh);
    }
    if (mine.empty()) return cudaSuccess;
    // The attribute belongs to the kernel symbol, not to the handle: always the device maximum, so that a
    // later handle with a smaller window can never lower it under a live handle's launches.
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_limit);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fn_store, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_limit);
    if (e != cudaSuccess) return e;
    for (SweepShape &sh : mine) {
        int occ_store = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&sh.occ, fn, 64 * sh.nb, sh.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_store, fn_store, 64 * sh.nb, sh.smem);
        if (e != cudaSuccess) return e;
        sh.occ = std::min(sh.occ, occ_store);
        if (sh.occ >= 1) H->shapes.push_back(sh);
    }
    return cudaSuccess;
}

static cudaError_t build_sweep_shapes(tnlm_handle *H, size_t smem_limit)
{
    cudaError_t e = cudaSuccess;
    switch ((H->patch - 1) / 2) {
        case 0: e = add_sweep_shapes<0, 8>(H, smem_limit); if (e == cudaSuccess) e = add_sweep_shapes<0, 10>(H, smem_limit); break;
        case 1: e = add_sweep_shapes<1, 8>(H, smem_limit); if (e == cudaSuccess) e = add_sweep_shapes<1, 10>(H, smem_limit); break;
        case 2: e = add_sweep_shapes<2, 8>(H, smem_limit); if (e == cudaSuccess) e = add_sweep_shapes<2, 10>(H, smem_limit); break;
        case 3: e = add_sweep_shapes<3, 8>(H, smem_limit); break;
        default: e = add_sweep_shapes<4, 4>(H, smem_limit); break;
    }
    return e;
}

// Cost model of one sweep over n_img images with shape sh, in (resident warps) x (rows marched) per SM: full waves
// of occ CTAs per SM, then the remainder spread over the SMs.  Measured on cfg 3 / cfg 4 sized sweeps: an SM with
// fewer than ~5 warps of this kernel is not faster per warp-row than one with 5 (so a remainder of half-size CTAs
// costs 0.65 of a full wave, not 0.5 and not 1); two half-size CTAs per SM hide each other's tile staging once there
// is more than one wave (-1.5 %), but stage more halo per band (+3 % in a single wave); one-band CTAs stage 2.2x
// the halo per band (+15 %).
static double sweep_cost(const tnlm_handle *H, const SweepShape &sh, int n_img)
{
    const int pb = (H->patch - 1) / 2;
    const long long th = (long long)sh.nb * sh.rb;
    const long long ctas = (long long)n_img * ((H->ny + th - 1) / th) * ((H->nx + SW_TW - 1) / SW_TW);
    const long long cap = (long long)H->n_sm * sh.occ;
    const long long full = ctas / cap, rem = ctas % cap;
    auto wave = [&](long long k) { return std::max((double)(k * 2 * sh.nb), 5.2) * (sh.rb + 2 * pb); };
    double c = (double)full * wave(sh.occ);
    if (rem) c += wave((rem + H->n_sm - 1) / H->n_sm);
    const double staging = sh.nb >= 4 ? 1.0 : (sh.nb == 2 ? (full >= 1 ? 0.985 : 1.03) : 1.15);
    return c * staging;
}

// Does some launchable sweep shape have rb rows per band and nb bands per CTA (0 = any)?
static bool sweep_shape_known(const tnlm_handle *H, int rb, int nb)
{
    for (const SweepShape &sh : H->shapes)
        if ((!rb || sh.rb == rb) && (!nb || sh.nb == nb)) return true;
    return false;
}

extern "C" int tnlm_create(const tnlm_geometry *geometry, int nx, int ny, int n_phase, int window, int patch,
                           float h, float mu, tnlm_handle **out)
{
    if (!out) return fail(nullptr, TNLM_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || n_phase < 1) return fail(nullptr, TNLM_INVALID_ARG, "nx, ny, n_phase must be >= 1");
    if (nx > 32000 || ny > 32000) return fail(nullptr, TNLM_UNSUPPORTED, "image side above 32000");
    if (window < 1 || patch < 1 || (window & 1) == 0 || (patch & 1) == 0)
        return fail(nullptr, TNLM_INVALID_ARG, "window and patch must be odd and >= 1");
    if (!(h > 0.f) || !std::isfinite(h)) return fail(nullptr, TNLM_INVALID_ARG, "h must be finite and > 0");
    if (h > 1e12f) return fail(nullptr, TNLM_INVALID_ARG, "h above 1e12: excluded candidates could no longer be given weight 0");
    if (!std::isfinite((float)(1.4426950408889634 / ((double)h * (double)h))))
        return fail(nullptr, TNLM_INVALID_ARG, "h below 1e-19: log2(e)/h^2 overflows fp32 (a zero patch distance would give NaN)");
    if (!(mu >= 0.f) || !std::isfinite(mu)) return fail(nullptr, TNLM_INVALID_ARG, "mu must be finite and >= 0");
    if (patch > MAX_PATCH || window > MAX_WINDOW)
        return fail(nullptr, TNLM_UNSUPPORTED, "patch > 9 or window > 31 not compiled");
    if (geometry) {
        const tnlm_geometry &g = *geometry;
        if (g.n_views < 1 || g.n_bins < 1 || !g.angles_rad) return fail(nullptr, TNLM_INVALID_ARG, "geometry: n_views, n_bins >= 1 and angles_rad required");
        if (!(g.sid_mm > 0) || !(g.sdd_mm > g.sid_mm)) return fail(nullptr, TNLM_INVALID_ARG, "geometry: need 0 < sid < sdd");
        if (!(g.bin_pitch_mm > 0) || !(g.pixel_mm > 0)) return fail(nullptr, TNLM_INVALID_ARG, "geometry: pitch and pixel size must be > 0");
        if (!g.detector_arc) return fail(nullptr, TNLM_UNSUPPORTED, "flat detector not built; the paper's detector is an arc");
        const double hx = 0.5 * nx * g.pixel_mm, hy = 0.5 * ny * g.pixel_mm;
        if (std::sqrt(hx * hx + hy * hy) >= g.sid_mm) return fail(nullptr, TNLM_INVALID_ARG, "geometry: image corner outside the source circle");
        if (g.sid_mm - std::sqrt(hx * hx + hy * hy) < 6.0 * g.pixel_mm)
            return fail(nullptr, TNLM_UNSUPPORTED, "geometry: source closer than six pixels to the image (the backprojector's candidate ranges assume at least that)");
        if ((long long)g.n_views * g.n_bins > 2000000000LL) return fail(nullptr, TNLM_UNSUPPORTED, "sinogram too large");
    }
    int dev = 0;
    cudaDeviceProp prop;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce == cudaSuccess) ce = cudaGetDeviceProperties(&prop, dev);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDeviceProperties");
    if (prop.major != 10) return fail(nullptr, TNLM_UNSUPPORTED, "device is not sm_100 (Blackwell B200)");

    tnlm_handle *H = new (std::nothrow) tnlm_handle();
    if (!H) return fail(nullptr, TNLM_ALLOC_FAILED, "host allocation failed");
    H->nx = nx; H->ny = ny; H->n_phase = n_phase; H->window = window; H->patch = patch; H->h = h; H->mu = mu;
    H->device = dev;
    if (const char *ev = std::getenv("TNLM_WEIGHT_CACHE_MB")) H->opt_cache_mb = std::strtoll(ev, nullptr, 10);
    if (const char *ev = std::getenv("TNLM_SWEEP_SHAPE")) std::sscanf(ev, "%d,%d", &H->opt_rb, &H->opt_nb);

    // TNLM parameters
    SweepParams &R = H->R;
    R.nx = nx; R.ny = ny; R.n_phase = n_phase; R.a = (window - 1) / 2;
    R.ngroups = (window + SW_G - 1) / SW_G;
    const double c = 1.4426950408889634 / ((double)h * (double)h);
    R.neg_c = (float)(-c);
    R.pos_c = (float)c;
    R.c_self = (float)(1.0 / (1.0 + (double)mu));
    R.c_nb = (float)((double)mu / (2.0 * (double)mu + 2.0));
    R.big_d = (float)std::fmin(1e30, 1e37 / c);
    R.margin = 100.0f;
    R.z_limit = 1.2676506e30f;      // 2^100
    R.a_limit = 1.3292280e36f;      // 2^120
    R.clip = 0;
    {
        H->apply_smem = (size_t)prop.sharedMemPerBlockOptin;     // per kernel symbol: always the device maximum
        for (const void *fn : {(const void *)gj_apply3_kernel<4>, (const void *)gj_apply3_kernel<8>, (const void *)gj_apply3_kernel<16>})
            if (ce == cudaSuccess) ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)H->apply_smem);
        if (ce != cudaSuccess) { delete H; return cuda_fail(nullptr, ce, "apply kernel setup"); }
    }
    H->n_sm = prop.multiProcessorCount;
    H->smem_per_sm = prop.sharedMemPerMultiprocessor;
    ce = build_sweep_shapes(H, (size_t)prop.sharedMemPerBlockOptin);
    if (ce != cudaSuccess) { delete H; return cuda_fail(nullptr, ce, "sweep kernel setup"); }
    if (H->shapes.empty()) {
        delete H;
        return fail(nullptr, TNLM_UNSUPPORTED, "window/patch need more shared memory than one CTA has");
    }
    if (!sweep_shape_known(H, H->opt_rb, H->opt_nb)) {
        delete H;
        return fail(nullptr, TNLM_INVALID_ARG, "TNLM_SWEEP_SHAPE=\"rb,nb\" names a sweep shape that is not available for this window and patch");
    }
    if (geometry) {
        const tnlm_geometry &g = *geometry;
        Geom &G = H->G;
        G.nx = nx; G.ny = ny; G.n_phase = n_phase; G.n_views = g.n_views; G.n_bins = g.n_bins;
        G.pix = (float)g.pixel_mm;
        G.sdd_over_pitch = (float)(g.sdd_mm / g.bin_pitch_mm);
        G.bin_centre = (float)(0.5 * (g.n_bins - 1) - g.bin_offset);
        {   // largest |tan(fan angle)| of any point of the image, seen from any source position
            const double hx = 0.5 * nx * g.pixel_mm, hy = 0.5 * ny * g.pixel_mm;
            const double rmax = std::sqrt(hx * hx + hy * hy) + g.pixel_mm;
            H->fan_poly = rmax / std::sqrt(std::fmax(g.sid_mm * g.sid_mm - rmax * rmax, 1e-30)) < 0.95;
        }
        {   // backproject_kernel's candidate half-width (see there): pix x bins per radian x 1.02 x 1/(1 - s), s = the
            // half-diagonal of a 2 x 2 pixel block over the smallest distance of a block centre from the source
            // plane (>= sid - image half-diagonal >= 6 pixels, checked above), 1/(1 - s) <= 1 + s + 2 s^2 for s <= 1/2
            const double hxm = 0.5 * nx * g.pixel_mm, hym = 0.5 * ny * g.pixel_mm;
            const double sn = 1.4143 * g.pixel_mm / (g.sid_mm - std::sqrt(hxm * hxm + hym * hym));
            G.hw_scale = (float)(1.02 * (1.0 + sn + 2.0 * sn * sn) * g.pixel_mm * g.sdd_mm / g.bin_pitch_mm);
        }
        std::vector<RayEntry> tab; std::vector<RayRange> rng; std::vector<float4> views; std::vector<int4> split;
        if (!build_tables(g, nx, ny, n_phase, tab, rng, views, split)) {
            tnlm_destroy(H);
            return fail(nullptr, TNLM_UNSUPPORTED, "geometry: a view's rays change between steep and shallow more than twice (fan of 180 degrees or more)");
        }
        bool ok = cudaMalloc(&H->d_split, split.size() * sizeof(int4)) == cudaSuccess &&
                  cudaMemcpy(H->d_split, split.data(), split.size() * sizeof(int4), cudaMemcpyHostToDevice) == cudaSuccess &&
                  cudaMalloc(&H->d_tab, tab.size() * sizeof(RayEntry)) == cudaSuccess &&
                  cudaMalloc(&H->d_rng, rng.size() * sizeof(RayRange)) == cudaSuccess &&
                  cudaMalloc(&H->d_views, views.size() * sizeof(float4)) == cudaSuccess;
        if (ok) ok = cudaMemcpy(H->d_tab, tab.data(), tab.size() * sizeof(RayEntry), cudaMemcpyHostToDevice) == cudaSuccess &&
                     cudaMemcpy(H->d_rng, rng.data(), rng.size() * sizeof(RayRange), cudaMemcpyHostToDevice) == cudaSuccess &&
                     cudaMemcpy(H->d_views, views.data(), views.size() * sizeof(float4), cudaMemcpyHostToDevice) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            tnlm_destroy(H);
            return fail(nullptr, TNLM_ALLOC_FAILED, "device allocation failed (geometry tables)");
        }
        {   // FBP tables (double precision on the host)
            const int B = g.n_bins, M = n_phase * g.n_views;
            const double dgam = g.bin_pitch_mm / g.sdd_mm, two_pi = 6.283185307179586476925;
            std::vector<double> gk(B);
            std::vector<float> cosw(B), wv(M);
            for (int k = 0; k < B; ++k) {
                const double sk = std::sin(k * dgam);
                gk[k] = (k == 0) ? dgam / (8.0 * dgam * dgam) : ((k & 1) ? -dgam / (2.0 * 9.869604401089358 * sk * sk) : 0.0);
                cosw[k] = (float)(g.sid_mm * std::cos((k - 0.5 * (B - 1) + g.bin_offset) * dgam));
            }
            // trapezoid weights over the sorted cyclic union of all source angles
            std::vector<std::pair<double, int>> ord(M);
            for (int j = 0; j < M; ++j) {
                double bj = std::fmod(g.angles_rad[j], two_pi);
                if (bj < 0) bj += two_pi;
                ord[j] = std::make_pair(bj, j);
            }
            std::stable_sort(ord.begin(), ord.end(), [](const std::pair<double, int> &x, const std::pair<double, int> &y) { return x.first < y.first; });
            for (int t = 0; t < M; ++t) {
                const double nxt = (t + 1 < M) ? ord[t + 1].first : ord[0].first + two_pi;
                const double prv = (t > 0) ? ord[t - 1].first : ord[M - 1].first - two_pi;
                wv[ord[t].second] = (float)(0.5 * (nxt - prv));
            }
            bool ok2 = cudaMalloc(&H->d_fbp_g, B * sizeof(double)) == cudaSuccess &&
                       cudaMalloc(&H->d_fbp_cosw, B * sizeof(float)) == cudaSuccess &&
                       cudaMalloc(&H->d_fbp_wv, M * sizeof(float)) == cudaSuccess;
            if (ok2) ok2 = cudaMemcpy(H->d_fbp_g, gk.data(), B * sizeof(double), cudaMemcpyHostToDevice) == cudaSuccess &&
                           cudaMemcpy(H->d_fbp_cosw, cosw.data(), B * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess &&
                           cudaMemcpy(H->d_fbp_wv, wv.data(), M * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess;
            if (!ok2) {
                cudaGetLastError();
                tnlm_destroy(H);
                return fail(nullptr, TNLM_ALLOC_FAILED, "device allocation failed (FBP tables)");
            }
        }
        H->has_geom = true;
    }
    *out = H;
    return TNLM_OK;
}

static void free_ws(tnlm_handle *H)
{
    float **bufs[] = {&H->d_s, &H->d_t, &H->d_g, &H->d_f, &H->d_ua, &H->d_ub, &H->d_imT, &H->d_imI, &H->d_fbp_q, &H->d_r, &H->d_rw, &H->d_q, &H->d_sw, &H->d_yh, &H->d_wh};
    for (float **b : bufs) { if (*b) cudaFree(*b); *b = nullptr; }
    H->ws_slices = 0;
}

extern "C" int tnlm_destroy(tnlm_handle *H)
{
    if (!H) return TNLM_INVALID_ARG;
    DeviceGuard dg(H->device);
    for (cudaEvent_t e : H->prof_ev) cudaEventDestroy(e);
    free_ws(H);
    if (H->d_scal) cudaFree(H->d_scal);
    // the evict_last lines of the stored weights (apply_resident_mb) keep their L2 priority until other evict_last
    // traffic claims it: no cudaCtxResetPersistingL2Cache() here, which would also drop the persisting lines of
    // every other handle and library in the context
    if (H->d_wts) cudaFree(H->d_wts);
    if (H->d_fbp_g) cudaFree(H->d_fbp_g);
    if (H->d_fbp_cosw) cudaFree(H->d_fbp_cosw);
    if (H->d_fbp_wv) cudaFree(H->d_fbp_wv);
    if (H->d_tab) cudaFree(H->d_tab);
    if (H->d_rng) cudaFree(H->d_rng);
    if (H->d_views) cudaFree(H->d_views);
    if (H->d_split) cudaFree(H->d_split);
    delete H;
    return TNLM_OK;
}

// Workspace for n_slices (grown, never shrunk).  Buffers are allocated on first need of their kind
// (cudaMalloc synchronises the device: see "Execution" in tnlm.h; tnlm_reserve front-loads it).
static int ensure_ws(tnlm_handle *H, int n_slices)
{
    if (n_slices <= H->ws_slices) return TNLM_OK;
    free_ws(H);
    H->ws_slices = n_slices;
    return TNLM_OK;
}
static int need(tnlm_handle *H, float **buf, size_t count)
{
    if (*buf) return TNLM_OK;
    cudaError_t e = cudaMalloc(buf, count * sizeof(float));
    if (e != cudaSuccess) { cudaGetLastError(); *buf = nullptr; return fail(H, TNLM_ALLOC_FAILED, "device allocation failed (workspace)"); }
    return TNLM_OK;
}
static size_t img_count(const tnlm_handle *H) { return (size_t)H->ws_slices * H->n_phase * H->nx * H->ny; }
static size_t sino_count(const tnlm_handle *H) { return (size_t)H->ws_slices * H->n_phase * H->G.n_views * H->G.n_bins; }

static int check_common(tnlm_handle *H, int n_slices, bool needs_geom)
{
    if (!H) return TNLM_INVALID_ARG;
    H->err.clear();
    if (n_slices < 1) return fail(H, TNLM_INVALID_ARG, "n_slices must be >= 1");
    if ((long long)n_slices * H->n_phase > 65535) return fail(H, TNLM_UNSUPPORTED, "n_slices * n_phase above 65535");
    if (needs_geom && !H->has_geom) return fail(H, TNLM_INVALID_ARG, "handle was created without geometry");
    return TNLM_OK;
}
#define ENTER(H, name, n_slices, needs_geom)                                   \
    NvtxRange nvtx_range__(name);                                              \
    {                                                                          \
        int rc__ = check_common(H, n_slices, needs_geom);                      \
        if (rc__) return rc__;                                                 \
    }                                                                          \
    DeviceGuard device_guard__((H)->device);                                   \
    if (device_guard__.err != cudaSuccess) return cuda_fail(H, device_guard__.err, "cudaSetDevice")

// ------------------------------------------------------------------------------ per-launch timing
// Event pair around one kernel launch, on the launching stream (tnlm_profile_kernels).
static int prof_mark(tnlm_handle *H, int kind, bool begin, cudaStream_t st)
{
    if (begin) {
        const size_t need = 2 * H->prof_kind.size() + 2;
        while (H->prof_ev.size() < need) {
            cudaEvent_t e;
            CU(H, cudaEventCreate(&e));
            H->prof_ev.push_back(e);
        }
        CU(H, cudaEventRecord(H->prof_ev[2 * H->prof_kind.size()], st));
        H->prof_kind.push_back(kind);
    } else {
        CU(H, cudaEventRecord(H->prof_ev[2 * H->prof_kind.size() - 1], st));
    }
    return TNLM_OK;
}
// Timing is best effort: a pair whose begin mark failed (event creation or recording) is not recorded at all, and
// after PROF_MAX_PAIRS undrained pairs (tnlm_kernel_times drains and recycles the events) recording pauses.
static constexpr size_t PROF_MAX_PAIRS = 1u << 20;
struct ProfScope {
    tnlm_handle *H;
    cudaStream_t st;
    bool on;
    ProfScope(tnlm_handle *h, int kind, cudaStream_t s) : H(h), st(s), on(h->prof && h->prof_kind.size() < PROF_MAX_PAIRS)
    {
        if (on) on = (prof_mark(H, kind, true, st) == TNLM_OK);
    }
    ~ProfScope() { if (on) prof_mark(H, 0, false, st); }
};

// ------------------------------------------------------------------------------ projector
// Which forward projector serves a call with n_slices slices, and how many of its slices (a multiple of 4, from
// slice 0) go through the interleaved copies (interleave4_kernel, project_il_kernel, cgls_update_us_il).
// The strip kernel issues ~1.4x the instructions of the gather kernel (staging, per-chunk extents) and has no
// memory stalls: measured 12.7 vs 29.0 us on cfg 1 (less than one wave of work: latency bound) and 289 vs 233 us
// on cfg 4 (issue bound).  Automatic choice: strips while the gather kernel would have fewer than 2048 ray-threads
// per SM (one full wave of resident threads).  The crossover is a count of threads, whatever project_block cuts
// them into: it was measured between cfg 1 (57.6 k rays) and cfg 4 (533 k) and does not move with the CTA size.
static bool use_strips(const tnlm_handle *H, int n_slices)
{
    const int nray = H->G.n_views * H->G.n_bins;
    const long long gather_units = (long long)((nray + 255) / 256) * n_slices * H->n_phase;     // of 256 ray-threads
    return H->opt_project == 1 || (H->opt_project < 0 && gather_units < (long long)H->n_sm * 8);
}
static int il_slices(const tnlm_handle *H, int n_slices)
{
    return (H->opt_project_il && !use_strips(H, n_slices)) ? (n_slices / 4) * 4 : 0;
}
// The copies of img the forward projector reads: for slices [0, n_il) the two interleaved ones (d_imI, d_imT),
// for the others the transposed image (their part of d_imT).
static int launch_copies(tnlm_handle *H, const float *img, int n_slices, cudaStream_t st)
{
    int rc;
    const int n_il = il_slices(H, n_slices);
    if ((rc = need(H, &H->d_imT, img_count(H)))) return rc;
    if (n_il && (rc = need(H, &H->d_imI, img_count(H)))) return rc;
    ProfScope ps(H, TNLM_KERNEL_TRANSPOSE, st);
    if (n_il) {
        dim3 tg((H->nx + 31) / 32, (H->ny + 31) / 32, (n_il / 4) * H->n_phase);
        interleave4_kernel<<<tg, dim3(32, 8), 0, st>>>(img, reinterpret_cast<float4 *>(H->d_imI), reinterpret_cast<float4 *>(H->d_imT),
                                                        H->nx, H->ny, H->n_phase);
        LAUNCHED(H);
    }
    if (n_slices > n_il) {
        dim3 tg((H->nx + 31) / 32, (H->ny + 31) / 32, (n_slices - n_il) * H->n_phase);
        transpose_kernel<<<tg, dim3(32, 8), 0, st>>>(img, H->d_imT, H->nx, H->ny, n_il * H->n_phase);
        LAUNCHED(H);
    }
    return TNLM_OK;
}
// copies_ready: the copies of img (launch_copies) are already in d_imI / d_imT (cgls_update_us wrote them).
template <int MODE>
static int launch_project(tnlm_handle *H, const float *img, bool copies_ready, const float *y, const float *sw,
                          float *out0, float *out1, double *red, int n_slices, cudaStream_t st)
{
    const int nray = H->G.n_views * H->G.n_bins;
    int rc;
    if (!copies_ready && (rc = launch_copies(H, img, n_slices, st))) return rc;
    const float *imgT = H->d_imT;
    ProfScope ps(H, TNLM_KERNEL_PROJECT, st);
    if (use_strips(H, n_slices)) {
        const int tasks = H->G.n_views * ((H->G.n_bins + 31) / 32);
        dim3 grid((tasks + PS_WARPS - 1) / PS_WARPS, n_slices * H->n_phase);
        project_strip_kernel<MODE><<<grid, 32 * PS_WARPS, 0, st>>>(H->G, H->d_tab, H->d_rng, img, imgT, y, sw, out0, out1, red);
        LAUNCHED(H);
        return TNLM_OK;
    }
    const int n_il = il_slices(H, n_slices);
    if (n_il) {                                      // groups of four slices from the interleaved copies
        const int bt = H->opt_project_block;
        dim3 grid((nray + bt - 1) / bt, (n_il / 4) * H->n_phase);
        project_il_kernel<MODE><<<grid, bt, 0, st>>>(H->G, H->d_tab, H->d_rng, reinterpret_cast<const float4 *>(H->d_imI),
                                                       reinterpret_cast<const float4 *>(H->d_imT), y, sw, out0, out1, red);
        LAUNCHED(H);
    }
    // the other slices (fewer than four, or the remainder of a batch) one per thread from the image and its transpose
    if (n_slices > n_il) {
        const int bt = H->opt_project_block;             // threads per CTA (256, 128 or 64)
        dim3 grid((nray + bt - 1) / bt, (n_slices - n_il) * H->n_phase);
        project_kernel<MODE, 1><<<grid, bt, 0, st>>>(H->G, H->d_tab, H->d_rng, img, imgT, y, sw, out0, out1, red, n_il);
        LAUNCHED(H);
    }
    return TNLM_OK;
}
template <bool POLY, int BR, int BC>
static int launch_backproject_groups(tnlm_handle *H, const float *sino, float *img, double *red, int n_slices, cudaStream_t st)
{
    const int max_ns = H->opt_backproject_group;
    int s0 = 0;
    for (int ns = 16; ns >= 1; ns >>= 1) {
        if (ns > max_ns) continue;
        const int groups = (n_slices - s0) / ns;
        if (groups < 1) continue;
        dim3 grid((H->nx + 8 * BC - 1) / (8 * BC), (H->ny + 16 * BR - 1) / (16 * BR), groups * H->n_phase);
        if (ns == 16) backproject_kernel<POLY, 16, BR, BC><<<grid, 128, 0, st>>>(H->G, H->d_tab, H->d_views, H->d_split, sino, img, red, s0);
        else if (ns == 8) backproject_kernel<POLY, 8, BR, BC><<<grid, 128, 0, st>>>(H->G, H->d_tab, H->d_views, H->d_split, sino, img, red, s0);
        else if (ns == 4) backproject_kernel<POLY, 4, BR, BC><<<grid, 128, 0, st>>>(H->G, H->d_tab, H->d_views, H->d_split, sino, img, red, s0);
        else if (ns == 2) backproject_kernel<POLY, 2, BR, BC><<<grid, 128, 0, st>>>(H->G, H->d_tab, H->d_views, H->d_split, sino, img, red, s0);
        else backproject_kernel<POLY, 1, BR, BC><<<grid, 128, 0, st>>>(H->G, H->d_tab, H->d_views, H->d_split, sino, img, red, s0);
        LAUNCHED(H);
        s0 += groups * ns;
    }
    return TNLM_OK;
}
static int launch_backproject(tnlm_handle *H, const float *sino, float *img, double *red, int n_slices, cudaStream_t st)
{
    // 2 x 2 pixels per thread: 2 x 4 blocks measured the same (372 vs 372 us on cfg 4, 2.13 vs 2.15 ms on cfg 3),
    // 4 x 4 blocks 15 % slower (longer candidate lists, more idle lanes per warp)
    ProfScope ps(H, TNLM_KERNEL_BACKPROJECT, st);
    return H->fan_poly ? launch_backproject_groups<true, 2, 2>(H, sino, img, red, n_slices, st)
                       : launch_backproject_groups<false, 2, 2>(H, sino, img, red, n_slices, st);
}

extern "C" int tnlm_project(tnlm_handle *H, const float *img, float *sino, int n_slices, void *stream)
{
    ENTER(H, "tnlm_project", n_slices, true);
    int rc;
    if (!img || !sino) return fail(H, TNLM_INVALID_ARG, "img and sino must not be NULL");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    return launch_project<FWD_PLAIN>(H, img, false, nullptr, nullptr, sino, nullptr, nullptr, n_slices, (cudaStream_t)stream);
}

extern "C" int tnlm_backproject(tnlm_handle *H, const float *sino, float *img, int n_slices, void *stream)
{
    ENTER(H, "tnlm_backproject", n_slices, true);
    if (!img || !sino) return fail(H, TNLM_INVALID_ARG, "img and sino must not be NULL");
    return launch_backproject(H, sino, img, nullptr, n_slices, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------ FBP initialisation
extern "C" int tnlm_fbp_init(tnlm_handle *H, const float *y, float *f0, int n_slices, void *stream)
{
    ENTER(H, "tnlm_fbp_init", n_slices, true);
    int rc;
    if (!y || !f0) return fail(H, TNLM_INVALID_ARG, "y and f0 must not be NULL");
    if ((size_t)H->G.n_bins * sizeof(float) > 48 * 1024) return fail(H, TNLM_UNSUPPORTED, "more than 12288 detector bins");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    if ((rc = need(H, &H->d_fbp_q, sino_count(H)))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int M = H->n_phase * H->G.n_views;
    {
        ProfScope ps(H, TNLM_KERNEL_FBP, st);
        fbp_filter_kernel<<<dim3(M, n_slices), 256, H->G.n_bins * sizeof(float), st>>>(y, H->d_fbp_q, H->d_fbp_cosw, H->d_fbp_g,
                                                                                          H->G.n_bins);
        LAUNCHED(H);
    }
    ProfScope ps(H, TNLM_KERNEL_FBP, st);
    fbp_backproject_kernel<<<dim3((H->nx + 31) / 32, (H->ny + 7) / 8, n_slices), dim3(32, 8), 0, st>>>(
        H->G, H->d_views, H->d_fbp_wv, H->d_fbp_q, f0);
    LAUNCHED(H);
    return TNLM_OK;
}

// ------------------------------------------------------------------------------ CGLS
static int ensure_scalars(tnlm_handle *H, int nscal)
{
    if (nscal <= H->scal_cap) return TNLM_OK;
    if (H->d_scal) cudaFree(H->d_scal);
    H->d_scal = nullptr; H->scal_cap = 0;
    if (cudaMalloc(&H->d_scal, (size_t)nscal * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return fail(H, TNLM_ALLOC_FAILED, "device allocation failed (scalars)"); }
    H->scal_cap = nscal;
    return TNLM_OK;
}
static int cgls_workspace(tnlm_handle *H, int m1, int n_slices, bool weighted)
{
    int rc;
    if (m1 == 0) return TNLM_OK;
    if ((rc = need(H, &H->d_s, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_t, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_imT, img_count(H)))) return rc;
    if (il_slices(H, n_slices) && (rc = need(H, &H->d_imI, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_r, sino_count(H)))) return rc;
    if ((rc = need(H, &H->d_rw, sino_count(H)))) return rc;
    if ((rc = need(H, &H->d_q, sino_count(H)))) return rc;
    if (weighted && (rc = need(H, &H->d_sw, sino_count(H)))) return rc;
    return ensure_scalars(H, (2 * m1 + 1) * n_slices * H->n_phase);
}
// sw = sqrt(w) into the handle's buffer (once per call; w is fixed across the outer iterations).
static int prepare_sqrt_weights(tnlm_handle *H, const float *w, int n_slices, cudaStream_t st)
{
    if (!w) return TNLM_OK;
    int rc;
    if ((rc = need(H, &H->d_sw, sino_count(H)))) return rc;
    const size_t n = (size_t)n_slices * H->n_phase * H->G.n_views * H->G.n_bins;
    ProfScope ps(H, TNLM_KERNEL_CGLS_VECTOR, st);
    sqrt_weights_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(w, H->d_sw, n);
    LAUNCHED(H);
    return TNLM_OK;
}

// sw = sqrt(w) (NULL = identity), already prepared by the caller.
static int cgls_device(tnlm_handle *H, const float *f_in, const float *y, const float *sw, int m1, float *g_out,
                       int n_slices, cudaStream_t st)
{
    const int nprob = n_slices * H->n_phase;
    const int npix = H->nx * H->ny, nray = H->G.n_views * H->G.n_bins;
    const size_t nimg = (size_t)nprob * npix;
    if (g_out != f_in) CU(H, cudaMemcpyAsync(g_out, f_in, nimg * sizeof(float), cudaMemcpyDeviceToDevice, st));
    if (m1 == 0) return TNLM_OK;
    int rc;
    if ((rc = cgls_workspace(H, m1, n_slices, sw != nullptr))) return rc;
    const int nscal = (2 * m1 + 1) * nprob;
    double *gam = H->d_scal, *qq = H->d_scal + (size_t)(m1 + 1) * nprob;
    CU(H, cudaMemsetAsync(H->d_scal, 0, (size_t)nscal * sizeof(double), st));
    float *u = g_out;
    dim3 gs((nray + 255) / 256, nprob);
    // init (L109): r = y_n - P_n u ; s = P_n^T r ; gamma_0 = ||s||^2
    if ((rc = launch_project<FWD_RESID>(H, u, false, y, sw, H->d_r, H->d_rw, nullptr, n_slices, st))) return rc;
    if ((rc = launch_backproject(H, H->d_rw, H->d_s, gam, n_slices, st))) return rc;
    // Slices [0, n_il) keep s in the interleaved copies the batch projector reads (made from d_s by the first
    // FWD_SCALE, updated in place by cgls_update_us_il); the others keep it in d_s with its transpose in d_imT.
    const int n_il = il_slices(H, n_slices), prob_il = n_il * H->n_phase;
    dim3 gt_il((H->nx + 31) / 32, (H->ny + 31) / 32, std::max(prob_il / 4, 1)), gt_rest((H->nx + 31) / 32, (H->ny + 31) / 32, std::max(nprob - prob_il, 1));
    float4 *sI = reinterpret_cast<float4 *>(H->d_imI), *sTI = reinterpret_cast<float4 *>(H->d_imT);
    bool copies_ready = false;                       // made by cgls_update_us from step 1 on
    for (int m = 0; m < m1; ++m) {
        // q = P_n s ; qq_m = ||q||^2
        if ((rc = launch_project<FWD_SCALE>(H, H->d_s, copies_ready, nullptr, sw, H->d_q, nullptr, qq + (size_t)m * nprob, n_slices, st))) return rc;
        if (m + 1 == m1) {                           // r, t, s of the last step feed nothing (g = u^(M1), L127)
            ProfScope ps(H, TNLM_KERNEL_CGLS_VECTOR, st);
            if (prob_il) {
                cgls_update_us_il<true><<<gt_il, dim3(32, 8), 0, st>>>(u, sI, nullptr, nullptr, H->nx, H->ny, H->n_phase, gam, qq, nprob, m);
                LAUNCHED(H);
            }
            if (nprob > prob_il) {
                cgls_update_us<true><<<gt_rest, dim3(32, 8), 0, st>>>(u, H->d_s, nullptr, nullptr, H->nx, H->ny, gam, qq, nprob, m, prob_il);
                LAUNCHED(H);
            }
            break;
        }
        {
            ProfScope ps(H, TNLM_KERNEL_CGLS_VECTOR, st);
            cgls_update_r<<<gs, 256, 0, st>>>(H->d_r, H->d_rw, H->d_q, sw, nray, gam, qq, nprob, m);
            LAUNCHED(H);
        }
        if ((rc = launch_backproject(H, H->d_rw, H->d_t, gam + (size_t)(m + 1) * nprob, n_slices, st))) return rc;
        {
            ProfScope ps(H, TNLM_KERNEL_CGLS_VECTOR, st);
            if (prob_il) {
                cgls_update_us_il<false><<<gt_il, dim3(32, 8), 0, st>>>(u, sI, H->d_t, sTI, H->nx, H->ny, H->n_phase, gam, qq, nprob, m);
                LAUNCHED(H);
            }
            if (nprob > prob_il) {
                cgls_update_us<false><<<gt_rest, dim3(32, 8), 0, st>>>(u, H->d_s, H->d_t, H->d_imT, H->nx, H->ny, gam, qq, nprob, m, prob_il);
                LAUNCHED(H);
            }
        }
        copies_ready = true;
    }
    return TNLM_OK;
}

extern "C" int tnlm_cgls_step(tnlm_handle *H, const float *f_in, const float *y, const float *w, int m1,
                              float *g_out, int n_slices, void *stream)
{
    ENTER(H, "tnlm_cgls_step", n_slices, true);
    int rc;
    if (!f_in || !y || !g_out) return fail(H, TNLM_INVALID_ARG, "f_in, y and g_out must not be NULL");
    if (m1 < 0) return fail(H, TNLM_INVALID_ARG, "m1 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (m1 > 0 && (rc = prepare_sqrt_weights(H, w, n_slices, st))) return rc;
    return cgls_device(H, f_in, y, w ? H->d_sw : nullptr, m1, g_out, n_slices, st);
}

// ------------------------------------------------------------------------------ TNLM
// The cheapest launchable shape for n_img images (cost model above).
static const SweepShape *pick_shape(tnlm_handle *H, int n_img)
{
    const SweepShape *best = nullptr;
    double best_cost = 0.0;
    for (const SweepShape &sh : H->shapes) {
        if ((H->opt_rb && sh.rb != H->opt_rb) || (H->opt_nb && sh.nb != H->opt_nb)) continue;   // tuning override
        const double c = sweep_cost(H, sh, n_img);
        if (!best || c < best_cost) { best = &sh; best_cost = c; }
    }
    if (!best) fail(H, TNLM_INVALID_ARG, "option sweep_rb/sweep_nb (TNLM_SWEEP_SHAPE) names a shape that is not available");
    return best;
}

static void fill_layout(const tnlm_handle *H, const SweepShape &sh, SweepParams &R)
{
    const int th = sh.nb * sh.rb;
    R.nb = sh.nb;
    R.rb = sh.rb;
    R.tiles_x = (H->nx + SW_TW - 1) / SW_TW;
    R.tiles_y = (H->ny + th - 1) / th;
    R.nbands = R.tiles_y * sh.nb;
}

// Stored-weight tasks (row pairs of 2 x 128 pixels, both sides: 2 W^2 pieces of 512 bytes) the option
// apply_resident_mb keeps in L2.
static long long resident_tasks(const tnlm_handle *H)
{
    const double task_bytes = 2.0 * H->window * H->window * 512.0;
    return (long long)((double)H->opt_resident_mb * 1048576.0 / task_bytes);
}

// One sweep with the weights computed on the fly; wts != NULL also stores them (bf16 chunks).
static int launch_sweep(tnlm_handle *H, const SweepShape &sh, const float *g, const float *u, float *out, int clip,
                        int n_slices, __nv_bfloat16 *wts, cudaStream_t st)
{
    const int nimg = n_slices * H->n_phase;
    SweepParams R = H->R;
    R.clip = clip;
    fill_layout(H, sh, R);
    R.res_tasks = resident_tasks(H);
    const long long ctas = (long long)nimg * R.tiles_x * R.tiles_y;
    if (ctas > 2147483647LL) return fail(H, TNLM_UNSUPPORTED, "too many tiles for one launch");
    void *args[] = {(void *)&R, (void *)&g, (void *)&u, (void *)&out, (void *)&wts};
    ProfScope ps(H, wts ? TNLM_KERNEL_SWEEP_STORE : TNLM_KERNEL_SWEEP, st);
    cudaError_t e = cudaLaunchKernel(wts ? sh.fn_store : sh.fn, dim3((unsigned)ctas), dim3(64 * sh.nb), args, sh.smem, st);
    if (e != cudaSuccess) return cuda_fail(H, e, "cudaLaunchKernel(gj_sweep_kernel)");
    LAUNCHED(H);
    return TNLM_OK;
}

// One sweep with the stored weights of this outer iteration (written by shape sh).
static int launch_apply(tnlm_handle *H, const SweepShape &sh, const float *g, const float *u, float *out, int clip,
                        int n_slices, const __nv_bfloat16 *wts, int sweep_index, cudaStream_t st)
{
    SweepParams R = H->R;
    R.clip = clip;
    R.res_tasks = resident_tasks(H);
    // the storing sweep (index 0) wrote the chunks front to back: sweep 1 starts from the back, where the
    // freshest lines are, sweep 2 from the front, ...
    R.ap_reverse = (H->opt_snake && (sweep_index & 1)) ? 1 : 0;
    fill_layout(H, sh, R);
    R.tiles_y = (H->ny + sh.rb - 1) / sh.rb;             // CTA = one band that holds image rows
    const long long ctas = (long long)n_slices * H->n_phase * R.tiles_x * R.tiles_y;
    if (ctas > 2147483647LL) return fail(H, TNLM_UNSUPPORTED, "too many tiles for one launch");
    // one CTA per stored band, the windows of both sides shared by its warps (gj_apply3_kernel)
    R.n_img = n_slices * H->n_phase;
    int dp = H->opt_depth ? H->opt_depth : 8;
    while (dp > 4 && apply3_smem_bytes(H->window, sh.rb, dp) > H->apply_smem) dp >>= 1;
    const size_t sm = apply3_smem_bytes(H->window, sh.rb, dp);
    if (sm > H->apply_smem) return fail(H, TNLM_UNSUPPORTED, "window needs more shared memory than one CTA has");
    const unsigned threads = 32u * (unsigned)(sh.rb / 2);
    ProfScope ps(H, TNLM_KERNEL_APPLY, st);
    switch (dp) {
        case 16: gj_apply3_kernel<16><<<(unsigned)ctas, threads, sm, st>>>(R, g, u, out, wts); break;
        case 8: gj_apply3_kernel<8><<<(unsigned)ctas, threads, sm, st>>>(R, g, u, out, wts); break;
        default: gj_apply3_kernel<4><<<(unsigned)ctas, threads, sm, st>>>(R, g, u, out, wts); break;
    }
    LAUNCHED(H);
    return TNLM_OK;
}

// Weight storage for m2 > 1 (opt-in: option weight_cache_mb / TNLM_WEIGHT_CACHE_MB > 0): 2 bytes x 2 sides x W^2 per
// pixel of the padded band/tile grid.  *wts = NULL (every sweep computes its weights in fp32) when the option is 0,
// the default, or when the need exceeds it.  An allocation that fails is an error of the call (TNLM_ALLOC_FAILED),
// not a silent change of path.
static int weight_cache(tnlm_handle *H, const SweepShape &sh, int n_slices, __nv_bfloat16 **wts)
{
    *wts = nullptr;
    SweepParams R = H->R;
    fill_layout(H, sh, R);
    const size_t need = (size_t)n_slices * H->n_phase * 2 * R.nbands * R.tiles_x * H->window * H->window * sh.rb * SW_TW;
    if (H->opt_cache_mb <= 0 || need * sizeof(__nv_bfloat16) > (size_t)H->opt_cache_mb * 1048576ull) return TNLM_OK;
    if (need > H->wts_cap) {
        if (H->d_wts) cudaFree(H->d_wts);
        H->d_wts = nullptr; H->wts_cap = 0;
        if (cudaMalloc(&H->d_wts, need * sizeof(__nv_bfloat16)) != cudaSuccess) {
            cudaGetLastError();
            return fail(H, TNLM_ALLOC_FAILED, "device allocation failed (stored weights: " + std::to_string(need * sizeof(__nv_bfloat16) >> 20) +
                        " MB; lower weight_cache_mb below that, or set it to 0, to compute the weights in every sweep)");
        }
        H->wts_cap = need;
    }
    *wts = H->d_wts;
    return TNLM_OK;
}

extern "C" int tnlm_fma_peak(double *tflops, void *stream)
{
    if (!tflops) return TNLM_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0;
    float *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (ce == cudaSuccess) ce = cudaMalloc(&d, sizeof(float));
    if (ce == cudaSuccess) ce = cudaEventCreate(&e0);
    if (ce == cudaSuccess) ce = cudaEventCreate(&e1);
    const int blocks = n_sm * 8, iters = 2048;
    double best = 0.0;
    for (int rep = 0; rep < 4 && ce == cudaSuccess; ++rep) {        // first launch warms up
        cudaEventRecord(e0, st);
        fp32_probe_kernel<<<blocks, 256, 0, st>>>(d, 1.0001f, 0.5f, iters);
        cudaEventRecord(e1, st);
        ce = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
        const double tf = 2.0 * 8 * 16 * (double)iters * 256.0 * blocks / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (d) cudaFree(d);
    if (ce != cudaSuccess) { cuda_fail(nullptr, ce, "tnlm_fma_peak"); return TNLM_CUDA_ERROR; }
    *tflops = best;
    return TNLM_OK;
}

extern "C" int tnlm_profile_kernels(tnlm_handle *H, int enable)
{
    if (!H) return TNLM_INVALID_ARG;
    H->err.clear();
    H->prof = enable != 0;
    H->prof_kind.clear();
    return TNLM_OK;
}

extern "C" int tnlm_kernel_times(tnlm_handle *H, float *ms, int *kind, int capacity, int *count)
{
    if (!H) return TNLM_INVALID_ARG;
    H->err.clear();
    if (!count || capacity < 0 || (capacity > 0 && (!ms || !kind))) return fail(H, TNLM_INVALID_ARG, "count, and ms/kind when capacity > 0, must not be NULL");
    DeviceGuard dg(H->device);
    const int n = (int)H->prof_kind.size();
    *count = n;
    for (int i = 0; i < n && i < capacity; ++i) {
        CU(H, cudaEventSynchronize(H->prof_ev[2 * i + 1]));
        CU(H, cudaEventElapsedTime(&ms[i], H->prof_ev[2 * i], H->prof_ev[2 * i + 1]));
        kind[i] = H->prof_kind[i];
    }
    H->prof_kind.clear();
    return TNLM_OK;
}

extern "C" int tnlm_set_option(tnlm_handle *H, const char *name, long long value)
{
    if (!H) return TNLM_INVALID_ARG;
    H->err.clear();
    if (!name) return fail(H, TNLM_INVALID_ARG, "option name is NULL");
    const std::string n(name);
    auto in = [&](long long lo, long long hi) { return value >= lo && value <= hi; };
    bool ok = true;
    if (n == "weight_cache_mb") H->opt_cache_mb = value;
    else if (n == "sweep_rb") { if ((ok = in(0, 64) && sweep_shape_known(H, (int)value, H->opt_nb))) H->opt_rb = (int)value; }
    else if (n == "sweep_nb") { if ((ok = in(0, 64) && sweep_shape_known(H, H->opt_rb, (int)value))) H->opt_nb = (int)value; }
    else if (n == "project_kernel") { if ((ok = in(-1, 1))) H->opt_project = (int)value; }
    else if (n == "apply_depth") { if ((ok = (value == 0 || value == 4 || value == 8 || value == 16))) H->opt_depth = (int)value; }
    else if (n == "project_interleave") { if ((ok = in(0, 1))) H->opt_project_il = (int)value; }
    else if (n == "project_block") { if ((ok = (value == 256 || value == 128 || value == 64))) H->opt_project_block = (int)value; }
    else if (n == "backproject_group") { if ((ok = (value == 1 || value == 2 || value == 4 || value == 8 || value == 16))) H->opt_backproject_group = (int)value; }
    else if (n == "apply_snake") { if ((ok = in(0, 1))) H->opt_snake = (int)value; }
    else if (n == "apply_resident_mb") { if ((ok = in(0, 1 << 20))) H->opt_resident_mb = value; }
    else return fail(H, TNLM_INVALID_ARG, "unknown option: " + n);
    if (!ok) return fail(H, TNLM_INVALID_ARG, "value out of range (or, for sweep_rb/sweep_nb, not an available shape) for option " + n);
    return TNLM_OK;
}

extern "C" int tnlm_device(const tnlm_handle *H) { return H ? H->device : -1; }

static int regularize_workspace(tnlm_handle *H, int m2, bool alias)
{
    int rc;
    if (m2 > 1 || alias) if ((rc = need(H, &H->d_ua, img_count(H)))) return rc;
    if (m2 > 2 || (alias && m2 > 1)) if ((rc = need(H, &H->d_ub, img_count(H)))) return rc;
    return TNLM_OK;
}

// g -> f_out; g and f_out are distinct device buffers or the same buffer.
static int regularize_device(tnlm_handle *H, const float *g, int m2, float *f_out, int n_slices, cudaStream_t st)
{
    const size_t n = (size_t)n_slices * H->n_phase * H->nx * H->ny;
    int rc;
    if (m2 == 0) {
        ProfScope ps(H, TNLM_KERNEL_CLIP, st);
        clip_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, f_out, n);
        LAUNCHED(H);
        return TNLM_OK;
    }
    const bool alias = (f_out == g);
    if ((rc = regularize_workspace(H, m2, alias))) return rc;
    const float *src = g;
    float *pp[2] = {H->d_ua, H->d_ub};
    int which = 0;
    const SweepShape *sh = pick_shape(H, n_slices * H->n_phase);
    if (!sh) return TNLM_INVALID_ARG;
    __nv_bfloat16 *wts = nullptr;                    // weights are those of g for all sweeps (L162); stored only on request
    if (m2 > 1 && (rc = weight_cache(H, *sh, n_slices, &wts))) return rc;
    for (int m = 0; m < m2; ++m) {
        const bool last = (m + 1 == m2);
        float *dst;
        if (last && !alias) dst = f_out;
        else { dst = pp[which]; if (dst == src) { which ^= 1; dst = pp[which]; } }
        const bool computes = (m == 0 || !wts);
        if (computes) rc = launch_sweep(H, *sh, g, src, dst, last ? 1 : 0, n_slices, wts, st);
        else rc = launch_apply(H, *sh, g, src, dst, last ? 1 : 0, n_slices, wts, m, st);
        if (rc) return rc;
        src = dst;
        which ^= 1;
    }
    if (alias) CU(H, cudaMemcpyAsync(f_out, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return TNLM_OK;
}

extern "C" int tnlm_regularize_step(tnlm_handle *H, const float *g, int m2, float *f_out, int n_slices, void *stream)
{
    ENTER(H, "tnlm_regularize_step", n_slices, false);
    int rc;
    if (!g || !f_out) return fail(H, TNLM_INVALID_ARG, "g and f_out must not be NULL");
    if (m2 < 0) return fail(H, TNLM_INVALID_ARG, "m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    return regularize_device(H, g, m2, f_out, n_slices, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------ TNLM step without allocation
// tnlm_regularize_step_noalloc (tnlm.h): for callers that cannot cudaMalloc -- HBM fully handed out to someone
// else's allocator, or other streams that must not be stalled by cudaMalloc's device-wide synchronisation.
// The two ping-pong images of the sweeps live in this array instead of the handle's cudaMalloc'ed d_ua / d_ub.
// It is part of the device image of this translation unit: 20 MiB on every GPU that loads it, until exit.
// One array per device, shared by all handles and streams: overlapping calls race (documented in tnlm.h).
static __device__ __align__(256) float g_noalloc_scratch[2 * (size_t)TNLM_NOALLOC_MAX_PIXELS];

// Device address of g_noalloc_scratch on the CURRENT device.  In host code the name g_noalloc_scratch is only a
// stand-in the runtime keys its lookup on, not a pointer a kernel may be given; the address differs per device, so
// it is looked up once per device, with that device current, and remembered.
static cudaError_t noalloc_scratch_address(int device, float **out)
{
    static std::mutex lock;
    static float *known[64] = {};
    std::lock_guard<std::mutex> hold(lock);
    if (device >= 0 && device < 64 && known[device]) { *out = known[device]; return cudaSuccess; }
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (device >= 0 && device < 64) known[device] = static_cast<float *>(p);
    *out = static_cast<float *>(p);
    return cudaSuccess;
}

extern "C" int tnlm_regularize_step_noalloc(tnlm_handle *H, const float *g, int m2, float *f_out, int n_slices, void *stream)
{
    ENTER(H, "tnlm_regularize_step_noalloc", n_slices, false);      // makes H->device current
    int rc;
    if (!g || !f_out) return fail(H, TNLM_INVALID_ARG, "g and f_out must not be NULL");
    if (m2 < 0) return fail(H, TNLM_INVALID_ARG, "m2 must be >= 0");
    const size_t n = (size_t)n_slices * H->n_phase * H->nx * H->ny;
    if (n > (size_t)TNLM_NOALLOC_MAX_PIXELS)
        return fail(H, TNLM_UNSUPPORTED, "tnlm_regularize_step_noalloc: n_slices * n_phase * ny * nx = " + std::to_string(n) +
                    " pixels is above the built-in scratch of TNLM_NOALLOC_MAX_PIXELS = " + std::to_string(TNLM_NOALLOC_MAX_PIXELS) +
                    "; use tnlm_regularize_step (which allocates) or fewer slices per call");
    float *scratch = nullptr;
    CU(H, noalloc_scratch_address(H->device, &scratch));
    cudaStream_t st = (cudaStream_t)stream;
    // per-launch timing would create events (prof_mark): not in a call that promises to allocate nothing
    struct ProfOff {
        tnlm_handle *H; bool was;
        explicit ProfOff(tnlm_handle *h) : H(h), was(h->prof) { h->prof = false; }
        ~ProfOff() { H->prof = was; }
    } prof_off(H);
    if (m2 == 0) {
        clip_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, f_out, n);
        LAUNCHED(H);
        return TNLM_OK;
    }
    const bool alias = (f_out == g);
    const SweepShape *sh = pick_shape(H, n_slices * H->n_phase);
    if (!sh) return TNLM_INVALID_ARG;
    float *pp[2] = {scratch, scratch + TNLM_NOALLOC_MAX_PIXELS};
    const float *src = g;
    for (int m = 0; m < m2; ++m) {
        const bool last = (m + 1 == m2);
        float *dst = (last && !alias) ? f_out : pp[m & 1];   // every sweep writes all n pixels of dst: no clearing needed
        if ((rc = launch_sweep(H, *sh, g, src, dst, last ? 1 : 0, n_slices, nullptr, st))) return rc;   // weights of g, fp32, every sweep
        src = dst;
    }
    if (alias) CU(H, cudaMemcpyAsync(f_out, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return TNLM_OK;
}

// ------------------------------------------------------------------------------ outer loop
static int reconstruct_device(tnlm_handle *H, const float *y, const float *w, const float *f0, int k_outer, int m1,
                              int m2, float *f_out, int n_slices, cudaStream_t st)
{
    const size_t n = (size_t)n_slices * H->n_phase * H->nx * H->ny;
    int rc;
    if (f0) { if (f_out != f0) CU(H, cudaMemcpyAsync(f_out, f0, n * sizeof(float), cudaMemcpyDeviceToDevice, st)); }
    else CU(H, cudaMemsetAsync(f_out, 0, n * sizeof(float), st));
    if (k_outer == 0) return TNLM_OK;
    if ((rc = need(H, &H->d_g, img_count(H)))) return rc;
    if (m1 > 0 && (rc = prepare_sqrt_weights(H, w, n_slices, st))) return rc;
    const float *sw = w ? H->d_sw : nullptr;
    for (int k = 0; k < k_outer; ++k) {
        if ((rc = cgls_device(H, f_out, y, sw, m1, H->d_g, n_slices, st))) return rc;      // step 2 (L176)
        if ((rc = regularize_device(H, H->d_g, m2, f_out, n_slices, st))) return rc;       // steps 3-5
    }
    return TNLM_OK;
}

extern "C" int tnlm_reconstruct(tnlm_handle *H, const float *y, const float *w, const float *f0, int k_outer, int m1,
                                int m2, float *f_out, int n_slices, void *stream)
{
    ENTER(H, "tnlm_reconstruct", n_slices, true);
    int rc;
    if (!y || !f_out) return fail(H, TNLM_INVALID_ARG, "y and f_out must not be NULL");
    if (k_outer < 0 || m1 < 0 || m2 < 0) return fail(H, TNLM_INVALID_ARG, "k_outer, m1, m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    return reconstruct_device(H, y, w, f0, k_outer, m1, m2, f_out, n_slices, (cudaStream_t)stream);
}

// All allocation a later call with these parameters would do, done now (cudaMalloc synchronises the device;
// after tnlm_reserve the enqueue calls with n_slices, m1, m2 up to the reserved ones never allocate).
extern "C" int tnlm_reserve(tnlm_handle *H, int n_slices, int m1, int m2, int host_entry_points)
{
    ENTER(H, "tnlm_reserve", n_slices, false);
    int rc;
    if (m1 < 0 || m2 < 0) return fail(H, TNLM_INVALID_ARG, "m1, m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    if ((rc = regularize_workspace(H, m2, true))) return rc;
    if (m2 > 1) {
        const SweepShape *sh = pick_shape(H, n_slices * H->n_phase);
        if (!sh) return TNLM_INVALID_ARG;
        __nv_bfloat16 *wts = nullptr;                // NULL (option 0, or over the cap) just means "recompute"
        if ((rc = weight_cache(H, *sh, n_slices, &wts))) return rc;
    }
    if ((rc = need(H, &H->d_g, img_count(H)))) return rc;
    if (host_entry_points && (rc = need(H, &H->d_f, img_count(H)))) return rc;
    if (H->has_geom) {
        if ((rc = cgls_workspace(H, std::max(m1, 1), n_slices, true))) return rc;
        if (host_entry_points) {
            if ((rc = need(H, &H->d_yh, sino_count(H)))) return rc;
            if ((rc = need(H, &H->d_wh, sino_count(H)))) return rc;
        }
    }
    return TNLM_OK;
}

// ------------------------------------------------------------------------------ host-buffer entry points
extern "C" int tnlm_regularize_step_host(tnlm_handle *H, const float *g_host, int m2, float *f_out_host, int n_slices, void *stream)
{
    ENTER(H, "tnlm_regularize_step_host", n_slices, false);
    int rc;
    if (!g_host || !f_out_host) return fail(H, TNLM_INVALID_ARG, "g_host and f_out_host must not be NULL");
    if (m2 < 0) return fail(H, TNLM_INVALID_ARG, "m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    if ((rc = need(H, &H->d_g, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_f, img_count(H)))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)n_slices * H->n_phase * H->nx * H->ny * sizeof(float);
    CU(H, cudaMemcpyAsync(H->d_g, g_host, bytes, cudaMemcpyHostToDevice, st));
    if ((rc = regularize_device(H, H->d_g, m2, H->d_f, n_slices, st))) return rc;
    CU(H, cudaMemcpyAsync(f_out_host, H->d_f, bytes, cudaMemcpyDeviceToHost, st));
    CU(H, cudaStreamSynchronize(st));
    return TNLM_OK;
}

extern "C" int tnlm_reconstruct_host(tnlm_handle *H, const float *y_host, const float *w_host, const float *f0_host,
                                     int k_outer, int m1, int m2, float *f_out_host, int n_slices, void *stream)
{
    ENTER(H, "tnlm_reconstruct_host", n_slices, true);
    int rc;
    if (!y_host || !f_out_host) return fail(H, TNLM_INVALID_ARG, "y_host and f_out_host must not be NULL");
    if (k_outer < 0 || m1 < 0 || m2 < 0) return fail(H, TNLM_INVALID_ARG, "k_outer, m1, m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    if ((rc = need(H, &H->d_f, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_yh, sino_count(H)))) return rc;
    if (w_host && (rc = need(H, &H->d_wh, sino_count(H)))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t ib = (size_t)n_slices * H->n_phase * H->nx * H->ny * sizeof(float);
    const size_t sb = (size_t)n_slices * H->n_phase * H->G.n_views * H->G.n_bins * sizeof(float);
    CU(H, cudaMemcpyAsync(H->d_yh, y_host, sb, cudaMemcpyHostToDevice, st));
    if (w_host) CU(H, cudaMemcpyAsync(H->d_wh, w_host, sb, cudaMemcpyHostToDevice, st));
    if (f0_host) CU(H, cudaMemcpyAsync(H->d_f, f0_host, ib, cudaMemcpyHostToDevice, st));
    if ((rc = reconstruct_device(H, H->d_yh, w_host ? H->d_wh : nullptr, f0_host ? H->d_f : nullptr, k_outer, m1, m2,
                                 H->d_f, n_slices, st))) return rc;
    CU(H, cudaMemcpyAsync(f_out_host, H->d_f, ib, cudaMemcpyDeviceToHost, st));
    CU(H, cudaStreamSynchronize(st));
    return TNLM_OK;
}
