// tnlm_api.cu -- C ABI of libtnlm (see include/tnlm.h): handle, argument checks, workspace,
// and the launch sequences of the five operations.  Host code only orchestrates; every step
// of the path runs in the kernels of projector.cuh, cgls.cuh and regularize.cuh.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/tnlm.h"
#include "cgls.cuh"
#include "common.cuh"
#include "projector.cuh"
#include "regularize.cuh"

using namespace tnlm;

static constexpr int MAX_PATCH = 9, MAX_WINDOW = 31;
static constexpr int REG_TX = 16, REG_TY = 8;          // CTA = 128 threads, 64 x 32 pixel tile

struct tnlm_handle {
    int nx = 0, ny = 0, n_phase = 0, window = 0, patch = 0;
    float h = 0.f, mu = 0.f;
    bool has_geom = false;
    Geom G{};
    RegParams R{};
    // geometry tables (device)
    RayEntry *d_tab = nullptr;
    RayRange *d_rng = nullptr;
    float4 *d_views = nullptr;
    // TNLM tile lists (device): interior tiles first, then border tiles
    int2 *d_tiles = nullptr;
    int n_interior = 0, n_border = 0;
    size_t reg_smem = 0;
    // workspace, sized for ws_slices
    int ws_slices = 0;
    float *d_s = nullptr, *d_t = nullptr, *d_g = nullptr, *d_f = nullptr;  // images
    float *d_ua = nullptr, *d_ub = nullptr;                                  // sweep ping-pong
    float *d_r = nullptr, *d_rw = nullptr, *d_q = nullptr;                   // sinograms
    float *d_yh = nullptr, *d_wh = nullptr;                                  // host-API staging
    double *d_scal = nullptr;
    int scal_cap = 0;
    long long launches = 0;
    std::string err;
};

static std::string g_create_error;

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

extern "C" const char *tnlm_version(void) { return "tnlm-b200 0.1 (sm_100a)"; }

extern "C" const char *tnlm_last_error(const tnlm_handle *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

extern "C" long long tnlm_launch_count(const tnlm_handle *h) { return h ? h->launches : 0; }

// ------------------------------------------------------------------------------ tables
// Ray (phase i, view v, bin k) in grid units (pixel c covers [c, c+1) in xi, row r in eta):
// source (xs, es), unit direction (dx, dy).  Steep (|dy| >= |dx|): xi(eta) = p0 + m*eta with
// m = dx/dy, p0 = xs - m*es, length per full row = pix/|dy|.  Shallow: roles swapped.
static void build_tables(const tnlm_geometry &g, int nx, int ny, int n_phase, std::vector<RayEntry> &tab,
                         std::vector<RayRange> &rng, std::vector<float4> &views)
{
    const int V = g.n_views, B = g.n_bins;
    tab.resize((size_t)n_phase * V * B);
    rng.resize(tab.size());
    views.resize((size_t)n_phase * V);
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
                e.p0 = (float)p0; e.m = (float)m; e.len = (float)len;
                e.inva = (e.m != 0.f) ? 1.0f / std::fabs(e.m) : 0.f;
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
                r.lo = (short)lo; r.hi = (short)hi; r.steep = steep ? 1 : 0;
                tab[((size_t)i * V + v) * B + k] = e;
                rng[((size_t)i * V + v) * B + k] = r;
            }
        }
}

static size_t reg_smem_bytes(int window, int patch)
{
    const int a = (window - 1) / 2, b = (patch - 1) / 2, halo = a + b;
    const int TW = REG_TX * TQ, TH = REG_TY * TQ;
    const int gw = TW + 2 * halo, gh = TH + 2 * halo, uh = TH + 2 * a;
    const int P = (((gw + 3) >> 2) | 1);
    return (size_t)(gh + uh) * 4 * P * sizeof(float);
}

template <int PB, bool BORDER>
static cudaError_t set_reg_attr(size_t smem)
{
    return cudaFuncSetAttribute(gj_sweep_kernel<PB, REG_TX, REG_TY, BORDER>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
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

    // TNLM parameters
    RegParams &R = H->R;
    R.nx = nx; R.ny = ny; R.n_phase = n_phase; R.a = (window - 1) / 2;
    const double c = 1.4426950408889634 / ((double)h * (double)h);
    R.neg_c = (float)(-c);
    R.c_self = (float)(1.0 / (1.0 + (double)mu));
    R.c_nb = (float)((double)mu / (2.0 * (double)mu + 2.0));
    R.big_d = (float)std::fmin(1e37, 1e30 / c);
    R.m_init = R.neg_c * R.big_d * 0.1f;
    R.clip = 0;
    H->reg_smem = reg_smem_bytes(window, patch);
    if (H->reg_smem > (size_t)prop.sharedMemPerBlockOptin) {
        delete H;
        return fail(nullptr, TNLM_UNSUPPORTED, "window/patch need more shared memory than one CTA has");
    }
    {
        cudaError_t e = cudaSuccess;
        switch ((patch - 1) / 2) {
            case 0: e = set_reg_attr<0, false>(H->reg_smem); if (e == cudaSuccess) e = set_reg_attr<0, true>(H->reg_smem); break;
            case 1: e = set_reg_attr<1, false>(H->reg_smem); if (e == cudaSuccess) e = set_reg_attr<1, true>(H->reg_smem); break;
            case 2: e = set_reg_attr<2, false>(H->reg_smem); if (e == cudaSuccess) e = set_reg_attr<2, true>(H->reg_smem); break;
            case 3: e = set_reg_attr<3, false>(H->reg_smem); if (e == cudaSuccess) e = set_reg_attr<3, true>(H->reg_smem); break;
            default: e = set_reg_attr<4, false>(H->reg_smem); if (e == cudaSuccess) e = set_reg_attr<4, true>(H->reg_smem); break;
        }
        if (e != cudaSuccess) { delete H; return cuda_fail(nullptr, e, "cudaFuncSetAttribute"); }
    }
    // tile lists
    {
        const int TW = REG_TX * TQ, TH = REG_TY * TQ, a = R.a;
        std::vector<int2> inner, border;
        for (int ty = 0; ty < ny; ty += TH)
            for (int tx = 0; tx < nx; tx += TW) {
                const bool in = tx - a >= 0 && ty - a >= 0 && tx + TW - 1 + a <= nx - 1 && ty + TH - 1 + a <= ny - 1;
                (in ? inner : border).push_back(make_int2(tx, ty));
            }
        H->n_interior = (int)inner.size(); H->n_border = (int)border.size();
        inner.insert(inner.end(), border.begin(), border.end());
        if (cudaMalloc(&H->d_tiles, inner.size() * sizeof(int2)) != cudaSuccess) { delete H; return fail(nullptr, TNLM_ALLOC_FAILED, "device allocation failed (tiles)"); }
        ce = cudaMemcpy(H->d_tiles, inner.data(), inner.size() * sizeof(int2), cudaMemcpyHostToDevice);
        if (ce != cudaSuccess) { cudaFree(H->d_tiles); delete H; return cuda_fail(nullptr, ce, "cudaMemcpy tiles"); }
    }
    if (geometry) {
        const tnlm_geometry &g = *geometry;
        Geom &G = H->G;
        G.nx = nx; G.ny = ny; G.n_phase = n_phase; G.n_views = g.n_views; G.n_bins = g.n_bins;
        G.pix = (float)g.pixel_mm;
        G.sdd_over_pitch = (float)(g.sdd_mm / g.bin_pitch_mm);
        G.bin_centre = (float)(0.5 * (g.n_bins - 1) - g.bin_offset);
        G.half_diag = (float)(g.pixel_mm * 0.70710678118654752);
        std::vector<RayEntry> tab; std::vector<RayRange> rng; std::vector<float4> views;
        build_tables(g, nx, ny, n_phase, tab, rng, views);
        bool ok = cudaMalloc(&H->d_tab, tab.size() * sizeof(RayEntry)) == cudaSuccess &&
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
        H->has_geom = true;
    }
    *out = H;
    return TNLM_OK;
}

static void free_ws(tnlm_handle *H)
{
    float **bufs[] = {&H->d_s, &H->d_t, &H->d_g, &H->d_f, &H->d_ua, &H->d_ub, &H->d_r, &H->d_rw, &H->d_q, &H->d_yh, &H->d_wh};
    for (float **b : bufs) { if (*b) cudaFree(*b); *b = nullptr; }
    H->ws_slices = 0;
}

extern "C" int tnlm_destroy(tnlm_handle *H)
{
    if (!H) return TNLM_INVALID_ARG;
    free_ws(H);
    if (H->d_scal) cudaFree(H->d_scal);
    if (H->d_tab) cudaFree(H->d_tab);
    if (H->d_rng) cudaFree(H->d_rng);
    if (H->d_views) cudaFree(H->d_views);
    if (H->d_tiles) cudaFree(H->d_tiles);
    delete H;
    return TNLM_OK;
}

// Workspace for n_slices (grown, never shrunk).  Buffers are allocated on first need of their kind.
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

// ------------------------------------------------------------------------------ projector
template <int MODE>
static int launch_project(tnlm_handle *H, const float *img, const float *y, const float *w, float *out0,
                          float *out1, double *red, int n_slices, cudaStream_t st)
{
    const int nray = H->G.n_views * H->G.n_bins;
    dim3 grid((nray + 255) / 256, n_slices * H->n_phase);
    project_kernel<MODE><<<grid, 256, 0, st>>>(H->G, H->d_tab, H->d_rng, img, y, w, out0, out1, red);
    LAUNCHED(H);
    return TNLM_OK;
}
static int launch_backproject(tnlm_handle *H, const float *sino, float *img, double *red, int n_slices, cudaStream_t st)
{
    dim3 grid((H->nx + 31) / 32, (H->ny + BP_ROWS - 1) / BP_ROWS, n_slices * H->n_phase);
    backproject_kernel<<<grid, dim3(32, BP_ROWS), 0, st>>>(H->G, H->d_tab, H->d_rng, H->d_views, sino, img, red);
    LAUNCHED(H);
    return TNLM_OK;
}

extern "C" int tnlm_project(tnlm_handle *H, const float *img, float *sino, int n_slices, void *stream)
{
    int rc = check_common(H, n_slices, true);
    if (rc) return rc;
    if (!img || !sino) return fail(H, TNLM_INVALID_ARG, "img and sino must not be NULL");
    return launch_project<FWD_PLAIN>(H, img, nullptr, nullptr, sino, nullptr, nullptr, n_slices, (cudaStream_t)stream);
}

extern "C" int tnlm_backproject(tnlm_handle *H, const float *sino, float *img, int n_slices, void *stream)
{
    int rc = check_common(H, n_slices, true);
    if (rc) return rc;
    if (!img || !sino) return fail(H, TNLM_INVALID_ARG, "img and sino must not be NULL");
    return launch_backproject(H, sino, img, nullptr, n_slices, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------ CGLS
static int cgls_device(tnlm_handle *H, const float *f_in, const float *y, const float *w, int m1, float *g_out,
                       int n_slices, cudaStream_t st)
{
    const int nprob = n_slices * H->n_phase;
    const int npix = H->nx * H->ny, nray = H->G.n_views * H->G.n_bins;
    const size_t nimg = (size_t)nprob * npix;
    if (g_out != f_in) CU(H, cudaMemcpyAsync(g_out, f_in, nimg * sizeof(float), cudaMemcpyDeviceToDevice, st));
    if (m1 == 0) return TNLM_OK;
    int rc;
    if ((rc = need(H, &H->d_s, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_t, img_count(H)))) return rc;
    if ((rc = need(H, &H->d_r, sino_count(H)))) return rc;
    if ((rc = need(H, &H->d_rw, sino_count(H)))) return rc;
    if ((rc = need(H, &H->d_q, sino_count(H)))) return rc;
    const int nscal = (2 * m1 + 1) * nprob;
    if (nscal > H->scal_cap) {
        if (H->d_scal) cudaFree(H->d_scal);
        H->d_scal = nullptr; H->scal_cap = 0;
        if (cudaMalloc(&H->d_scal, (size_t)nscal * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return fail(H, TNLM_ALLOC_FAILED, "device allocation failed (scalars)"); }
        H->scal_cap = nscal;
    }
    double *gam = H->d_scal, *qq = H->d_scal + (size_t)(m1 + 1) * nprob;
    CU(H, cudaMemsetAsync(H->d_scal, 0, (size_t)nscal * sizeof(double), st));
    float *u = g_out;
    dim3 gi((npix + 255) / 256, nprob), gs((nray + 255) / 256, nprob);
    // init (L109): r = y_n - P_n u ; s = P_n^T r ; gamma_0 = ||s||^2
    if ((rc = launch_project<FWD_RESID>(H, u, y, w, H->d_r, H->d_rw, nullptr, n_slices, st))) return rc;
    if ((rc = launch_backproject(H, H->d_rw, H->d_s, gam, n_slices, st))) return rc;
    for (int m = 0; m < m1; ++m) {
        // q = P_n s ; qq_m = ||q||^2
        if ((rc = launch_project<FWD_SCALE>(H, H->d_s, nullptr, w, H->d_q, nullptr, qq + (size_t)m * nprob, n_slices, st))) return rc;
        cgls_update_u<<<gi, 256, 0, st>>>(u, H->d_s, npix, gam, qq, nprob, m);
        LAUNCHED(H);
        if (m + 1 == m1) break;      // r, t, s of the last step feed nothing (g = u^(M1), L127)
        cgls_update_r<<<gs, 256, 0, st>>>(H->d_r, H->d_rw, H->d_q, w, nray, gam, qq, nprob, m);
        LAUNCHED(H);
        if ((rc = launch_backproject(H, H->d_rw, H->d_t, gam + (size_t)(m + 1) * nprob, n_slices, st))) return rc;
        cgls_update_s<<<gi, 256, 0, st>>>(H->d_s, H->d_t, npix, gam, qq, nprob, m);
        LAUNCHED(H);
    }
    return TNLM_OK;
}

extern "C" int tnlm_cgls_step(tnlm_handle *H, const float *f_in, const float *y, const float *w, int m1,
                              float *g_out, int n_slices, void *stream)
{
    int rc = check_common(H, n_slices, true);
    if (rc) return rc;
    if (!f_in || !y || !g_out) return fail(H, TNLM_INVALID_ARG, "f_in, y and g_out must not be NULL");
    if (m1 < 0) return fail(H, TNLM_INVALID_ARG, "m1 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    return cgls_device(H, f_in, y, w, m1, g_out, n_slices, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------ TNLM
template <int PB>
static int launch_sweep_pb(tnlm_handle *H, const float *g, const float *u, float *out, int clip, int n_slices, cudaStream_t st)
{
    RegParams R = H->R;
    R.clip = clip;
    const int nimg = n_slices * H->n_phase;
    const int per = H->n_interior + H->n_border;
    if (H->n_interior > 0) {
        gj_sweep_kernel<PB, REG_TX, REG_TY, false><<<H->n_interior * nimg, REG_TX * REG_TY, H->reg_smem, st>>>(
            R, g, u, out, H->d_tiles, H->n_interior);
        LAUNCHED(H);
    }
    if (H->n_border > 0) {
        gj_sweep_kernel<PB, REG_TX, REG_TY, true><<<H->n_border * nimg, REG_TX * REG_TY, H->reg_smem, st>>>(
            R, g, u, out, H->d_tiles + H->n_interior, H->n_border);
        LAUNCHED(H);
    }
    (void)per;
    return TNLM_OK;
}
static int launch_sweep(tnlm_handle *H, const float *g, const float *u, float *out, int clip, int n_slices, cudaStream_t st)
{
    switch ((H->patch - 1) / 2) {
        case 0: return launch_sweep_pb<0>(H, g, u, out, clip, n_slices, st);
        case 1: return launch_sweep_pb<1>(H, g, u, out, clip, n_slices, st);
        case 2: return launch_sweep_pb<2>(H, g, u, out, clip, n_slices, st);
        case 3: return launch_sweep_pb<3>(H, g, u, out, clip, n_slices, st);
        default: return launch_sweep_pb<4>(H, g, u, out, clip, n_slices, st);
    }
}

// g -> f_out; g and f_out are distinct device buffers or the same buffer.
static int regularize_device(tnlm_handle *H, const float *g, int m2, float *f_out, int n_slices, cudaStream_t st)
{
    const size_t n = (size_t)n_slices * H->n_phase * H->nx * H->ny;
    int rc;
    if (m2 == 0) {
        clip_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, f_out, n);
        LAUNCHED(H);
        return TNLM_OK;
    }
    const bool alias = (f_out == g);
    if (m2 > 1 || alias) if ((rc = need(H, &H->d_ua, img_count(H)))) return rc;
    if (m2 > 2 || (alias && m2 > 1)) if ((rc = need(H, &H->d_ub, img_count(H)))) return rc;
    const float *src = g;
    float *pp[2] = {H->d_ua, H->d_ub};
    int which = 0;
    for (int m = 0; m < m2; ++m) {
        const bool last = (m + 1 == m2);
        float *dst;
        if (last && !alias) dst = f_out;
        else { dst = pp[which]; if (dst == src) { which ^= 1; dst = pp[which]; } }
        if ((rc = launch_sweep(H, g, src, dst, last ? 1 : 0, n_slices, st))) return rc;
        src = dst;
        which ^= 1;
    }
    if (alias) CU(H, cudaMemcpyAsync(f_out, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return TNLM_OK;
}

extern "C" int tnlm_regularize_step(tnlm_handle *H, const float *g, int m2, float *f_out, int n_slices, void *stream)
{
    int rc = check_common(H, n_slices, false);
    if (rc) return rc;
    if (!g || !f_out) return fail(H, TNLM_INVALID_ARG, "g and f_out must not be NULL");
    if (m2 < 0) return fail(H, TNLM_INVALID_ARG, "m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    return regularize_device(H, g, m2, f_out, n_slices, (cudaStream_t)stream);
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
    for (int k = 0; k < k_outer; ++k) {
        if ((rc = cgls_device(H, f_out, y, w, m1, H->d_g, n_slices, st))) return rc;       // step 2 (L176)
        if ((rc = regularize_device(H, H->d_g, m2, f_out, n_slices, st))) return rc;       // steps 3-5
    }
    return TNLM_OK;
}

extern "C" int tnlm_reconstruct(tnlm_handle *H, const float *y, const float *w, const float *f0, int k_outer, int m1,
                                int m2, float *f_out, int n_slices, void *stream)
{
    int rc = check_common(H, n_slices, true);
    if (rc) return rc;
    if (!y || !f_out) return fail(H, TNLM_INVALID_ARG, "y and f_out must not be NULL");
    if (k_outer < 0 || m1 < 0 || m2 < 0) return fail(H, TNLM_INVALID_ARG, "k_outer, m1, m2 must be >= 0");
    if ((rc = ensure_ws(H, n_slices))) return rc;
    return reconstruct_device(H, y, w, f0, k_outer, m1, m2, f_out, n_slices, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------ host-buffer entry points
extern "C" int tnlm_regularize_step_host(tnlm_handle *H, const float *g_host, int m2, float *f_out_host, int n_slices, void *stream)
{
    int rc = check_common(H, n_slices, false);
    if (rc) return rc;
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
    int rc = check_common(H, n_slices, true);
    if (rc) return rc;
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
