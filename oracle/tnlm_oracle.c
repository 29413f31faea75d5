/*
 * tnlm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU restatement of the hot path of
 * "Low-dose 4DCT Reconstruction via Temporal Nonlocal Means" (arxiv 1009.1351),
 * written from /root/reference/PAPER.md (cited below as PAPER.md:L<line>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  It shares no code, header, table or helper with the
 * CUDA path under paper_1009_1351_b200/ and is never imported by it.
 *
 * What it computes, in the paper's order and notation:
 *   oracle_project / oracle_backproject   P_i f and P_i^T g
 *   oracle_cgls_step                      "CGLS Algorithm"
 *   oracle_tnlm_*                         Eq.(3)/(8) weights
 *   oracle_regularize_step                "Gauss-Jacobi iteration"
 *   oracle_reconstruct                    "TNLM Algorithm"
 *   oracle_cost                           Eq.(1), Eq.(2)
 *
 * No blocking, no box sums, no symmetric reuse, no fusion: the patch distance is the
 * plain O(d^2) loop per (pixel, candidate) and P^T is the scatter form of P's own ray
 * loop, so the code can be checked against the paper by eye.
 *
 * Parity pins: see tests/test_oracle_*.py.  oracle_cost (Eq. 1 value) is "parity
 * unpinned" as a whole (its data term and J term are pinned separately on tiny cases,
 * but the paper proves no property of the summed value).
 *
 * Readings of silent/garbled passages follow DESIGN.md section "Readings".
 *
 * Layouts (all double, row-major, contiguous):
 *   images    [S][N][ny][nx]        pixel (r,c): centre X=(c-(nx-1)/2)*pix, Y=(r-(ny-1)/2)*pix
 *   sinograms [S][N][V][B]
 *   angles    [N][V]  (radians)
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int nx, ny, n_phase;
    int n_views, n_bins;
    double sid, sdd, pitch, bin_offset, pix;
    const double *angles; /* [n_phase][n_views] */
} geom_t;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* Geometry (fan beam, arc detector, source-isocentre SID,    */
/* source-detector SDD).  Source of view angle th: S = SID*(cos th, sin th). */
/* Bin k sits at fan angle gam_k = (k-(B-1)/2+off)*pitch/SDD on the arc; its  */
/* pencil ray leaves S in direction -(cos(th+gam_k), sin(th+gam_k)).          */
/* ------------------------------------------------------------------------- */
static void ray_of(const geom_t *G, int phase, int view, int bin,
                   double *sx, double *sy, double *dx, double *dy)
{
    double th = G->angles[(size_t)phase * G->n_views + view];
    double gam = ((double)bin - 0.5 * (G->n_bins - 1) + G->bin_offset) * G->pitch / G->sdd;
    *sx = G->sid * cos(th);
    *sy = G->sid * sin(th);
    *dx = -cos(th + gam);
    *dy = -sin(th + gam);
}

/* Length of the line S + t*d (|d| = 1) inside the box [x0,x1]x[y0,y1].  A ray running
 * exactly along a grid line (measure zero) is attributed to the pixel on its upper side
 * only (half-open [x0,x1)), so that it is counted once. */
static double clip_len(double sx, double sy, double dx, double dy,
                       double x0, double x1, double y0, double y1)
{
    double t0 = -INFINITY, t1 = INFINITY;
    if (dx != 0.0) {
        double ta = (x0 - sx) / dx, tb = (x1 - sx) / dx;
        if (ta > tb) { double t = ta; ta = tb; tb = t; }
        if (ta > t0) t0 = ta;
        if (tb < t1) t1 = tb;
    } else if (sx < x0 || sx >= x1) {
        return 0.0;
    }
    if (dy != 0.0) {
        double ta = (y0 - sy) / dy, tb = (y1 - sy) / dy;
        if (ta > tb) { double t = ta; ta = tb; tb = t; }
        if (ta > t0) t0 = ta;
        if (tb < t1) t1 = tb;
    } else if (sy < y0 || sy >= y1) {
        return 0.0;
    }
    return (t1 > t0) ? (t1 - t0) : 0.0;
}

/* One ray against the pixel grid, row by row (radiological path, Siddon ref. 24,
 * PAPER.md:L212).  For each row the ray can only touch the columns between its x
 * positions at the row's two y-faces; every such pixel is clipped individually.
 *   mode 0 (P)  : returns sum_pix len*img[pix]
 *   mode 1 (P^T): img[pix] += len*val          (same loop => exact transpose)
 */
static double ray_walk(const geom_t *G, double sx, double sy, double dx, double dy,
                       double *img, int mode, double val)
{
    const int nx = G->nx, ny = G->ny;
    const double pix = G->pix;
    const double xleft = -0.5 * nx * pix, ybot = -0.5 * ny * pix;
    double acc = 0.0;
    for (int r = 0; r < ny; ++r) {
        double y0 = ybot + r * pix, y1 = y0 + pix;
        int c_lo = 0, c_hi = nx - 1;
        if (dy != 0.0) {
            double ta = (y0 - sy) / dy, tb = (y1 - sy) / dy;
            double xa = sx + ta * dx, xb = sx + tb * dx;
            double xmin = xa < xb ? xa : xb, xmax = xa < xb ? xb : xa;
            double fl = floor((xmin - xleft) / pix) - 1.0, fh = floor((xmax - xleft) / pix) + 1.0;
            if (fh < 0.0 || fl > (double)(nx - 1)) continue;
            if (fl > 0.0) c_lo = (int)fl;
            if (fh < (double)(nx - 1)) c_hi = (int)fh;
        } else if (sy < y0 || sy >= y1) {
            continue;
        }
        for (int c = c_lo; c <= c_hi; ++c) {
            double x0 = xleft + c * pix;
            double len = clip_len(sx, sy, dx, dy, x0, x0 + pix, y0, y1);
            if (len > 0.0) {
                if (mode == 0) acc += len * img[(size_t)r * nx + c];
                else           img[(size_t)r * nx + c] += len * val;
            }
        }
    }
    return acc;
}

static geom_t make_geom(int nx, int ny, int n_phase, int n_views, int n_bins, double sid,
                        double sdd, double pitch, double bin_offset, double pix,
                        const double *angles)
{
    geom_t G;
    G.nx = nx; G.ny = ny; G.n_phase = n_phase; G.n_views = n_views; G.n_bins = n_bins;
    G.sid = sid; G.sdd = sdd; G.pitch = pitch; G.bin_offset = bin_offset; G.pix = pix;
    G.angles = angles;
    return G;
}

/* (P f)[v,k] = sum_pix len(ray_{v,k} ∩ pix) * f[pix] */
static void project_phase(const geom_t *G, int phase, const double *img, double *sino)
{
    const int V = G->n_views, B = G->n_bins;
#pragma omp parallel for schedule(dynamic, 1)
    for (int v = 0; v < V; ++v)
        for (int k = 0; k < B; ++k) {
            double sx, sy, dx, dy;
            ray_of(G, phase, v, k, &sx, &sy, &dx, &dy);
            sino[(size_t)v * B + k] = ray_walk(G, sx, sy, dx, dy, (double *)img, 0, 0.0);
        }
}

/* (P^T g)[pix] = sum_{v,k} len(ray_{v,k} ∩ pix) * g[v,k]     PAPER.md:L79 ("T denotes the
 * matrix transpose").  Scatter form of the same ray loop; threads own private images
 * that are summed in thread order at the end. */
static void backproject_phase(const geom_t *G, int phase, const double *sino, double *img)
{
    const int V = G->n_views, B = G->n_bins;
    const size_t npix = (size_t)G->nx * G->ny;
    int nt = oracle_num_threads();
    double *priv = (double *)calloc(npix * (size_t)nt, sizeof(double));
#pragma omp parallel
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        double *mine = priv + npix * (size_t)tid;
#pragma omp for schedule(static)   /* fixed view->thread map: reproducible summation order */
        for (int v = 0; v < V; ++v)
            for (int k = 0; k < B; ++k) {
                double sx, sy, dx, dy;
                ray_of(G, phase, v, k, &sx, &sy, &dx, &dy);
                ray_walk(G, sx, sy, dx, dy, mine, 1, sino[(size_t)v * B + k]);
            }
    }
    for (size_t p = 0; p < npix; ++p) {
        double s = 0.0;
        for (int t = 0; t < nt; ++t) s += priv[npix * (size_t)t + p];
        img[p] = s;
    }
    free(priv);
}

int oracle_project(int nx, int ny, int n_phase, int n_views, int n_bins, double sid, double sdd,
                   double pitch, double bin_offset, double pix, const double *angles,
                   const double *img, double *sino, int n_slices)
{
    geom_t G = make_geom(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles);
    const size_t npix = (size_t)nx * ny, nray = (size_t)n_views * n_bins;
    for (int s = 0; s < n_slices; ++s)
        for (int i = 0; i < n_phase; ++i)
            project_phase(&G, i, img + ((size_t)s * n_phase + i) * npix,
                          sino + ((size_t)s * n_phase + i) * nray);
    return 0;
}

int oracle_backproject(int nx, int ny, int n_phase, int n_views, int n_bins, double sid, double sdd,
                       double pitch, double bin_offset, double pix, const double *angles,
                       const double *sino, double *img, int n_slices)
{
    geom_t G = make_geom(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles);
    const size_t npix = (size_t)nx * ny, nray = (size_t)n_views * n_bins;
    for (int s = 0; s < n_slices; ++s)
        for (int i = 0; i < n_phase; ++i)
            backproject_phase(&G, i, sino + ((size_t)s * n_phase + i) * nray,
                              img + ((size_t)s * n_phase + i) * npix);
    return 0;
}

/* Sampled outputs for full-size parity: rays[q] = flat index into [N][V][B] of ONE slice. */
int oracle_project_rays(int nx, int ny, int n_phase, int n_views, int n_bins, double sid, double sdd,
                        double pitch, double bin_offset, double pix, const double *angles,
                        const double *img, int n_rays, const long long *rays, double *out)
{
    geom_t G = make_geom(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles);
    const size_t npix = (size_t)nx * ny;
#pragma omp parallel for schedule(dynamic, 16)
    for (int q = 0; q < n_rays; ++q) {
        long long id = rays[q];
        int k = (int)(id % n_bins), v = (int)((id / n_bins) % n_views), i = (int)(id / ((long long)n_bins * n_views));
        double sx, sy, dx, dy;
        ray_of(&G, i, v, k, &sx, &sy, &dx, &dy);
        out[q] = ray_walk(&G, sx, sy, dx, dy, (double *)(img + (size_t)i * npix), 0, 0.0);
    }
    return 0;
}

/* pixels[q] = flat index into [N][ny][nx] of ONE slice.  Brute force: every ray of the
 * phase is clipped against that one pixel square. */
int oracle_backproject_pixels(int nx, int ny, int n_phase, int n_views, int n_bins, double sid,
                              double sdd, double pitch, double bin_offset, double pix,
                              const double *angles, const double *sino, int n_pixels,
                              const long long *pixels, double *out)
{
    geom_t G = make_geom(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles);
    const size_t nray = (size_t)n_views * n_bins;
    const double xleft = -0.5 * nx * pix, ybot = -0.5 * ny * pix;
#pragma omp parallel for schedule(dynamic, 1)
    for (int q = 0; q < n_pixels; ++q) {
        long long id = pixels[q];
        int c = (int)(id % nx), r = (int)((id / nx) % ny), i = (int)(id / ((long long)nx * ny));
        double x0 = xleft + c * pix, y0 = ybot + r * pix, acc = 0.0;
        for (int v = 0; v < n_views; ++v)
            for (int k = 0; k < n_bins; ++k) {
                double sx, sy, dx, dy;
                ray_of(&G, i, v, k, &sx, &sy, &dx, &dy);
                double len = clip_len(sx, sy, dx, dy, x0, x0 + pix, y0, y0 + pix);
                if (len > 0.0) acc += len * sino[(size_t)i * nray + (size_t)v * n_bins + k];
            }
        out[q] = acc;
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* CGLS Algorithm, per phase, on P_n = Sigma^{-1/2} P,    */
/* y_n = Sigma^{-1/2} y (L103).  w = diagonal of Sigma^{-1} (NULL = identity). */
/* Breakdown (||P_n s||^2 = 0 or ||P_n^T r||^2 = 0): that phase stops, u stays. */
/* ------------------------------------------------------------------------- */
static double dot_self(const double *a, size_t n)
{
    double s = 0.0;
    for (size_t i = 0; i < n; ++i) s += a[i] * a[i];
    return s;
}

static void cgls_phase(const geom_t *G, int phase, const double *f_in, const double *y,
                       const double *w, int m1, double *g_out)
{
    const size_t npix = (size_t)G->nx * G->ny, nray = (size_t)G->n_views * G->n_bins;
    double *u = (double *)malloc(npix * sizeof(double));
    double *s = (double *)malloc(npix * sizeof(double));
    double *t = (double *)malloc(npix * sizeof(double));
    double *r = (double *)malloc(nray * sizeof(double));
    double *q = (double *)malloc(nray * sizeof(double));
    double *tmp = (double *)malloc(nray * sizeof(double));
    double *sw = (double *)malloc(nray * sizeof(double));
    for (size_t j = 0; j < nray; ++j) sw[j] = w ? sqrt(w[j]) : 1.0;

    /* Initialize: u0 = f^(k-1); r0 = y_n - P_n u0; s0 = P_n^T r0          (L109) */
    memcpy(u, f_in, npix * sizeof(double));
    project_phase(G, phase, u, q);
    for (size_t j = 0; j < nray; ++j) r[j] = sw[j] * y[j] - sw[j] * q[j];
    for (size_t j = 0; j < nray; ++j) tmp[j] = sw[j] * r[j];
    backproject_phase(G, phase, tmp, s);
    double gamma = dot_self(s, npix);            /* ||P_n^T r^(0)||^2 */

    for (int m = 0; m < m1; ++m) {
        if (!(gamma > 0.0)) break;
        project_phase(G, phase, s, q);
        for (size_t j = 0; j < nray; ++j) q[j] *= sw[j];          /* q = P_n s^(m) */
        double qq = dot_self(q, nray);
        if (!(qq > 0.0)) break;
        double a = gamma / qq;                                    /* step 1 (L112) */
        for (size_t p = 0; p < npix; ++p) u[p] += a * s[p];       /* step 2 (L114) */
        for (size_t j = 0; j < nray; ++j) r[j] -= a * q[j];       /* step 3 (L115) */
        for (size_t j = 0; j < nray; ++j) tmp[j] = sw[j] * r[j];
        backproject_phase(G, phase, tmp, t);                      /* P_n^T r^(m+1) */
        double gamma_new = dot_self(t, npix);
        double b = gamma_new / gamma;                             /* step 4 (L125) */
        for (size_t p = 0; p < npix; ++p) s[p] = t[p] + b * s[p]; /* step 5 (L126) */
        gamma = gamma_new;
    }
    memcpy(g_out, u, npix * sizeof(double));                      /* step 6 (L127) */
    free(u); free(s); free(t); free(r); free(q); free(tmp); free(sw);
}

int oracle_cgls_step(int nx, int ny, int n_phase, int n_views, int n_bins, double sid, double sdd,
                     double pitch, double bin_offset, double pix, const double *angles,
                     const double *f_in, const double *y, const double *w, int m1,
                     double *g_out, int n_slices)
{
    geom_t G = make_geom(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles);
    const size_t npix = (size_t)nx * ny, nray = (size_t)n_views * n_bins;
    for (int s = 0; s < n_slices; ++s)
        for (int i = 0; i < n_phase; ++i) {
            size_t io = ((size_t)s * n_phase + i) * npix, so = ((size_t)s * n_phase + i) * nray;
            cgls_phase(&G, i, f_in + io, y + so, w ? w + so : NULL, m1, g_out + io);
        }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* TNLM weights, Eq.(3)/(8): PAPER.md:L88-L94, L162-L165; window L204.        */
/* Patches are d x d, zero-extended outside the image; candidates y = x+delta */
/* range over the W x W window, in-image only (readings 5-7).       */
/* ------------------------------------------------------------------------- */
static double pix_or_zero(const double *im, int ny, int nx, int r, int c)
{
    return (r < 0 || r >= ny || c < 0 || c >= nx) ? 0.0 : im[(size_t)r * nx + c];
}

/* || R_gi(x) - R_gj(y) ||_2^2, plain sum over the d x d patch (L90). */
static double patch_dist(const double *gi, const double *gj, int ny, int nx, int b,
                         int xr, int xc, int yr, int yc)
{
    double D = 0.0;
    for (int pr = -b; pr <= b; ++pr)
        for (int pc = -b; pc <= b; ++pc) {
            double e = pix_or_zero(gi, ny, nx, xr + pr, xc + pc) -
                       pix_or_zero(gj, ny, nx, yr + pr, yc + pc);
            D += e * e;
        }
    return D;
}

/* exp(-||R_i(x)-R_j(y)||^2/h^2): the weight "before normalization" (L206). */
double oracle_tnlm_raw_weight(const double *gi, const double *gj, int ny, int nx, int patch,
                              double h, int xr, int xc, int yr, int yc)
{
    return exp(-patch_dist(gi, gj, ny, nx, (patch - 1) / 2, xr, xc, yr, yc) / (h * h));
}

/* Normalised weights omega_{i,j}(x, x+delta) of one pixel x, row-major over delta in
 * [-a,a]^2 (0 where x+delta is outside the image).  Z makes them sum to 1 (L94); the
 * common factor exp(D_min/h^2) is taken out of numerator and denominator so Z >= 1. */
void oracle_tnlm_weights_pixel(const double *gi, const double *gj, int ny, int nx, int window,
                               int patch, double h, int xr, int xc, double *omega)
{
    const int a = (window - 1) / 2, b = (patch - 1) / 2;
    double Dmin = INFINITY;
    for (int dr = -a; dr <= a; ++dr)
        for (int dc = -a; dc <= a; ++dc) {
            int yr = xr + dr, yc = xc + dc;
            double *o = &omega[(size_t)(dr + a) * window + (dc + a)];
            if (yr < 0 || yr >= ny || yc < 0 || yc >= nx) { *o = -1.0; continue; }
            *o = patch_dist(gi, gj, ny, nx, b, xr, xc, yr, yc);
            if (*o < Dmin) Dmin = *o;
        }
    double Z = 0.0;
    for (int q = 0; q < window * window; ++q)
        if (omega[q] >= 0.0) { omega[q] = exp(-(omega[q] - Dmin) / (h * h)); Z += omega[q]; }
        else omega[q] = 0.0;
    for (int q = 0; q < window * window; ++q) omega[q] /= Z;
}

/* One Gauss-Jacobi sweep, step 1 of the listing (L153), all phases simultaneously:
 *   u_i^{m+1}(x) = g_i(x)/(1+mu) + mu/(2mu+2) [ sum_y u_{i-1}^m(y) w_{i,i-1}(x,y)
 *                                             + sum_y u_{i+1}^m(y) w_{i,i+1}(x,y) ]
 * with cyclic phases f_{N+1} = f_1 (L81) and weights from g (Eq. 8). */
static void gj_sweep(const double *g, const double *u, double *unew, int n_phase, int ny, int nx,
                     int window, int patch, double h, double mu)
{
    const int a = (window - 1) / 2;
    const size_t npix = (size_t)ny * nx;
#pragma omp parallel
    {
        double *omega = (double *)malloc(sizeof(double) * window * window);
#pragma omp for collapse(2) schedule(dynamic, 4)
        for (int i = 0; i < n_phase; ++i)
            for (int r = 0; r < ny; ++r)
                for (int c = 0; c < nx; ++c) {
                    double nb = 0.0;
                    for (int side = -1; side <= 1; side += 2) {
                        int j = ((i + side) % n_phase + n_phase) % n_phase;
                        oracle_tnlm_weights_pixel(g + i * npix, g + j * npix, ny, nx, window,
                                                  patch, h, r, c, omega);
                        double A = 0.0;
                        for (int dr = -a; dr <= a; ++dr)
                            for (int dc = -a; dc <= a; ++dc) {
                                double wq = omega[(size_t)(dr + a) * window + (dc + a)];
                                if (wq != 0.0)
                                    A += wq * u[j * npix + (size_t)(r + dr) * nx + (c + dc)];
                            }
                        nb += A;
                    }
                    unew[i * npix + (size_t)r * nx + c] =
                        g[i * npix + (size_t)r * nx + c] / (1.0 + mu) + mu / (2.0 * mu + 2.0) * nb;
                }
        free(omega);
    }
}

/* Steps 3-5 of the TNLM Algorithm (L177-L179): weights from g, M2 sweeps from u^0 = g,
 * then f = 0 where f < 0 (L167), once, after the sweeps. */
int oracle_regularize_step(int nx, int ny, int n_phase, int window, int patch, double h, double mu,
                           const double *g, int m2, double *f_out, int n_slices)
{
    const size_t nvol = (size_t)n_phase * ny * nx;
    double *u = (double *)malloc(nvol * sizeof(double));
    double *un = (double *)malloc(nvol * sizeof(double));
    for (int s = 0; s < n_slices; ++s) {
        const double *gs = g + (size_t)s * nvol;
        memcpy(u, gs, nvol * sizeof(double));
        for (int m = 0; m < m2; ++m) {
            gj_sweep(gs, u, un, n_phase, ny, nx, window, patch, h, mu);
            double *t = u; u = un; un = t;
        }
        for (size_t p = 0; p < nvol; ++p) f_out[(size_t)s * nvol + p] = u[p] < 0.0 ? 0.0 : u[p];
    }
    free(u); free(un);
    return 0;
}

/* One sweep evaluated only at sampled pixels (full-size parity): pixels[q] indexes
 * [N][ny][nx] of one slice; u is the current iterate, weights come from g. No clip. */
int oracle_gj_sweep_pixels(int nx, int ny, int n_phase, int window, int patch, double h, double mu,
                           const double *g, const double *u, int n_pixels, const long long *pixels,
                           double *out)
{
    const int a = (window - 1) / 2;
    const size_t npix = (size_t)ny * nx;
#pragma omp parallel
    {
        double *omega = (double *)malloc(sizeof(double) * window * window);
#pragma omp for schedule(dynamic, 8)
        for (int q = 0; q < n_pixels; ++q) {
            long long id = pixels[q];
            int c = (int)(id % nx), r = (int)((id / nx) % ny), i = (int)(id / ((long long)nx * ny));
            double nb = 0.0;
            for (int side = -1; side <= 1; side += 2) {
                int j = ((i + side) % n_phase + n_phase) % n_phase;
                oracle_tnlm_weights_pixel(g + i * npix, g + j * npix, ny, nx, window, patch, h, r, c, omega);
                for (int dr = -a; dr <= a; ++dr)
                    for (int dc = -a; dc <= a; ++dc) {
                        double wq = omega[(size_t)(dr + a) * window + (dc + a)];
                        if (wq != 0.0) nb += wq * u[j * npix + (size_t)(r + dr) * nx + (c + dc)];
                    }
            }
            out[q] = g[i * npix + (size_t)r * nx + c] / (1.0 + mu) + mu / (2.0 * mu + 2.0) * nb;
        }
        free(omega);
    }
    return 0;
}

/* TNLM Algorithm (L169-L180): f^0 = f0 (NULL = zeros; the paper's FBP start, L175, is
 * supplied by the caller); for k = 1..K: g = CGLS(f^{k-1}); f^k = steps 3-5 (g). */
int oracle_reconstruct(int nx, int ny, int n_phase, int n_views, int n_bins, double sid, double sdd,
                       double pitch, double bin_offset, double pix, const double *angles,
                       int window, int patch, double h, double mu, const double *y, const double *w,
                       const double *f0, int k_outer, int m1, int m2, double *f_out, int n_slices)
{
    const size_t nvol = (size_t)n_phase * ny * nx, n = nvol * (size_t)n_slices;
    double *f = (double *)calloc(n, sizeof(double));
    double *g = (double *)malloc(n * sizeof(double));
    if (f0) memcpy(f, f0, n * sizeof(double));
    for (int k = 0; k < k_outer; ++k) {
        oracle_cgls_step(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles,
                         f, y, w, m1, g, n_slices);
        oracle_regularize_step(nx, ny, n_phase, window, patch, h, mu, g, m2, f, n_slices);
    }
    memcpy(f_out, f, n * sizeof(double));
    free(f); free(g);
    return 0;
}

/* Cost function Eq.(1) (L77) with J of Eq.(2) (L83), one slice.  Weights are built from
 * gref (pass f itself for "weights from the current images"), restricted to the window.
 * out[0] = data term sum_i (P f_i - y_i)^T Sigma^-1 (P f_i - y_i)
 * out[1] = sum_i [J(f_i,f_{i-1}) + J(f_i,f_{i+1})]        (to be scaled by mu/2)
 * Pass n_views = 0 to skip the data term.  PARITY UNPINNED as a summed value. */
int oracle_cost(int nx, int ny, int n_phase, int n_views, int n_bins, double sid, double sdd,
                double pitch, double bin_offset, double pix, const double *angles, int window,
                int patch, double h, const double *f, const double *gref, const double *y,
                const double *w, double *out)
{
    const size_t npix = (size_t)nx * ny, nray = (size_t)n_views * n_bins;
    const int a = (window - 1) / 2;
    double data = 0.0, reg = 0.0;
    if (n_views > 0) {
        geom_t G = make_geom(nx, ny, n_phase, n_views, n_bins, sid, sdd, pitch, bin_offset, pix, angles);
        double *p = (double *)malloc(nray * sizeof(double));
        for (int i = 0; i < n_phase; ++i) {
            project_phase(&G, i, f + i * npix, p);
            for (size_t j = 0; j < nray; ++j) {
                double e = p[j] - y[i * nray + j];
                data += e * e * (w ? w[i * nray + j] : 1.0);
            }
        }
        free(p);
    }
    double *omega = (double *)malloc(sizeof(double) * window * window);
    for (int i = 0; i < n_phase; ++i)
        for (int side = -1; side <= 1; side += 2) {
            int j = ((i + side) % n_phase + n_phase) % n_phase;
            for (int r = 0; r < ny; ++r)
                for (int c = 0; c < nx; ++c) {
                    oracle_tnlm_weights_pixel(gref + i * npix, gref + j * npix, ny, nx, window, patch, h, r, c, omega);
                    for (int dr = -a; dr <= a; ++dr)
                        for (int dc = -a; dc <= a; ++dc) {
                            double wq = omega[(size_t)(dr + a) * window + (dc + a)];
                            if (wq != 0.0) {
                                double e = f[i * npix + (size_t)r * nx + c] -
                                           f[j * npix + (size_t)(r + dr) * nx + (c + dc)];
                                reg += e * e * wq;
                            }
                        }
                }
        }
    free(omega);
    out[0] = data;
    out[1] = reg;
    return 0;
}
