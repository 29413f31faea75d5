/*
 * tnlm.h -- C ABI of libtnlm: the data-parallel hot path of
 * "Low-dose 4DCT Reconstruction via Temporal Nonlocal Means" (arxiv 1009.1351) on one
 * NVIDIA B200 (sm_100a).  Citations are PAPER.md:L<line>.
 *
 * One modified forward-backward-splitting iteration over all N respiratory phases of a CT
 * slice at once ("TNLM Algorithm"):
 *     g^(k) = CGLS_{M1}( f^(k-1) ; P, P^T, Sigma^-1, y )               step 2   (L103-L135)
 *     w     = TNLM weights of g^(k) to the two cyclic neighbour phases  step 3   (Eq. 8)
 *     f^(k) = max( GaussJacobi_{M2}( g^(k) ; w, mu ), 0 )               steps 4-5 (Eq. 7)
 *
 * Conventions
 *   N = n_phase, image ny x nx (row-major), S = n_slices independent slices.
 *   Pixel (r,c) is the square of side pixel_mm centred at
 *       X = (c-(nx-1)/2)*pixel_mm,  Y = (r-(ny-1)/2)*pixel_mm           (isocentre = grid centre).
 *   Fan beam, equiangular arc detector (L212).  View angle th: source S = sid*(cos th, sin th);
 *   bin k sits at fan angle gam_k = (k-(n_bins-1)/2+bin_offset)*bin_pitch/sdd; its pencil ray
 *   leaves S in direction -(cos(th+gam_k), sin(th+gam_k)).
 *   (P f)[v,k] = sum_pix length(ray_{v,k} ∩ pixel) * f[pix]   (radiological path, Siddon, L212);
 *   P^T is its exact matrix transpose (L79).  A ray lying exactly on a grid line is attributed
 *   to the pixel on its upper side.
 *   TNLM: window W x W (odd, a=(W-1)/2), patch d x d (odd, b=(d-1)/2).  Patches are extended by
 *   zero outside the image; candidates y = x+delta, delta in [-a,a]^2, outside the image are
 *   excluded from the sums and from Z.  Phases are cyclic: f_{N+1} = f_1 (L81).
 *       D(x,delta)   = sum_{p in [-b,b]^2} ( g_i(x+p) - g_j(x+delta+p) )^2               (L90)
 *       w_ij(x,x+delta) = exp(-D/h^2) / Z,  Z = sum over in-image delta               (Eq. 3/8, L94)
 *       u_i' (x) = g_i(x)/(1+mu) + mu/(2mu+2) * sum_{j=i-1,i+1} sum_delta w_ij u_j(x+delta)  (Eq. 7)
 *   `mu` is the paper's mu-hat = mu/beta (L141).  The softmax is evaluated in a shifted,
 *   overflow/underflow-safe form; the value is the one defined above.
 *
 * Memory
 *   Every `float *` of the device entry points is a DEVICE pointer to a caller-owned,
 *   contiguous fp32 buffer:  images [S][N][ny][nx],  sinograms / weights [S][N][V][B].
 *   The `_host` entry points take HOST pointers with the same layouts.  The library never
 *   frees or keeps caller buffers.  Inputs are never modified.  Outputs may alias the input
 *   image of the same call where stated.  Workspace is owned by the handle, grown lazily to the
 *   largest n_slices seen, and freed by tnlm_destroy.
 *
 * Execution
 *   Device entry points enqueue work on `stream` (a cudaStream_t passed as void*, NULL = the
 *   legacy default stream) and return without waiting for it; all scalars of CGLS stay on the
 *   device.  The FIRST call that needs a workspace buffer of some kind, and any call with a larger
 *   n_slices than seen before, allocates it with cudaMalloc inside the call (a larger n_slices first
 *   releases every workspace buffer of the handle with cudaFree); both synchronise the device.
 *   tnlm_reserve does all of that up front, after which the enqueue calls never allocate or free.
 *   `_host` entry points copy in, run, copy out and synchronise `stream` before returning.  A handle belongs to the CUDA device that was current at tnlm_create: every entry
 *   point makes that device current for the call and restores the caller's; device pointers and
 *   the stream must belong to it.  A handle must not be used from two streams or threads at once.
 *
 * Stored weights and tuning knobs
 *   The weights belong to g^(k) and are the same in all m2 sweeps (L162).  By DEFAULT every sweep computes
 *   them again in fp32: that path meets the 1e-4 single-step bar on every valid input (1e-6 measured).
 *   OPT-IN (option weight_cache_mb > 0): for m2 > 1 the first sweep also stores the unnormalised weights
 *   (bf16, 2*W^2*2 bytes per pixel, handle-owned) and the later sweeps stream them (L206 "reusing this
 *   factor ... instead of recomputing"; 1.8x faster for m2 = 10); accumulation stays fp32.  Precision of the
 *   stored path: a stored weight is off by up to 2^-9 relative, which moves the result of a sweep by at most
 *   mu/(2 mu + 2) * 2^-7 * (spread of u inside the window).  On thorax-like images (BASELINE.json configs)
 *   that is 2e-6 relative L2 against the fp64 oracle; on binary images of 100 % contrast with a sharp softmax
 *   and mu >= 2 it reaches 2e-4 (1.3e-3 of the maximum), i.e. it can miss the 1e-4 bar: that is why it is
 *   not the default.  If the stored weights cannot be allocated the call fails with TNLM_ALLOC_FAILED.
 *   Options, read from the environment ONCE at tnlm_create and changed later with tnlm_set_option:
 *   weight_cache_mb / TNLM_WEIGHT_CACHE_MB (default 0 = never store; n > 0 = store when the weights of
 *   the call fit in n MB, e.g. 16384; larger needs recompute) and sweep_rb, sweep_nb / TNLM_SWEEP_SHAPE="rb,nb"
 *   (pin the launch shape of the sweep instead of the cost model's choice; 0 = free; values that name no
 *   compiled shape are refused).  Options without an environment variable (results are bit-identical either
 *   way): apply_depth (ring depth of the stored-weight sweep: 4, 8, 16; 0 = chosen by the library), apply_snake
 *   (1, the default: successive stored-weight sweeps take the stored bands in opposite orders, so a sweep starts
 *   on the bytes the previous one left in L2), apply_resident_mb (default 32: that many MB of the stored weights
 *   are written and read with an L2 evict_last policy, the rest with evict_first; 0 = all evict_first;
 *   tnlm_destroy does not reset the context's persisting L2 lines -- that would hit every other user of the
 *   context -- so those lines keep their priority until other evict_last traffic displaces them),
 *   project_kernel (-1 = by size, the default; 1 = shared-memory strips per warp; 0 = L1 gathers),
 *   backproject_group (16, the default; 8, 4, 2, 1): the slices of one call share the geometry (nothing couples
 *   them, L77), so one backprojector thread serves up to that many slices with one evaluation of the ray
 *   geometry; per slice the arithmetic and its order do not change; project_interleave (1, the default: in a call
 *   with four or more slices the forward projector reads handle-owned copies of the image in which the four
 *   slices of a group are interleaved per pixel, one 16-byte gather per cell for four slices; 0 = every slice
 *   from its own image and transposed copy), project_block (threads per CTA of the forward projector: 128, the
 *   default, 256 or 64; changes only how the ||q||^2 partial sums are grouped).
 *
 * Value range
 *   The shifted softmax keeps every weight sum below 2^100, so the numerators sum_delta w u_j stay
 *   finite for |u| < 2^17 (1.3e5; HU-scaled images are fine).  h must be <= 1e12, and large enough for
 *   log2(e)/h^2 to be a finite fp32 number (h > 7e-20); tnlm_create refuses others.
 *
 * Errors
 *   Every call returns a tnlm_status; nothing throws, exits or falls back to the CPU.
 *   tnlm_last_error(handle) gives a handle-owned message for the last failing call.
 */
#ifndef TNLM_H
#define TNLM_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TNLM_OK = 0,
    TNLM_INVALID_ARG = 1, /* NULL handle/buffer, bad sizes, even/too small window or patch, h<=0,
                             mu<0, negative iteration counts, projector call without geometry,
                             sid>=sdd, image not strictly inside the source circle */
    TNLM_CUDA_ERROR = 2,  /* a CUDA runtime call failed; message from cudaGetErrorString */
    TNLM_ALLOC_FAILED = 3,
    TNLM_UNSUPPORTED = 4  /* device is not sm_100, patch/window above the compiled maximum
                             (patch <= 9, window <= 31), flat detector, a fan of 180 degrees or more,
                             a source closer than six pixels to the circle around the image */
} tnlm_status;

typedef struct tnlm_handle tnlm_handle; /* opaque: geometry tables + workspace */

/* Scan geometry of one slice.  Read once by tnlm_create; not kept. */
typedef struct {
    int n_views;              /* views per phase, V */
    int n_bins;               /* detector bins, B */
    double sid_mm;            /* source to rotation centre */
    double sdd_mm;            /* source to detector */
    double bin_pitch_mm;      /* bin spacing along the arc */
    double bin_offset;        /* detector shift in bins, 0 = centred */
    double pixel_mm;          /* square pixel side */
    int detector_arc;         /* 1 = equiangular arc (the paper's); 0 = flat -> TNLM_UNSUPPORTED */
    const double *angles_rad; /* HOST, [n_phase][n_views] source angles; P_i differs per phase (L75) */
} tnlm_geometry;

/* Create a handle.  `geometry` may be NULL: TNLM-only handle, projector/CGLS/reconstruct
 * calls then return TNLM_INVALID_ARG.  window/patch odd >= 1; h > 0 finite; mu >= 0. */
int tnlm_create(const tnlm_geometry *geometry, int nx, int ny, int n_phase, int window, int patch,
                float h, float mu, tnlm_handle **out);
int tnlm_destroy(tnlm_handle *handle);

/* sino = P img.  img [S][N][ny][nx] -> sino [S][N][V][B]; must not alias. */
int tnlm_project(tnlm_handle *handle, const float *img, float *sino, int n_slices, void *stream);

/* img = P^T sino, the exact transpose of tnlm_project; must not alias. */
int tnlm_backproject(tnlm_handle *handle, const float *sino, float *img, int n_slices, void *stream);

/* "CGLS Algorithm": m1 steps on P_n = Sigma^-1/2 P, y_n = Sigma^-1/2 y,
 * per phase and slice, warm-started at f_in; g_out = u^(m1).  w = diagonal of Sigma^-1
 * (NULL = identity).  No positivity clip.  m1 = 0 copies f_in.  If ||P_n s||^2 or
 * ||P_n^T r||^2 is 0 for a phase that phase stops and keeps its iterate (no NaN).
 * g_out may alias f_in. */
int tnlm_cgls_step(tnlm_handle *handle, const float *f_in, const float *y, const float *w, int m1,
                   float *g_out, int n_slices, void *stream);

/* Steps 3-5: weights from g (Eq. 8), m2 Gauss-Jacobi sweeps of Eq. (7)
 * from u^0 = g with the weights fixed, then f = max(u, 0) once.  m2 = 0 gives max(g, 0).
 * f_out may alias g. */
int tnlm_regularize_step(tnlm_handle *handle, const float *g, int m2, float *f_out, int n_slices,
                         void *stream);

/* "TNLM Algorithm": f^0 = f0 (NULL = zeros; the paper's FBP start is the
 * caller's to supply), k_outer times { cgls_step(m1) ; regularize_step(m2) }.  k_outer = 0
 * copies f0.  f_out may alias f0. */
int tnlm_reconstruct(tnlm_handle *handle, const float *y, const float *w, const float *f0,
                     int k_outer, int m1, int m2, float *f_out, int n_slices, void *stream);

/* Step 1 of the "TNLM Algorithm": f0 = the filtered backprojection of ALL
 * projections of ALL n_phase phases (equiangular fan-beam FBP, ramp filter, views weighted by the
 * trapezoid rule over the sorted union of all source angles), the same image written to every
 * phase.  y [S][N][V][B] -> f0 [S][N][ny][nx]; feed it to tnlm_reconstruct as `f0`. */
int tnlm_fbp_init(tnlm_handle *handle, const float *y, float *f0, int n_slices, void *stream);

/* Same operations with HOST buffers: host->device copies, the device path above, the
 * device->host copy of the result, and a stream synchronise, all inside the call. */
int tnlm_regularize_step_host(tnlm_handle *handle, const float *g_host, int m2, float *f_out_host,
                              int n_slices, void *stream);
int tnlm_reconstruct_host(tnlm_handle *handle, const float *y_host, const float *w_host,
                          const float *f0_host, int k_outer, int m1, int m2, float *f_out_host,
                          int n_slices, void *stream);

/* tnlm_regularize_step for callers that must not allocate device memory.
 *
 * Who that is: a reconstruction service whose HBM is already handed out in full (to a framework's
 * caching allocator holding a 64-slice batch, or to another job sharing the GPU), where cudaMalloc
 * fails; and a scanner-side loop that keeps other streams busy (the upload of the next slice, a display
 * kernel) and cannot take the device-wide synchronisation cudaMalloc implies.  tnlm_regularize_step
 * allocates its ping-pong images and stored weights on first use, so neither can call it unprepared.
 *
 * What it does: the same result as tnlm_regularize_step (weights of g, m2 Gauss-Jacobi sweeps, clip;
 * same arguments, f_out may alias g), with the weights recomputed in fp32 in every sweep (nothing is
 * stored) and the intermediate sweeps written to a scratch array that is compiled into the library
 * (a file-scope __device__ array of 2 * TNLM_NOALLOC_MAX_PIXELS floats = 20 MiB).  It calls no
 * cudaMalloc, cudaFree or any other allocating routine; a TNLM-only handle (geometry = NULL) owns no
 * device memory either, so with such a handle the whole path is allocation-free.  Per-launch timing
 * (tnlm_profile_kernels) does not cover this call, because recording would create events.
 *
 * Limits and sharp edges
 *   - n_slices * n_phase * ny * nx must not exceed TNLM_NOALLOC_MAX_PIXELS (one 10-phase 512 x 512
 *     slice); larger calls return TNLM_UNSUPPORTED with a message naming both numbers.
 *   - The array is part of the library's device image: every GPU on which the library's CUDA code is
 *     loaded holds those 20 MiB until the process exits, whether or not this call is ever made.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with
 *     that device current), which can make the CUDA runtime load the library's device code.  Make
 *     that first call during set-up, before any stream capture is begun.
 *   - There is ONE array per device, shared by every handle, stream and thread.  Two calls that
 *     overlap on the GPU (different streams, or different handles without ordering between them) race on
 *     it and corrupt each other's sweeps; order them on one stream or with events.
 *   - The array keeps what the last call left in it.  Nothing has to be cleared: every sweep writes
 *     every pixel of its destination before the next sweep reads it, and pixels beyond the current
 *     call's size are never read. */
#define TNLM_NOALLOC_MAX_PIXELS 2621440
int tnlm_regularize_step_noalloc(tnlm_handle *handle, const float *g, int m2, float *f_out,
                                 int n_slices, void *stream);

/* Message of the last failing call on this handle ("" if none); handle-owned, valid until the
 * next call on the handle.  NULL handle -> message of the calling thread's last failed tnlm_create. */
const char *tnlm_last_error(const tnlm_handle *handle);

/* Allocate now everything a later tnlm_cgls_step / tnlm_regularize_step / tnlm_reconstruct call
 * with up to n_slices slices, m1 CGLS steps and m2 sweeps would allocate on first use
 * (host_entry_points != 0: also the staging buffers of the _host calls).  Synchronises the device. */
int tnlm_reserve(tnlm_handle *handle, int n_slices, int m1, int m2, int host_entry_points);

/* Change a tuning option of this handle (see "Stored weights and tuning knobs"): name is one of
 * "weight_cache_mb", "sweep_rb", "sweep_nb", "apply_depth", "apply_snake", "apply_resident_mb",
 * "project_kernel", "project_interleave", "project_block", "backproject_group"; 0 restores the
 * heuristic for the shape options.  Unknown names: TNLM_INVALID_ARG. */
int tnlm_set_option(tnlm_handle *handle, const char *name, long long value);

/* The CUDA device ordinal the handle was created on (-1 for a NULL handle). */
int tnlm_device(const tnlm_handle *handle);

/* Per-launch device timing of every kernel of the path, for benchmarks and rooflines.
 * tnlm_profile_kernels(handle, 1) makes every later call bracket each kernel launch with a CUDA
 * event pair on the call's stream (0 switches it off; either call forgets the launches recorded
 * so far).  One pair covers one operation on the whole batch: a projector application whose slices
 * run as several group sizes (say 8 + 2 + 1 slices per thread) is a few back-to-back launches inside
 * one pair.  tnlm_kernel_times waits for the recorded launches, writes up to `capacity` durations
 * (milliseconds, launch order) into the HOST arrays ms[] and kind[] (a tnlm_kernel_kind), stores
 * the number recorded in *count, and forgets them. */
typedef enum {
    TNLM_KERNEL_SWEEP = 0,       /* weights computed on the fly + one Gauss-Jacobi sweep (Eq. 3/8, Eq. 7) */
    TNLM_KERNEL_SWEEP_STORE = 1, /* the same, also storing the weights of g^(k) for sweeps 2..m2 */
    TNLM_KERNEL_APPLY = 2,       /* one Gauss-Jacobi sweep of Eq. (7) from the stored weights */
    TNLM_KERNEL_PROJECT = 3,     /* forward projector P with the CGLS epilogue (L75, L109, L112) */
    TNLM_KERNEL_BACKPROJECT = 4, /* backprojector P^T with the norm reduction (L79, L109, L124) */
    TNLM_KERNEL_TRANSPOSE = 5,   /* the image copies P reads: transposed (shallow rays) or, in a batch, four slices interleaved */
    TNLM_KERNEL_CGLS_VECTOR = 6, /* CGLS vector updates (L114-L126) and sqrt(w) */
    TNLM_KERNEL_CLIP = 7,        /* positivity clip alone (m2 = 0) */
    TNLM_KERNEL_FBP = 8          /* FBP initialisation kernels (L175) */
} tnlm_kernel_kind;
int tnlm_profile_kernels(tnlm_handle *handle, int enable);
int tnlm_kernel_times(tnlm_handle *handle, float *ms, int *kind, int capacity, int *count);

/* Measured FP32 (non-tensor) FMA peak of the current device in TFLOP/s (2 flops per FFMA): an
 * 8-chain FFMA kernel on every SM, best of 3 timed launches on `stream` (synchronises).  The
 * roofline denominator of the ALU-bound TNLM kernels; no handle needed. */
int tnlm_fma_peak(double *tflops, void *stream);

/* Number of CUDA kernels this handle has launched so far (for benchmark bookkeeping). */
long long tnlm_launch_count(const tnlm_handle *handle);

/* Library version string, e.g. "tnlm-b200 0.3 (sm_100a)". */
const char *tnlm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TNLM_H */
