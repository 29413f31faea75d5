"""Independent pins for the oracle (numpy, pure Python loops; tiny inputs only).

Nothing here calls oracle/ or the CUDA path.  Each function restates a DEFINITION from
the paper in the most literal way, so that the oracle's faster organisation (row walk,
window, min-subtracted softmax) is checked against something other than itself.
"""
import numpy as np


# ----------------------------------------------------------------------------- geometry
def ray(sid, sdd, pitch, n_bins, theta, k, off=0.0):
    """Source point and unit direction of bin k at view angle theta."""
    gam = (k - 0.5 * (n_bins - 1) + off) * pitch / sdd
    s = np.array([sid * np.cos(theta), sid * np.sin(theta)])
    d = -np.array([np.cos(theta + gam), np.sin(theta + gam)])
    return s, d


def chord_by_edges(s, d, x0, x1, y0, y1):
    """Length of the line s+t*d inside the rectangle, from its crossings of the 4 EDGE LINES
    (not a slab clip): collect crossing points that lie on the rectangle's boundary and
    return the distance between the two extreme ones."""
    ts = []
    eps = 1e-12
    if d[0] != 0.0:
        for xe in (x0, x1):
            t = (xe - s[0]) / d[0]
            y = s[1] + t * d[1]
            if y0 - eps <= y <= y1 + eps:
                ts.append(t)
    if d[1] != 0.0:
        for ye in (y0, y1):
            t = (ye - s[1]) / d[1]
            x = s[0] + t * d[0]
            if x0 - eps <= x <= x1 + eps:
                ts.append(t)
    if len(ts) < 2:
        return 0.0
    return (max(ts) - min(ts)) * float(np.hypot(d[0], d[1]))


def pixel_box(r, c, ny, nx, pix):
    xc = (c - 0.5 * (nx - 1)) * pix
    yc = (r - 0.5 * (ny - 1)) * pix
    return xc - 0.5 * pix, xc + 0.5 * pix, yc - 0.5 * pix, yc + 0.5 * pix


def dense_system_matrix(sid, sdd, pitch, n_bins, thetas, ny, nx, pix):
    """A[(v,k), (r,c)] = length of ray (v,k) inside pixel (r,c), every pair brute force."""
    A = np.zeros((len(thetas) * n_bins, ny * nx))
    for v, th in enumerate(thetas):
        for k in range(n_bins):
            s, d = ray(sid, sdd, pitch, n_bins, th, k)
            for r in range(ny):
                for c in range(nx):
                    A[v * n_bins + k, r * nx + c] = chord_by_edges(s, d, *pixel_box(r, c, ny, nx, pix))
    return A


# --------------------------------------------------------------------------------- TNLM
def _patch(im, r, c, b):
    """d x d patch around (r,c), zero outside the image."""
    ny, nx = im.shape
    out = np.zeros((2 * b + 1, 2 * b + 1))
    for pr in range(-b, b + 1):
        for pc in range(-b, b + 1):
            rr, cc = r + pr, c + pc
            if 0 <= rr < ny and 0 <= cc < nx:
                out[pr + b, pc + b] = im[rr, cc]
    return out


def weights_unrestricted(gi, gj, patch, h):
    """omega_{i,j}(x,y) of Eq.(3)/(8) for ALL pixel pairs (no search window):
    [ny,nx,ny,nx], normalised so that sum_y omega(x,y) = 1."""
    ny, nx = gi.shape
    b = (patch - 1) // 2
    om = np.zeros((ny, nx, ny, nx))
    for xr in range(ny):
        for xc in range(nx):
            Rx = _patch(gi, xr, xc, b)
            for yr in range(ny):
                for yc in range(nx):
                    om[xr, xc, yr, yc] = np.exp(-np.sum((Rx - _patch(gj, yr, yc, b)) ** 2) / h ** 2)
            om[xr, xc] /= om[xr, xc].sum()
    return om


def gauss_jacobi_unrestricted(g, patch, h, mu, m2):
    """Listing PAPER.md:L147-L158 with window-free weights from g, then clip (L167)."""
    N = g.shape[0]
    om = {}
    for i in range(N):
        for side in (-1, 1):
            j = (i + side) % N
            om[(i, side)] = weights_unrestricted(g[i], g[j], patch, h)
    u = g.copy()
    for _ in range(m2):
        un = np.zeros_like(u)
        for i in range(N):
            acc = np.zeros_like(g[i])
            for side in (-1, 1):
                j = (i + side) % N
                acc += np.einsum("abcd,cd->ab", om[(i, side)], u[j])
            un[i] = g[i] / (1.0 + mu) + mu / (2.0 * mu + 2.0) * acc
        u = un
    return np.maximum(u, 0.0)


def J_unrestricted(fi, fj, gi, gj, patch, h):
    """Eq.(2): sum_x sum_y [f_i(x)-f_j(y)]^2 omega_{i,j}(x,y), weights from (gi,gj)."""
    om = weights_unrestricted(gi, gj, patch, h)
    diff = fi[:, :, None, None] - fj[None, None, :, :]
    return float(np.sum(diff ** 2 * om))
