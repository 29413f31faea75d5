"""CPU oracle of the FBP initialisation -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Step 1 of the "TNLM Algorithm": "Initialize f_i^(0) for i = 1..N to be the image
reconstructed by FBP with all projections from all N phases."  The paper names the method and nothing
else, so this is the textbook filtered backprojection for an equiangular fan beam (Kak & Slaney,
"Principles of Computerized Tomographic Imaging", section 3.4.1, eqs. 92-96), written out step by step
in fp64 numpy with no blocking or reordering (reading 24):

  1. views: the union of the N*V (phase, view) source angles beta_j; weight of a view =
     (gap to its cyclic neighbours in the sorted union)/2, i.e. the trapezoid rule of the integral over
     beta, so unequal or repeated angles are handled;
  2. R'_j(n) = y_j(n) * SID * cos(gamma_n),  gamma_n = (n - (B-1)/2 + off) * dgamma,  dgamma = pitch/SDD;
  3. Q_j(n)  = dgamma * sum_m R'_j(m) g((n-m) dgamma),   g(0) = 1/(8 dgamma^2),  g(k dgamma) = 0 (k even),
     -1/(2 pi^2 sin^2(k dgamma)) (k odd)                      (ramp filter, eq. 96);
  4. f(x)    = sum_j dbeta_j * Q_j(gamma'(x)) / L_j(x)^2,  L = distance source - pixel centre,
     gamma' = fan angle of the pixel centre, Q linearly interpolated between bins (0 outside the detector);
     (the 1/2 for a 2 pi scan measuring every line twice is the 1/2 inside g, eq. 96);
  5. every phase gets the same image.

Geometry conventions are those of include/tnlm.h: source S = SID (cos beta, sin beta); the ray of fan
angle gamma leaves S in direction -(cos(beta+gamma), sin(beta+gamma)).
Only tests/, __graft_entry__.smoke() and bench.py may import this module.
"""
import numpy as np


def view_weights(angles_rad):
    """dbeta_j of the trapezoid rule over the sorted cyclic union of all source angles; same shape as input."""
    ang = np.asarray(angles_rad, dtype=np.float64)
    flat = np.mod(ang.ravel(), 2.0 * np.pi)
    order = np.argsort(flat, kind="stable")
    s = flat[order]
    nxt = np.roll(s, -1)
    prv = np.roll(s, 1)
    nxt[-1] += 2.0 * np.pi
    prv[0] -= 2.0 * np.pi
    w = np.empty_like(flat)
    w[order] = 0.5 * (nxt - prv)
    return w.reshape(ang.shape)


def ramp_kernel(n_bins, dgamma):
    """g(k dgamma) for k = -(B-1) .. B-1 (index k + B - 1)."""
    k = np.arange(-(n_bins - 1), n_bins)
    g = np.zeros(k.shape, dtype=np.float64)
    odd = (k % 2) != 0
    g[odd] = -1.0 / (2.0 * np.pi ** 2 * np.sin(k[odd] * dgamma) ** 2)
    g[k == 0] = 1.0 / (8.0 * dgamma ** 2)
    return g


def filtered(y, geom):
    """Steps 2-3 for sinograms [..., B] -> Q [..., B]."""
    B = geom.n_bins
    dgamma = geom.bin_pitch_mm / geom.sdd_mm
    gam = (np.arange(B) - 0.5 * (B - 1) + geom.bin_offset) * dgamma
    rp = np.asarray(y, dtype=np.float64) * (geom.sid_mm * np.cos(gam))
    g = ramp_kernel(B, dgamma)
    q = np.zeros_like(rp)
    for n in range(B):                       # Q(n) = dgamma * sum_m R'(m) g(n - m)
        q[..., n] = dgamma * (rp * g[(n - np.arange(B)) + B - 1]).sum(axis=-1)
    return q


def fbp_init(geom, y, nx, ny):
    """y: [N][V][B] (one slice) -> f0 [N][ny][nx], all N images equal."""
    y = np.asarray(y, dtype=np.float64)
    N, V, B = y.shape
    ang = np.asarray(geom.angles_rad, dtype=np.float64)
    assert ang.shape == (N, V)
    w = view_weights(ang)
    q = filtered(y, geom)
    dgamma = geom.bin_pitch_mm / geom.sdd_mm
    X = (np.arange(nx) - 0.5 * (nx - 1)) * geom.pixel_mm
    Y = (np.arange(ny) - 0.5 * (ny - 1)) * geom.pixel_mm
    XX, YY = np.meshgrid(X, Y)               # [ny][nx]
    img = np.zeros((ny, nx), dtype=np.float64)
    for i in range(N):
        for v in range(V):
            beta = ang[i, v]
            sx, sy = geom.sid_mm * np.cos(beta), geom.sid_mm * np.sin(beta)
            px, py = XX - sx, YY - sy
            L2 = px * px + py * py
            # pixel = S - L (cos(beta+gamma), sin(beta+gamma))  =>  beta + gamma = atan2(-py, -px)
            gam = np.arctan2(-py, -px) - beta
            gam = (gam + np.pi) % (2.0 * np.pi) - np.pi
            k = gam / dgamma + 0.5 * (B - 1) - geom.bin_offset
            k0 = np.floor(k).astype(np.int64)
            fr = k - k0
            qa = np.where((k0 >= 0) & (k0 < B), q[i, v][np.clip(k0, 0, B - 1)], 0.0)
            qb = np.where((k0 + 1 >= 0) & (k0 + 1 < B), q[i, v][np.clip(k0 + 1, 0, B - 1)], 0.0)
            img += w[i, v] * ((1.0 - fr) * qa + fr * qb) / L2
    return np.broadcast_to(img, (N, ny, nx)).copy()
