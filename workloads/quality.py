"""Image-quality figures of the paper's section 3 on the synthetic phantom (evaluation only: no
arithmetic of the reconstruction method lives here).

  SNR (Eq. 11):  10 log10( ||f - mean(f)||^2 / ||f - f*||^2 ),  f* = ground truth
  CNR (Eq. 10):  |mu_s - mu_b| / sigma_b  of a signal ROI against a nearby background ROI

The paper's ROIs (Fig. 4: a small high-contrast structure in the lung; the vertebral body) belong to
the NCAT phantom, which is not available; `tumour_rois` gives the analogue on the ellipse phantom:
signal = the tumour disc, background = the lung ring around it.
"""
import numpy as np


def snr_db(f, f_true):
    f = np.asarray(f, dtype=np.float64)
    t = np.asarray(f_true, dtype=np.float64)
    return float(10.0 * np.log10(np.sum((f - f.mean()) ** 2) / np.sum((f - t) ** 2)))


def cnr(f, signal_mask, background_mask):
    f = np.asarray(f, dtype=np.float64)
    s, b = f[signal_mask], f[background_mask]
    return float(abs(s.mean() - b.mean()) / b.std())


def tumour_rois(phantom, lung_value=0.004, tumour_value=0.02, ring=6):
    """(signal, background) masks of one phase image of the ellipse phantom: the tumour's interior pixels
    and the lung pixels within `ring` pixels of it."""
    ph = np.asarray(phantom)
    lung = np.isclose(ph, lung_value)
    body_or_tumour = np.isclose(ph, tumour_value)
    # the tumour is the tumour-valued component enclosed by lung: pixels whose 4-neighbourhood at distance
    # `ring` in every direction still is lung or tumour
    ny, nx = ph.shape
    sig = np.zeros_like(lung)
    rr, cc = np.nonzero(body_or_tumour)
    for r, c in zip(rr, cc):
        r0, r1, c0, c1 = max(r - ring, 0), min(r + ring, ny - 1), max(c - ring, 0), min(c + ring, nx - 1)
        if lung[r0, c] and lung[r1, c] and lung[r, c0] and lung[r, c1]:
            sig[r, c] = True
    if not sig.any():
        raise ValueError("no tumour found")
    r_s, c_s = np.nonzero(sig)
    box = np.zeros_like(lung)
    box[max(r_s.min() - ring, 0):r_s.max() + ring + 1, max(c_s.min() - ring, 0):c_s.max() + ring + 1] = True
    return sig, lung & box
