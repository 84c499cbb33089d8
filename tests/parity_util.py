"""Shared helpers for the GPU-vs-oracle parity tests (tolerances from BASELINE.json north_star)."""
import numpy as np

SLOPE_TOL = 1e-4       # max |delta slope| in detector pixels
IMAGE_TOL = 1e-5       # relative L2 on images and PSFs, per (step, source) array
PHASE_TOL = 1e-6       # relative L2 on phase (proposed bar)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    den = np.sqrt((b * b).sum())
    return float(np.sqrt(((a - b) ** 2).sum()) / den) if den > 0 else float(np.abs(a).max())


def check_wfs(cfg, geo, ref, w, images, slopes, n_steps, label=""):
    """images [k][sel][nsa][P][P], slopes [k][sel][2][nsa] torch tensors vs oracle.forward() result."""
    sel = cfg.sources_of_wfs(w)
    worst_img, worst_slp = 0.0, 0.0
    for si, s in enumerate(sel):
        for k in range(n_steps):
            if images is not None:
                e = rel_l2(images[k, si].cpu().numpy(), ref["images"][s][k])
                worst_img = max(worst_img, e)
            if slopes is not None:
                d = np.abs(slopes[k, si].cpu().numpy().astype(np.float64) - ref["slopes"][s][k]).max()
                worst_slp = max(worst_slp, d)
    assert worst_img <= IMAGE_TOL, f"{label} images rel L2 {worst_img:.3e}"
    assert worst_slp <= SLOPE_TOL, f"{label} slopes max abs {worst_slp:.3e}"
    return worst_img, worst_slp
