"""Shared helpers for the GPU-vs-oracle parity tests (tolerances from BASELINE.json north_star)."""
import json
import os

import numpy as np

SLOPE_TOL = 1e-4       # max |delta slope| in detector pixels
IMAGE_TOL = 1e-5       # relative L2 on images and PSFs, per (step, source) array
PHASE_TOL = 1e-6       # relative L2 on phase (proposed bar)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    den = np.sqrt((b * b).sum())
    return float(np.sqrt(((a - b) ** 2).sum()) / den) if den > 0 else float(np.abs(a).max())


def per_subap_max_rel_l2(got, ref, valid=None):
    """SURVEY.md section 8(c) "Parity bars": the per-subaperture maximum beside the array L2.
    got, ref: [nsa][P][P]; relative L2 of every subaperture image on its own, maximum over the valid ones
    (an invalid subaperture must be exactly zero on both sides)."""
    g = np.asarray(got, dtype=np.float64).reshape(len(got), -1)
    r = np.asarray(ref, dtype=np.float64).reshape(len(ref), -1)
    den = np.sqrt((r * r).sum(axis=1))
    num = np.sqrt(((g - r) ** 2).sum(axis=1))
    lit = den > 0 if valid is None else np.asarray(valid).astype(bool)
    assert np.all(g[~lit] == 0.0) and np.all(r[~lit] == 0.0), "invalid subapertures must give zero images"
    return float((num[lit] / den[lit]).max()) if lit.any() else 0.0


def check_wfs(cfg, geo, ref, w, images, slopes, n_steps, label="", sources=None, steps=None):
    """images [k][sel][nsa][P][P], slopes [k][sel][2][nsa] torch tensors vs oracle.forward() result.
    `sources` restricts the comparison to some global source indices (the oracle ran on a subset);
    `steps` maps the oracle's step index to the index along k of the GPU arrays (default: identity).
    Returns (worst array rel L2 of the images, worst |delta slope|, worst per-subaperture rel L2)."""
    sel = cfg.sources_of_wfs(w)
    worst_img, worst_slp, worst_sub = 0.0, 0.0, 0.0
    for si, s in enumerate(sel):
        if sources is not None and s not in sources:
            continue
        for k in range(n_steps):
            kk = k if steps is None else steps[k]
            if images is not None:
                got = images[kk, si].cpu().numpy()
                worst_img = max(worst_img, rel_l2(got, ref["images"][s][k]))
                worst_sub = max(worst_sub, per_subap_max_rel_l2(got, ref["images"][s][k], ref["valid"][w]))
            if slopes is not None:
                d = np.abs(slopes[kk, si].cpu().numpy().astype(np.float64) - ref["slopes"][s][k]).max()
                worst_slp = max(worst_slp, d)
    assert worst_img <= IMAGE_TOL, f"{label} images rel L2 {worst_img:.3e}"
    assert worst_slp <= SLOPE_TOL, f"{label} slopes max abs {worst_slp:.3e}"
    return worst_img, worst_slp, worst_sub


def report(name, **values):
    """Append one line of measured parity margins to gpurun_out/parity_report.jsonl (scratch; the numbers
    quoted in DESIGN.md come from it).  Never fails a test."""
    try:
        root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
        out = os.path.join(root, "gpurun_out")
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_report.jsonl"), "a") as f:
            f.write(json.dumps({"case": name, **{k: (float(v) if isinstance(v, (int, float, np.floating)) else v)
                                                  for k, v in values.items()}}) + "\n")
    except Exception:
        pass
