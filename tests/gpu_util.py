"""Helpers shared by the -m gpu parity tests (comparison norms of DESIGN.md 'Tolerances')."""
import numpy as np


def sort_pairs(p):
    p = np.asarray(p, dtype=np.uint32).reshape(-1, 2)
    key = (p[:, 0].astype(np.uint64) << np.uint64(32)) | p[:, 1].astype(np.uint64)
    return p[np.argsort(key, kind="stable")]


def force_rel_err(F, Fref):
    """R11: err_i = |F_i - Fref_i|_inf / max(|Fref_i|_inf, 1e-3 F_rms); returns max_i err_i."""
    F = np.asarray(F); Fref = np.asarray(Fref)
    frms = np.sqrt(np.mean(np.sum(Fref * Fref, axis=1)))
    den = np.maximum(np.abs(Fref).max(axis=1), 1e-3 * frms)
    den = np.where(den > 0, den, 1.0)
    return float((np.abs(F - Fref).max(axis=1) / den).max())


def min_image_diff(a, b, box):
    d = np.asarray(a) - np.asarray(b)
    return d - box * np.rint(d / box)
