"""Helpers shared by the parity tests (no method arithmetic here)."""
import numpy as np


def components(valid):
    from scipy import ndimage
    lab, n = ndimage.label(valid)       # face connectivity = the stencil's links
    return lab, n


def rel_l2_after_mean_removal(P_gpu, P_or, valid):
    """|| (P_gpu - mean) - (P_or - mean) ||_2 / || P_or - mean ||_2, means per connected component of the valid set
    (A12)."""
    lab, n = components(valid)
    a = np.array(P_gpu, dtype=np.float64)
    b = np.array(P_or, dtype=np.float64)
    num = den = 0.0
    idx = lab.ravel()
    af, bf = a.ravel(), b.ravel()
    if n == 1:
        m = idx == 1
        da = af[m] - af[m].mean()
        db = bf[m] - bf[m].mean()
        return float(np.linalg.norm(da - db) / max(np.linalg.norm(db), 1e-300))
    cnt = np.bincount(idx, minlength=n + 1).astype(np.float64)
    ma = np.bincount(idx, weights=np.where(idx > 0, af, 0.0), minlength=n + 1) / np.maximum(cnt, 1)
    mb = np.bincount(idx, weights=np.where(idx > 0, bf, 0.0), minlength=n + 1) / np.maximum(cnt, 1)
    m = idx > 0
    da = af[m] - ma[idx[m]]
    db = bf[m] - mb[idx[m]]
    return float(np.linalg.norm(da - db) / max(np.linalg.norm(db), 1e-300))


def to_dev(a, dtype=None):
    import torch
    if a is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def spacing3(d):
    return (d[0], d[1], d[2] if len(d) > 2 else 1.0)
