"""Shared test helpers (comparison metrics only; no method arithmetic)."""
import numpy as np


def blockwise_rel_err(G, O, S=None, cfloor=1e-3):
    """Reading R14: max over blocks of ||G_b - O_b||_F / den_b.  G, O: (nblocks, ...).

    Without S: den_b = ||O_b||_F; blocks with O_b == 0 exactly are measured against max_b ||O_b||_F.
    With S (same shape; the blockwise magnitude sum, e.g. |P|^T |A| |P| for A_c): den_b =
    max(||O_b||_F, cfloor * ||S_b||_F), i.e. a block that cancels by more than 3 digits is measured against its
    cancellation-limited scale (the standard dot-product error bound is relative to S_b, not to O_b)."""
    G = np.asarray(G, dtype=np.float64).reshape(G.shape[0], -1)
    O = np.asarray(O, dtype=np.float64).reshape(O.shape[0], -1)
    if O.shape[0] == 0:
        return 0.0
    on = np.linalg.norm(O, axis=1)
    dn = np.linalg.norm(G - O, axis=1)
    if S is not None:
        sn = np.linalg.norm(np.asarray(S, dtype=np.float64).reshape(O.shape[0], -1), axis=1)
        den = np.maximum(on, cfloor * sn)
        ok = den > 0
        e = (dn[ok] / den[ok]).max() if ok.any() else 0.0
        if (~ok).any() and dn[~ok].max() > 0:
            return float("inf")
        return float(e)
    big = on.max()
    nz = on > 0
    e1 = (dn[nz] / on[nz]).max() if nz.any() else 0.0
    e0 = (dn[~nz] / big).max() if (~nz).any() and big > 0 else (dn[~nz].max() if (~nz).any() else 0.0)
    return float(max(e1, e0))


def vec_blockwise_rel_err(g, o, bs, s=None):
    return blockwise_rel_err(np.asarray(g).reshape(-1, bs), np.asarray(o).reshape(-1, bs),
                             None if s is None else np.asarray(s).reshape(-1, bs))
