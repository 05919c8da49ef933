"""Layout-independent list checks shared by the oracle pins and the GPU parity tests.
Pure numpy/scipy; no arithmetic of the method beyond 'distance below a radius'."""
import numpy as np
from scipy.spatial import cKDTree


def shift_id(s):
    s = np.asarray(s).astype(np.int64)
    return (s[..., 0] + 1) * 9 + (s[..., 1] + 1) * 3 + (s[..., 2] + 1)


def triple_keys(ci, cj, s):
    return (np.asarray(ci).astype(np.int64) << 36) | (np.asarray(cj).astype(np.int64) << 8) | shift_id(s)


def canonicalise(ci, cj, s, mask=None, C=8):
    """Maps (ci,cj,s) to the canonical half: s >lex 0, or s == 0 and cj >= ci; the
    equivalent triple is (cj,ci,-s) with the pair mask transposed."""
    ci, cj, s = np.asarray(ci).copy(), np.asarray(cj).copy(), np.asarray(s).astype(np.int64).copy()
    lex = np.where(s[:, 0] != 0, s[:, 0], np.where(s[:, 1] != 0, s[:, 1], s[:, 2]))
    flip = (lex < 0) | ((lex == 0) & (cj < ci))
    ci2 = np.where(flip, cj, ci)
    cj2 = np.where(flip, ci, cj)
    s2 = np.where(flip[:, None], -s, s)
    if mask is None:
        return ci2, cj2, s2
    m = np.asarray(mask, dtype=np.uint64)
    mt = np.zeros_like(m)
    for a in range(C):
        for b in range(C):
            bit = (m >> np.uint64(a * C + b)) & np.uint64(1)
            mt |= bit << np.uint64(b * C + a)
    return ci2, cj2, s2, np.where(flip, mt, m)


def close_atom_pairs(atom_of_slot, xq, box, radius, subset=None):
    """All slot pairs (si<sj, valid atoms) with fp64 minimum-image distance < radius, with the
    image vector s such that d = x_si + s L - x_sj is that minimum image.  `subset` (bool per slot)
    restricts the search to pairs with BOTH atoms in it (a spatial sample of a large box)."""
    aos = np.asarray(atom_of_slot)
    ok = aos >= 0
    if subset is not None:
        ok = ok & np.asarray(subset)
    valid = np.nonzero(ok)[0]
    box = np.asarray(box, dtype=np.float64)
    x = np.asarray(xq, dtype=np.float64).reshape(-1, 4)[valid, :3]
    xw = np.mod(x, box)
    xw = np.where(xw >= box, 0.0, xw)
    pairs = cKDTree(xw, boxsize=box).query_pairs(radius, output_type="ndarray")
    si, sj = valid[pairs[:, 0]], valid[pairs[:, 1]]
    d = x[pairs[:, 0]] - x[pairs[:, 1]]
    s = -np.rint(d / box).astype(np.int64)
    dist = np.linalg.norm(d + s * box, axis=1)
    keep = dist < radius
    return si[keep], sj[keep], s[keep], dist[keep]


def coverage_missing(atom_of_slot, xq, box, radius, ci, cj, s, C=8, subset=None):
    """Number of atom pairs closer than `radius` whose canonical cluster triple is NOT in the
    given triple set (must be 0 for a complete list), and the number of pairs checked."""
    si, sj, sp, _ = close_atom_pairs(atom_of_slot, xq, box, radius, subset)
    pci, pcj, ps = canonicalise(si // C, sj // C, sp)
    have = np.unique(triple_keys(*canonicalise(ci, cj, s)))
    need = triple_keys(pci, pcj, ps)
    return int((~np.isin(need, have)).sum()), int(need.size)


def z_slab_subset(xq, box, z0, thickness):
    """Slots whose wrapped z lies in [z0, z0 + thickness) modulo Lz (a slab; z0 + thickness > Lz makes it
    straddle the periodic face, which exercises the shifted list entries)."""
    z = np.mod(np.asarray(xq, dtype=np.float64).reshape(-1, 4)[:, 2] - z0, float(box[2]))
    return z < thickness


def half_entry_keys(ci, entry, s, kind):
    """Unique int64 key per entry of the compact half-cluster inner list (same packing as oracle.HalfListResult.keys)."""
    return ((np.asarray(ci).astype(np.int64) << 38) | (np.asarray(entry).astype(np.int64) << 9)
            | (shift_id(s) << 1) | np.asarray(kind).astype(np.int64))
