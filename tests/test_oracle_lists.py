"""Pins of the list oracle (oracle_lists): special cases that reduce to a library k-d tree,
hand-built shift cases, brute-force completeness, mask rules.  CPU only."""
import numpy as np
import pytest
from scipy.spatial import cKDTree

from oracle import oracle as O
from paper_2006_09167_b200 import workloads as W
from tests import listcheck as LC


def _simple_layout(w, C=8, pad_every=5):
    """A layout the test makes up (NOT the library's): atoms sorted by a coarse cell index,
    chunked into clusters of C with a few padding slots sprinkled in."""
    x = w.x.astype(np.float64)
    cell = np.floor(x / (w.box.astype(np.float64) / 3)).astype(int)
    order = np.lexsort((x[:, 2], cell[:, 2], cell[:, 1], cell[:, 0]))
    slots = []
    k = 0
    while k < len(order):
        take = C - 1 if (len(slots) // C) % pad_every == 0 else C
        chunk = list(order[k:k + take])
        k += take
        slots += chunk + [-1] * (C - len(chunk))
    aos = np.array(slots, dtype=np.int32)
    xq = np.zeros((aos.size, 4), dtype=np.float32)
    xq[aos >= 0, :3] = w.x[aos[aos >= 0]]
    xq[aos >= 0, 3] = w.q[aos[aos >= 0]]
    xq[aos < 0, :3] = 1e6  # padding coordinates must not matter
    return aos, xq


@pytest.fixture(scope="module")
def small():
    return W.small_water(60, 1.9, seed=3, rc=0.8, rlist_outer=0.9, rlist_inner=0.84,
                         box_scale=(1.0, 1.05, 1.15))


def test_cluster_size_one_reduces_to_plain_verlet_list(small):
    """With C = 1 the bounding box of a cluster is its atom, so the outer list is exactly the
    set of atom pairs within rlist -- compare with scipy's periodic k-d tree."""
    w = small
    n = w.natoms
    aos = np.arange(n, dtype=np.int32)
    xq = np.concatenate([w.x, w.q[:, None]], axis=1).astype(np.float32)
    none = (np.zeros(n + 1, np.int32), np.zeros(0, np.int32))
    r = 0.9
    res = O.lists(aos, xq, w.box, r, r, *none, cluster_size=1)
    # drop the trivial self entries (ci,ci,0) that the bb predicate always lists
    self_e = (res.ci == res.cj) & (res.s == 0).all(axis=1)
    assert self_e.sum() == n and not res.inner[self_e].any()
    got = set(zip(res.ci[~self_e].tolist(), res.cj[~self_e].tolist()))
    box = w.box.astype(np.float64)
    t = cKDTree(np.mod(w.x.astype(np.float64), box), boxsize=box)
    lo = set(map(tuple, np.sort(t.query_pairs(r - 1e-5, output_type="ndarray"), axis=1).tolist()))
    hi = set(map(tuple, np.sort(t.query_pairs(r + 1e-5, output_type="ndarray"), axis=1).tolist()))
    got_sorted = set((min(a, b), max(a, b)) for a, b in got)
    assert lo <= got_sorted <= hi and len(got_sorted) == len(got)
    # inner == outer here (same radius, one atom per cluster)
    assert res.inner[~self_e].all()
    # each listed triple's shift really is the minimum image: |x_i + sL - x_j| < r
    d = xq[res.ci, :3].astype(np.float64) + res.s * box - xq[res.cj, :3].astype(np.float64)
    assert (np.linalg.norm(d, axis=1)[~self_e] < r + 1e-5).all()


def test_shift_direction_hand_case():
    """Two one-atom clusters across the +x face: the canonical triple is (low-x atom,
    high-x atom, s=(+1,0,0)) because d = x_a + s L - x_b must be the short vector."""
    box = np.array([2.0, 2.0, 2.0], np.float32)
    xq = np.array([[0.05, 1, 1, 0], [1.95, 1, 1, 0]], np.float32)
    aos = np.array([0, 1], np.int32)
    none = (np.zeros(3, np.int32), np.zeros(0, np.int32))
    res = O.lists(aos, xq, box, 0.2, 0.2, *none, cluster_size=1)
    trip = set(zip(res.ci.tolist(), res.cj.tolist(), map(tuple, res.s.tolist())))
    assert trip == {(0, 0, (0, 0, 0)), (1, 1, (0, 0, 0)), (0, 1, (1, 0, 0))}
    # swapped storage order: now the pair is (1, 0, (+1,0,0))
    res = O.lists(aos, xq[::-1].copy(), box, 0.2, 0.2, *none, cluster_size=1)
    trip = set(zip(res.ci.tolist(), res.cj.tolist(), map(tuple, res.s.tolist())))
    assert (1, 0, (1, 0, 0)) in trip and (0, 1, (1, 0, 0)) not in trip


def test_completeness_uniqueness_and_masks(small):
    w = small
    aos, xq = _simple_layout(w)
    res = O.lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    keys = res.keys()
    assert np.unique(keys).size == keys.size  # no duplicate triples
    # canonical half only
    lex = np.where(res.s[:, 0] != 0, res.s[:, 0], np.where(res.s[:, 1] != 0, res.s[:, 1], res.s[:, 2]))
    assert ((lex > 0) | ((lex == 0) & (res.cj >= res.ci))).all()
    # every atom pair within the radius is covered (outer at rlist_outer, inner at rlist_inner)
    miss, n = LC.coverage_missing(aos, xq, w.box, w.rlist_outer - 1e-6, res.ci, res.cj, res.s)
    assert miss == 0 and n > 1000
    inn = res.inner
    miss, n = LC.coverage_missing(aos, xq, w.box, w.rlist_inner - 1e-6, res.ci[inn], res.cj[inn], res.s[inn])
    assert miss == 0
    # inner is a strict subset here, and an inner triple really has a close atom pair
    assert 0 < inn.sum() < inn.size
    si, sj, sp, dist = LC.close_atom_pairs(aos, xq, w.box, w.rlist_inner + 1e-6)
    close_keys = np.unique(LC.triple_keys(*LC.canonicalise(si // 8, sj // 8, sp)))
    assert np.isin(res.keys("inner"), close_keys).all()
    # pairmask: recompute from the topology with numpy
    mol = w.mol_of_atom
    for k in np.random.default_rng(0).choice(keys.size, size=300, replace=False):
        ci, cj, s = int(res.ci[k]), int(res.cj[k]), res.s[k]
        diag = ci == cj and not s.any()
        m = 0
        for a in range(8):
            for b in range(8):
                ia, jb = aos[ci * 8 + a], aos[cj * 8 + b]
                if ia < 0 or jb < 0 or (diag and b <= a) or ia == jb or mol[ia] == mol[jb]:
                    continue
                m |= 1 << (a * 8 + b)
        assert int(res.pairmask[k]) == m
    # a diagonal triple is listed for every non-empty cluster
    ncl = aos.size // 8
    diag_listed = set(res.ci[(res.ci == res.cj) & (res.s == 0).all(axis=1)].tolist())
    assert diag_listed == set(range(ncl))


def test_sub_range_enumeration_matches_full(small):
    w = small
    aos, xq = _simple_layout(w)
    full = O.lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    part = O.lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx, c_begin=3, c_end=6)
    sel = ((full.ci >= 3) & (full.ci < 6)) | ((full.cj >= 3) & (full.cj < 6))
    assert np.array_equal(np.sort(full.keys()[sel]), np.sort(part.keys()))


def test_canonicalise_roundtrip():
    ci = np.array([5, 2, 7]); cj = np.array([2, 5, 7]); s = np.array([[0, 0, 0], [-1, 0, 1], [0, 0, 0]])
    m = np.array([1 << (1 * 8 + 2), 1 << (3 * 8 + 4), 5], dtype=np.uint64)
    a, b, t, mt = LC.canonicalise(ci, cj, s, m)
    assert a.tolist() == [2, 5, 7] and b.tolist() == [5, 2, 7]
    assert t.tolist() == [[0, 0, 0], [1, 0, -1], [0, 0, 0]]
    assert mt.tolist() == [1 << (2 * 8 + 1), 1 << (4 * 8 + 3), 5]


# ---------------------------------------------------------------- fp32 recomputation in numpy (reading A12)
def _fma32(a, b, c):
    """fmaf for float32 arrays: the product of two float32 is exact in float64; the sum is rounded to
    float64 and then to float32 (a double rounding could differ from fmaf only when the float64 sum
    lands exactly on a float32 midpoint, ~1e-9 per operation; inputs are seeded, so deterministic)."""
    return (a.astype(np.float64) * b.astype(np.float64) + c.astype(np.float64)).astype(np.float32)


def _cluster_bbs(aos, xq, C=8):
    x = np.where((aos >= 0)[:, None], xq[:, :3], np.nan).reshape(-1, C, 3)
    with np.errstate(all="ignore"):
        return np.nanmin(x, axis=1).astype(np.float32), np.nanmax(x, axis=1).astype(np.float32)


def _all_canonical_triples(ncl):
    ci, cj, sx, sy, sz = np.meshgrid(np.arange(ncl), np.arange(ncl), *[np.arange(-1, 2)] * 3, indexing="ij")
    ci, cj = ci.ravel(), cj.ravel()
    s = np.stack([sx.ravel(), sy.ravel(), sz.ravel()], axis=1)
    lex = np.where(s[:, 0] != 0, s[:, 0], np.where(s[:, 1] != 0, s[:, 1], s[:, 2]))
    keep = (lex > 0) | ((lex == 0) & (cj >= ci))
    return ci[keep], cj[keep], s[keep]


def _bb_dist2_np(lo, hi, ci, cj, s, box):
    sL = (s.astype(np.float32) * box[None, :].astype(np.float32))          # exact: s in {-1,0,1}
    a = (sL + lo[ci]).astype(np.float32) - hi[cj]                            # fmaf(s,L,lo_i) - hi_j
    b = lo[cj] - (sL + hi[ci]).astype(np.float32)                            # lo_j - fmaf(s,L,hi_i)
    g = np.maximum(np.maximum(a, b), np.float32(0)).astype(np.float32)
    return _fma32(g[:, 2], g[:, 2], _fma32(g[:, 1], g[:, 1], (g[:, 0] * g[:, 0]).astype(np.float32)))


def _atom_d2_np(xq, slots_i, slots_j, s, box):
    """[n, len(slots_i[0]), len(slots_j[0])] float32 distances d = x_a + s L - x_b in the A12 order."""
    sL = (s.astype(np.float32) * box[None, :].astype(np.float32))
    xi = (xq[slots_i, :3] + sL[:, None, :]).astype(np.float32)               # fmaf(s, L, x_a): s L exact
    d = (xi[:, :, None, :] - xq[slots_j, :3][:, None, :, :]).astype(np.float32)
    return _fma32(d[..., 2], d[..., 2], _fma32(d[..., 1], d[..., 1], (d[..., 0] * d[..., 0]).astype(np.float32)))


def test_bb_predicate_is_exact_both_ways(small):
    """Pin against OVER-listing as well as under-listing at C = 8: over ALL canonical (ci, cj, s) of a
    test-made layout, listed <=> D2_bb < fl32(r^2) with D2_bb recomputed in numpy float32.  A lo/hi mix-up,
    a shift on the wrong side or a wrong sign in the gap changes the listed set."""
    w = small
    aos, xq = _simple_layout(w)
    res = O.lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    lo, hi = _cluster_bbs(aos, xq)
    ncl = aos.size // 8
    ci, cj, s = _all_canonical_triples(ncl)
    d2 = _bb_dist2_np(lo, hi, ci, cj, s, w.box)
    r2 = np.float32(w.rlist_outer) * np.float32(w.rlist_outer)
    want = d2 < r2
    listed = np.isin(LC.triple_keys(ci, cj, s), res.keys())
    assert want.sum() > 500 and (~want).sum() > 500
    assert np.array_equal(listed, want)
    # the band around the threshold is populated on both sides: the comparison really is decided there
    near = np.abs(np.sqrt(d2.astype(np.float64)) - w.rlist_outer) < 0.05
    assert (want & near).sum() > 20 and (~want & near).sum() > 20


def test_half_lists_against_numpy(small):
    """oracle_half_lists recomputed in numpy float32 on a test-made layout: whole masked cluster pairs and
    surviving halves of the unmasked ones, bit-exact as sets; halves are consistent with the inner flag
    of oracle_lists; every atom pair within rlist_inner is covered; every listed half has a close pair."""
    w = small
    aos, xq = _simple_layout(w)
    res = O.lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    hl = O.half_lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    assert np.unique(hl.keys()).size == hl.keys().size
    valid = (aos >= 0).reshape(-1, 8)
    full = np.zeros(res.ci.size, dtype=np.uint64)
    for a in range(8):
        for b in range(8):
            full |= (valid[res.ci, a] & valid[res.cj, b]).astype(np.uint64) << np.uint64(a * 8 + b)
    masked = res.pairmask != full
    diag = (res.ci == res.cj) & (res.s == 0).all(axis=1)
    assert masked[diag].all() and masked.sum() > diag.sum()           # water: intramolecular exclusions too
    ri2 = np.float32(w.rlist_inner) * np.float32(w.rlist_inner)
    si = res.ci[:, None] * 8 + np.arange(8)[None, :]
    sj = res.cj[:, None] * 8 + np.arange(8)[None, :]
    d2 = _atom_d2_np(xq, si, sj, res.s.astype(np.int64), w.box)       # [n, 8, 8]
    ok = valid[res.ci][:, :, None] & valid[res.cj][:, None, :]
    close = (d2 < ri2) & ok
    upper = np.triu(np.ones((8, 8), bool), 1)                          # diagonal cluster pair: b > a only
    close_m = np.where(diag[:, None, None], close & upper[None], close)
    want = set()
    sid = LC.shift_id(res.s)
    for k in range(res.ci.size):
        if masked[k]:
            if close_m[k].any():
                want.add((int(res.ci[k]), int(res.cj[k]), int(sid[k]), 1))
        else:
            for h in range(2):
                if close[k][:, 4 * h:4 * h + 4].any():
                    want.add((int(res.ci[k]), 2 * int(res.cj[k]) + h, int(sid[k]), 0))
    got = set(zip(hl.ci.tolist(), hl.entry.tolist(), LC.shift_id(hl.s).tolist(), hl.kind.tolist()))
    assert got == want and sum(1 for g in got if g[3] == 0) > 300 and sum(1 for g in got if g[3] == 1) > 20
    # consistency with oracle_lists: the cluster pairs spanned by the entries are exactly the inner triples
    spanned = {(c, e // 2 if kd == 0 else e, k) for c, e, k, kd in got}
    inner = set(zip(res.ci[res.inner].tolist(), res.cj[res.inner].tolist(), sid[res.inner].tolist()))
    assert spanned == inner
    # strictly finer than whole clusters: some surviving unmasked cluster pairs keep one half only
    unm = [(c, e // 2, k) for c, e, k, kd in got if kd == 0]
    assert len(unm) > len(set(unm)) > 0.55 * len(unm)
    # completeness in fp64, layout-independent (k-d tree): every atom pair closer than rlist_inner is covered
    pi, pj, sp, _ = LC.close_atom_pairs(aos, xq, w.box, w.rlist_inner - 1e-6)
    ka, kb = LC.shift_id(sp), LC.shift_id(-sp)
    miss = 0
    for a, b, k1, k2 in zip(pi.tolist(), pj.tolist(), ka.tolist(), kb.tolist()):
        if not ((a // 8, b // 4, k1, 0) in got or (b // 8, a // 4, k2, 0) in got
                or (a // 8, b // 8, k1, 1) in got or (b // 8, a // 8, k2, 1) in got):
            miss += 1
    assert miss == 0 and pi.size > 1000
    # sub-range enumeration = selection of the full one
    part = O.half_lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx, c_begin=3, c_end=6)
    cj_full = np.where(hl.kind == 0, hl.entry // 2, hl.entry)
    sel = ((hl.ci >= 3) & (hl.ci < 6)) | ((cj_full >= 3) & (cj_full < 6))
    assert np.array_equal(np.sort(hl.keys()[sel]), np.sort(part.keys()))


def test_atom_lists_against_numpy(small):
    """oracle_atom_lists (reading A22, single-j-atom granularity) recomputed in numpy float32 on a test-made layout:
    whole masked cluster pairs, and of the unmasked ones exactly the real j atoms that have a real i atom of the cluster
    within fl32(rlist_inner^2), bit-exact as sets; consistent with oracle_lists (spanned cluster pairs = inner triples)
    and with oracle_half_lists (a half is listed iff one of its atoms is); every atom pair within rlist_inner is covered
    (k-d tree, fp64); no padding slot is ever listed; a sub-range is a selection of the full enumeration."""
    w = small
    aos, xq = _simple_layout(w)
    res = O.lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    hl = O.half_lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    al = O.atom_lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx)
    assert np.unique(al.keys()).size == al.keys().size
    valid = (aos >= 0).reshape(-1, 8)
    full = np.zeros(res.ci.size, dtype=np.uint64)
    for a in range(8):
        for b in range(8):
            full |= (valid[res.ci, a] & valid[res.cj, b]).astype(np.uint64) << np.uint64(a * 8 + b)
    masked = res.pairmask != full
    diag = (res.ci == res.cj) & (res.s == 0).all(axis=1)
    ri2 = np.float32(w.rlist_inner) * np.float32(w.rlist_inner)
    si = res.ci[:, None] * 8 + np.arange(8)[None, :]
    sj = res.cj[:, None] * 8 + np.arange(8)[None, :]
    d2 = _atom_d2_np(xq, si, sj, res.s.astype(np.int64), w.box)       # [n, 8 (i atom), 8 (j atom)]
    ok = valid[res.ci][:, :, None] & valid[res.cj][:, None, :]
    close = (d2 < ri2) & ok
    upper = np.triu(np.ones((8, 8), bool), 1)
    close_m = np.where(diag[:, None, None], close & upper[None], close)
    sid = LC.shift_id(res.s)
    want = set()
    for k in range(res.ci.size):
        if masked[k]:
            if close_m[k].any():
                want.add((int(res.ci[k]), int(res.cj[k]), int(sid[k]), 1))
        else:
            for b in np.nonzero(close[k].any(axis=0))[0]:
                want.add((int(res.ci[k]), 8 * int(res.cj[k]) + int(b), int(sid[k]), 0))
    got = set(zip(al.ci.tolist(), al.entry.tolist(), LC.shift_id(al.s).tolist(), al.kind.tolist()))
    assert got == want and sum(1 for g in got if g[3] == 0) > 1000
    assert all(aos[e] >= 0 for _, e, _, kd in got if kd == 0)          # padding slots are never listed
    # the cluster pairs spanned by the entries are exactly the inner triples of oracle_lists
    spanned = {(c, e // 8 if kd == 0 else e, k) for c, e, k, kd in got}
    inner = set(zip(res.ci[res.inner].tolist(), res.cj[res.inner].tolist(), sid[res.inner].tolist()))
    assert spanned == inner
    # a half j-cluster is listed iff one of its atoms is; masked entries are the same
    half = set(zip(hl.ci.tolist(), hl.entry.tolist(), LC.shift_id(hl.s).tolist(), hl.kind.tolist()))
    assert {(c, e // 4, k, 0) for c, e, k, kd in got if kd == 0} == {h for h in half if h[3] == 0}
    assert {g for g in got if g[3] == 1} == {h for h in half if h[3] == 1}
    # strictly finer than halves: fewer atom entries than 4 per listed half
    n_atoms, n_halves = sum(1 for g in got if g[3] == 0), sum(1 for h in half if h[3] == 0)
    assert 0.5 * 4 * n_halves < n_atoms < 0.95 * 4 * n_halves
    # completeness in fp64, layout-independent (k-d tree): every atom pair closer than rlist_inner is covered, from either side
    pi, pj, sp, _ = LC.close_atom_pairs(aos, xq, w.box, w.rlist_inner - 1e-6)
    ka, kb = LC.shift_id(sp), LC.shift_id(-sp)
    miss = 0
    for a, b, k1, k2 in zip(pi.tolist(), pj.tolist(), ka.tolist(), kb.tolist()):
        if not ((a // 8, b, k1, 0) in got or (b // 8, a, k2, 0) in got
                or (a // 8, b // 8, k1, 1) in got or (b // 8, a // 8, k2, 1) in got):
            miss += 1
    assert miss == 0 and pi.size > 1000
    part = O.atom_lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx, c_begin=3, c_end=6)
    cj_full = np.where(al.kind == 0, al.entry // 8, al.entry)
    sel = ((al.ci >= 3) & (al.ci < 6)) | ((cj_full >= 3) & (cj_full < 6))
    assert np.array_equal(np.sort(al.keys()[sel]), np.sort(part.keys()))
