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
