"""GPU parity tests (run on the B200 box with -m gpu): the CUDA path, driven through the C ABI,
against the fp64 oracle on the same seeded inputs.  Tolerances are BASELINE.json's: lists and
masks bit-exact as sets, relative RMS force error <= 1e-5, relative energy error <= 1e-5;
virial: same bound on the Frobenius norm."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2006_09167_b200 import workloads as W
from tests import listcheck as LC
from tests.gpu_util import Driver, oracle_forces, rel_rms

pytestmark = pytest.mark.gpu

TOL_F = 1e-5
TOL_E = 1e-5


@pytest.fixture(scope="module")
def small_rect():
    # rectangular box, two super-cluster columns per axis at most, rc close to L/2 in x
    return W.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84, box_scale=(1.0, 1.1, 1.25))


def check_layout(d, w):
    lay = d.ctx.get_layout()
    aos, xq = d.slots()
    assert lay["cluster_size"] == 8 and lay["nslots"] == lay["nsuper"] * 64 == lay["nclusters"] * 8 == aos.size
    real = aos[aos >= 0]
    assert real.size == w.natoms and np.array_equal(np.sort(real), np.arange(w.natoms))   # T13: each atom once
    # slot coordinates are the atom's coordinates up to whole box vectors; charges match
    dx = xq[aos >= 0, :3].astype(np.float64) - w.x[real].astype(np.float64)
    k = np.rint(dx / w.box)
    assert np.abs(dx - k * w.box).max() < 2e-6
    assert np.array_equal(xq[aos >= 0, 3], w.q[real])
    # wrapped into the box (up to rounding)
    assert (xq[aos >= 0, :3] > -1e-5).all() and (xq[aos >= 0, :3] < w.box + 1e-5).all()
    # within a cluster real atoms come first; within a super-cluster partly-filled clusters come last
    v = (aos >= 0).reshape(-1, 8)
    assert (np.diff(v.astype(int), axis=1) <= 0).all()
    cnt = v.sum(axis=1).reshape(-1, 8)
    assert (np.diff(cnt, axis=1) <= 0).all()
    # padding is small: fewer than 64 slots per grid column
    st = d.ctx.get_stats()
    assert (aos < 0).sum() < 64 * st["ncolumns_x"] * st["ncolumns_y"]
    # super-clusters of a column are z-ordered slabs: find columns by xy cell and compare z ranges
    z = np.where(aos >= 0, xq[:, 2], np.nan).reshape(-1, 64)
    zmin, zmax = np.nanmin(z, axis=1), np.nanmax(z, axis=1)
    same_col_next = cnt.sum(axis=1)[:-1] == 64   # a full slab is followed by a slab of the same column or a new column
    cx = np.floor(np.nanmean(np.where(aos >= 0, xq[:, 0], np.nan).reshape(-1, 64), axis=1) * st["ncolumns_x"] / w.box[0])
    cy = np.floor(np.nanmean(np.where(aos >= 0, xq[:, 1], np.nan).reshape(-1, 64), axis=1) * st["ncolumns_y"] / w.box[1])
    samecol = (cx[1:] == cx[:-1]) & (cy[1:] == cy[:-1]) & same_col_next
    assert (zmax[:-1][samecol] <= zmin[1:][samecol]).all()
    return aos, xq


def check_lists(d, w, rl_outer, rl_inner, c_range=None):
    aos, xq = d.slots()
    kw = {} if c_range is None else dict(c_begin=c_range[0], c_end=c_range[1])
    ref = O.lists(aos, xq, w.box, rl_outer, rl_inner, w.excl_off, w.excl_idx, **kw)

    def sel(ci, cj):
        if c_range is None:
            return np.ones(ci.shape, bool)
        return ((ci >= c_range[0]) & (ci < c_range[1])) | ((cj >= c_range[0]) & (cj < c_range[1]))

    for which, rkeys in ((0, ref.keys("outer")), (1, ref.keys("inner"))):
        ci, cj, s, pm, part = d.dump(which)
        assert ci.size == d.ctx.list_count(which)
        ci2, cj2, s2, pm2 = LC.canonicalise(ci, cj, s, pm)
        assert np.array_equal(ci2, ci) and np.array_equal(cj2, cj)   # the library stores the canonical half
        keys = LC.triple_keys(ci2, cj2, s2)
        assert np.unique(keys).size == keys.size, "duplicate cluster pair in the list"
        m = sel(ci2, cj2)
        got = np.sort(keys[m])
        want = np.sort(rkeys)
        assert got.size == want.size and np.array_equal(got, want), (which, got.size, want.size)
        # pair masks, bit-exact
        order_g = np.argsort(keys[m])
        rk = ref.keys("outer") if which == 0 else ref.keys("inner")
        rmask = ref.pairmask if which == 0 else ref.pairmask[ref.inner]
        order_r = np.argsort(rk)
        assert np.array_equal(pm2[m][order_g], rmask[order_r])
    return ref


def test_config0_layout_lists_forces(cfg0):
    w = cfg0
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    check_layout(d, w)
    # before any prune the inner list is the outer list
    assert d.ctx.list_count(0) == d.ctx.list_count(1)
    f_outer = d.forces()
    d.ctx.prune(w.rlist_inner)
    ref_l = check_lists(d, w, w.rlist_outer, w.rlist_inner)
    aos, xq = d.slots()
    # layout-independent completeness: every atom pair within rlist_inner is in a listed inner pair
    ci, cj, s, _, _ = d.dump(1)
    miss, n = LC.coverage_missing(aos, xq, w.box, w.rlist_inner - 1e-6, ci, cj, s)
    assert miss == 0 and n > 50000
    assert 0.4 < ref_l.inner.mean() < 0.95
    ref = oracle_forces(w)
    f = d.forces()
    assert rel_rms(f, ref.f) <= TOL_F
    assert rel_rms(f_outer, ref.f) <= TOL_F           # T10: pruning does not change the forces
    assert rel_rms(f, f_outer) < 2e-6
    frms = np.sqrt((ref.f**2).sum(1).mean())
    assert np.linalg.norm(f.sum(0)) / (w.natoms * frms) < 1e-6   # T6 on the GPU
    f2, e, vir = d.forces(energy=True, virial=True)
    assert rel_rms(f2, ref.f) <= TOL_F
    assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    assert abs(e[0] - ref.e_lj) <= TOL_E * abs(ref.energy) and abs(e[1] - ref.e_coul) <= TOL_E * abs(ref.energy)
    assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    # image brute force agrees too (T5 through the GPU)
    img = oracle_forces(w, method="images")
    assert rel_rms(f, img.f) <= TOL_F
    st = d.ctx.get_stats()
    assert st["n_pairs_inner"] == ref_l.inner.sum() and st["n_pairs_outer"] == ref_l.inner.size
    assert st["slots_last_forces"] == 64 * st["n_pairs_inner"]
    # mean number of set interaction-mask bits per joint entry: the paper's "approximately four of eight" (L135)
    assert 2.5 < st["n_pairs_outer"] / st["n_joint_outer"] < 6.5


@pytest.mark.parametrize("coulomb", ["ewald", "rf"])
def test_small_rectangular_box(coulomb):
    w = W.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84,
                      box_scale=(1.0, 1.1, 1.25), coulomb=coulomb)
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    check_layout(d, w)
    d.ctx.prune(w.rlist_inner)
    check_lists(d, w, w.rlist_outer, w.rlist_inner)
    ref = oracle_forces(w)
    f, e, vir = d.forces(energy=True, virial=True)
    assert rel_rms(f, ref.f) <= TOL_F
    assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    assert rel_rms(d.forces(), ref.f) <= TOL_F


def test_lj_only_flavour():
    """LJ-only kernel flavour on the Fig. 6 stand-in (no charges, no exclusions) and on
    a water box whose charges must be ignored; lists bit-exact, forces / energy / virial vs the oracle."""
    w = W.lj_fluid(12, rc=0.9)
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    check_layout(d, w)
    d.ctx.prune(w.rlist_inner)
    check_lists(d, w, w.rlist_outer, w.rlist_inner)
    ref = oracle_forces(w)
    f, e, vir = d.forces(energy=True, virial=True)
    assert rel_rms(f, ref.f) <= TOL_F
    assert e[1] == 0.0 and abs(e[0] - ref.e_lj) / abs(ref.e_lj) <= TOL_E
    assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    assert rel_rms(d.forces(), ref.f) <= TOL_F
    ww = W.small_water(150, 2.0, seed=23, rc=0.8, rlist_outer=0.9, rlist_inner=0.84, coulomb="none")
    d = Driver(ww)
    d.put()
    d.ctx.search(ww.rlist_outer)
    d.ctx.prune(ww.rlist_inner)
    ref = oracle_forces(ww)
    f, e = d.forces(energy=True)
    assert rel_rms(f, ref.f) <= TOL_F
    assert e[1] == 0.0 and abs(e[0] - ref.e_lj) / abs(ref.e_lj) <= TOL_E


def test_modifiers_none_and_finite_eps_rf(small_rect):
    w = small_rect
    from paper_2006_09167_b200 import nb
    d = Driver(w, lj_modifier=nb.NB_MOD_NONE, coul_modifier=nb.NB_MOD_NONE)
    d.put()
    d.ctx.search(w.rlist_outer)
    ref = oracle_forces(w, lj_shift=False, coul_shift=False)
    f, e = d.forces(energy=True)
    assert rel_rms(f, ref.f) <= TOL_F and abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    d2 = Driver(w, coulomb="rf", eps_rf=78.0)
    d2.put()
    d2.ctx.search(w.rlist_outer)
    p = O.Params(rc=w.rc, ntypes=w.ntypes, coulomb="rf", eps_rf=78.0)
    ref2 = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p)
    f, e = d2.forces(energy=True)
    assert rel_rms(f, ref2.f) <= TOL_F and abs(e.sum() - ref2.energy) / abs(ref2.energy) <= TOL_E


def test_exclusion_extremes(small_rect):
    """T15 on the GPU: no exclusions, and a topology where everything within a molecule-sized
    group of 24 atoms is excluded (dense masks)."""
    w = small_rect
    n = w.natoms
    import copy
    w0 = copy.copy(w)
    w0.excl_off, w0.excl_idx = np.zeros(n + 1, np.int32), np.zeros(0, np.int32)
    d = Driver(w0)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_outer)
    check_lists(d, w0, w.rlist_outer, w.rlist_outer)
    ref = oracle_forces(w0)
    f, e = d.forces(energy=True)
    assert rel_rms(f, ref.f) <= TOL_F and abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    grp = np.arange(n) // 24
    idx = [np.setdiff1d(np.nonzero(grp == grp[i])[0], [i]) for i in range(n)]
    w1 = copy.copy(w)
    w1.excl_off = np.concatenate([[0], np.cumsum([len(v) for v in idx])]).astype(np.int32)
    w1.excl_idx = np.concatenate(idx).astype(np.int32)
    d = Driver(w1)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_outer)
    check_lists(d, w1, w.rlist_outer, w.rlist_outer)
    ref = oracle_forces(w1)
    f, e = d.forces(energy=True)
    assert rel_rms(f, ref.f) <= TOL_F and abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E


def test_translation_and_broken_molecules(cfg0):
    """T7 on the GPU: whole-box translation and per-atom box-vector shifts leave f, E unchanged."""
    w = cfg0
    ref = oracle_forces(w)
    rng = np.random.default_rng(9)
    xs = [np.mod(w.x.astype(np.float64) + rng.uniform(-3, 3, 3), w.box).astype(np.float32),
          (w.x + rng.integers(-2, 3, size=w.x.shape) * w.box).astype(np.float32)]
    for x in xs:
        d = Driver(w)
        d.put(x)
        d.ctx.search(w.rlist_outer)
        f, e = d.forces(energy=True)
        r = oracle_forces(w, x=x)
        assert rel_rms(f, r.f) <= TOL_F
        assert abs(e.sum() - ref.energy) / abs(ref.energy) <= 2 * TOL_E


def test_config1_parity_and_rolling_prune(cfg1):
    w = cfg1
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    check_layout(d, w)
    ref = oracle_forces(w, method="cells")
    # full-size list parity on a sample of clusters (the oracle's all-pairs bb loop is O(n^2))
    ncl = d.ctx.get_layout()["nclusters"]
    d.ctx.prune(w.rlist_inner)
    for c0 in (0, ncl // 2 + 3, ncl - 24):
        check_lists(d, w, w.rlist_outer, w.rlist_inner, c_range=(c0, c0 + 24))
    f, e, vir = d.forces(energy=True, virial=True)
    assert rel_rms(f, ref.f) <= TOL_F
    assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    st = d.ctx.get_stats()
    assert 3.5 < st["n_pairs_outer"] / st["n_joint_outer"] < 5.5      # P:L135 "approximately four of eight"
    inner_full = st["n_pairs_inner"]
    assert 0.5 < inner_full / st["n_pairs_outer"] < 0.8
    # T11: pruning the k parts one after the other at fixed x == one full prune
    full = d.dump(1)
    d.ctx.search(w.rlist_outer)
    for p in range(w.nparts):
        d.ctx.prune(w.rlist_inner, p, w.nparts)
    rolled = d.dump(1)
    for a, b in zip(full[:4], rolled[:4]):
        assert np.array_equal(a, b)
    assert set(np.unique(rolled[4]).tolist()) == set(range(w.nparts))
    # rolling over moving atoms (motion recipe): forces stay equal to the all-pairs oracle
    for t in (1, 2, 50, 99):
        x = w.positions_at(t)
        d.put(x)
        before = d.dump(1)
        part = t % w.nparts
        d.ctx.prune(w.rlist_inner, part, w.nparts)
        after = d.dump(1)
        # only entries of the pruned part may change
        kb = LC.triple_keys(before[0], before[1], before[2])[before[4] != part]
        ka = LC.triple_keys(after[0], after[1], after[2])[after[4] != part]
        assert np.array_equal(kb, ka)
        r = oracle_forces(w, x=x, method="cells")
        assert rel_rms(d.forces(), r.f) <= TOL_F
    # determinism (T16): same inputs, same dump
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner)
    again = d.dump(1)
    for a, b in zip(full[:4], again[:4]):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("which", ["cfg2_ewald", "cfg2_rf", "cfg4", "cfg3"])
def test_full_size_configs_in_bench_schedule(which):
    """BASELINE.json configs[2] (both Coulomb flavours), [4] and [3] at full size, driven the way bench.py
    drives them (search, full prune, then rolling parts on the motion recipe): list parity on sampled
    cluster ranges (the list oracle is O(n^2)), forces / energy / virial against the fp64 linked-cell
    oracle (pinned equal to all-pairs), effective pair count against the oracle's."""
    w = {"cfg2_ewald": lambda: W.config2("ewald"), "cfg2_rf": lambda: W.config2("rf"), "cfg4": W.config4,
         "cfg3": W.config3}[which]()
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    check_layout(d, w)
    d.ctx.prune(w.rlist_inner)
    ncl = d.ctx.get_layout()["nclusters"]
    for c0 in (0, ncl // 3 + 5, ncl - 16):
        check_lists(d, w, w.rlist_outer, w.rlist_inner, c_range=(c0, c0 + 16))
    ref = oracle_forces(w, method="cells")
    f, e, vir = d.forces(energy=True, virial=True)
    assert rel_rms(f, ref.f) <= TOL_F
    assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    npairs, _ = d.ctx.count_pairs()
    assert abs(npairs - ref.npairs) <= 2 + 1e-6 * ref.npairs     # fp32 vs fp64 at r = rc
    fsum = np.abs(f.sum(axis=0)).max() / (np.sqrt((f**2).mean()) * w.natoms)
    assert fsum < 1e-6                                           # T6 on the GPU
    for t in (1, 2, w.nparts + 1):
        x = w.positions_at(t)
        d.put(x)
        d.ctx.prune(w.rlist_inner, t % w.nparts, w.nparts)
        r = oracle_forces(w, x=x, method="cells")
        assert rel_rms(d.forces(), r.f) <= TOL_F


@pytest.mark.parametrize("which", ["cfg0", "rect_rf", "lj"])
def test_half_cluster_inner_list(which):
    """The compact inner list the force kernel streams is kept at half-j-cluster granularity (DESIGN.md
    section 5).  Layout-independent check in fp64 on the library's own slot table, with a 1e-6 nm guard band
    around rlist_inner (the kernel decides in fp32): COMPLETE -- every atom pair closer than rlist_inner
    is covered by a listed half-cluster of the other atom's cluster or by a masked cluster pair -- and
    MINIMAL -- every listed half has an atom within rlist_inner of the i-cluster; the cluster pairs it
    spans are exactly the inner list of nb_list_dump."""
    w = {"cfg0": W.config0, "lj": lambda: W.lj_fluid(12, rc=0.9),
         "rect_rf": lambda: W.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84,
                                          box_scale=(1.0, 1.1, 1.25), coulomb="rf")}[which]()
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    for x, part, nparts in ((None, 0, 1), (w.positions_at(40), 0, 2), (w.positions_at(40), 1, 2)):
        d.put(x)
        d.ctx.prune(w.rlist_inner, part, nparts)
    aos, xq = d.slots()
    box = np.asarray(w.box, dtype=np.float64)
    ci, ent, sid, kind = d.ctx.inner_dump()
    svec = d.nb.shift_vectors(sid).astype(np.int64)
    half = kind == 0
    skey = LC.shift_id(svec)
    hkeys = set(zip(ci[half].tolist(), ent[half].tolist(), skey[half].tolist()))
    mkeys = set(zip(ci[~half].tolist(), ent[~half].tolist(), skey[~half].tolist()))
    assert len(hkeys) == int(half.sum()) and len(mkeys) == int((~half).sum())      # no duplicates
    # complete
    si, sj, sp, _ = LC.close_atom_pairs(aos, xq, box, w.rlist_inner - 1e-6)
    ka, kb = LC.shift_id(sp), LC.shift_id(-sp)
    missing = 0
    for a, b, k1, k2 in zip(si.tolist(), sj.tolist(), ka.tolist(), kb.tolist()):
        if ((a // 8, b // 4, k1) in hkeys or (b // 8, a // 4, k2) in hkeys or (a // 8, b // 8, k1) in mkeys
                or (b // 8, a // 8, k2) in mkeys):
            continue
        missing += 1
    assert missing == 0 and si.size > 1000
    # minimal: every listed half has a real atom within rlist_inner (+ guard) of a real atom of ci
    x = np.asarray(xq, dtype=np.float64).reshape(-1, 4)[:, :3]
    real = np.asarray(aos) >= 0
    hci, hent, hs = ci[half], ent[half], svec[half]
    xi = x[hci[:, None] * 8 + np.arange(8)[None, :]] + (hs * box)[:, None, :]           # [n,8,3], shift on the i side
    xj = x[hent[:, None] * 4 + np.arange(4)[None, :]]                                   # [n,4,3]
    d2 = ((xi[:, :, None, :] - xj[:, None, :, :]) ** 2).sum(-1)
    ok = real[hci[:, None] * 8 + np.arange(8)[None, :]][:, :, None] & real[hent[:, None] * 4 + np.arange(4)[None, :]][:, None, :]
    dmin = np.sqrt(np.where(ok, d2, np.inf).min(axis=(1, 2)))
    assert (dmin < w.rlist_inner + 1e-6).all()
    # same cluster pairs as the bit-plane inner list
    dci, dcj, dsv, _, _ = d.dump(1)
    planes = set(zip(dci.tolist(), dcj.tolist(), LC.shift_id(dsv).tolist()))
    spanned = {(a, e // 2, k) for a, e, k in hkeys} | mkeys
    assert spanned == planes


def test_work_efficiency_table_against_oracle():
    """SURVEY 8.1 (f3), Fig. 5 definition: the table's numerator is the oracle's count of atom pairs
    within rc (interacting + excluded), its denominator 64 x the listed cluster pairs; the efficiency falls
    with the buffer, the pruned list is at least as efficient as the searched one, and both stay below 1x1."""
    from paper_2006_09167_b200 import work_efficiency as WE
    tab = WE.efficiency_table(10, [0.8, 1.0], [0.0, 0.1, 0.2])
    w = W.water_box(10)
    for rc in (0.8, 1.0):
        rows = [r for r in tab["rows"] if r["rc"] == rc]
        assert len(rows) == 3
        ref = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx,
                       O.Params(rc=rc, ntypes=w.ntypes, coulomb="ewald", beta=O.beta_from_rtol(rc, 1e-5)))
        for r in rows:
            assert abs(r["pairs_within_rc"] - (ref.npairs + ref.npairs_excl)) <= 2
            assert r["cluster_pairs_pruned"] <= r["cluster_pairs_searched"]
            assert r["eff_searched"] <= r["eff_pruned"] < r["eff_1x1_ideal"] <= 1.0
        effs = [r["eff_searched"] for r in rows]
        assert effs[0] > effs[1] > effs[2]


@pytest.mark.parametrize("n", [1, 2, 7, 9, 65])
def test_tiny_and_ragged_systems(n):
    """Degenerate sizes: one atom (no pair at all), two atoms (one cluster, diagonal pair only), fewer atoms
    than a cluster, one more than a cluster, one more than a super-cluster; sparse box, most slots padding."""
    rng = np.random.default_rng(100 + n)
    L = 2.8
    # n ADJACENT sites of a jittered 0.35 nm lattice (a compact droplet in an otherwise empty box): nearest
    # neighbours at liquid-like distances, so the relative force tolerance is meaningful
    g = np.stack(np.meshgrid(*[np.arange(8)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)
    order = np.argsort(((g - 3.5) ** 2).sum(axis=1), kind="stable")
    x = ((g[order[:n]] + 0.5) * (L / 8) + rng.uniform(-0.04, 0.04, (n, 3))).astype(np.float32)
    q = rng.uniform(-0.5, 0.5, n).astype(np.float32)
    typ = (np.arange(n) % 2).astype(np.int32)
    tab = W.lj_table(np.array([0.3, 0.25]), np.array([0.6, 0.3]))
    eo, ei = np.zeros(n + 1, np.int32), np.zeros(0, np.int32)
    import torch
    from paper_2006_09167_b200 import nb
    for coul in ("ewald", "rf", "none"):
        ctx = nb.Context(n, tab, eo, ei, rc=1.0, coulomb=coul, ewald_rtol=1e-5)
        dev = torch.device("cuda", 0)
        xd, qd, td = (torch.from_numpy(a).to(dev) for a in (x, q, typ))
        f = torch.full((n, 3), float("nan"), dtype=torch.float32, device=dev)
        e = torch.zeros(2, dtype=torch.float64, device=dev)
        v = torch.zeros(9, dtype=torch.float64, device=dev)
        box = np.full(3, L, np.float32)
        ctx.put_atoms(xd, qd, td, box)
        ctx.search(1.2)
        for part in range(3):
            ctx.prune(1.1, part, 3)          # more parts than work units is legal
        ctx.forces(f, e, v)
        torch.cuda.synchronize()
        ref = O.forces(x, q, typ, box, tab, eo, ei,
                       O.Params(rc=1.0, ntypes=2, coulomb=coul, beta=O.beta_from_rtol(1.0, 1e-5) if coul == "ewald" else 0.0))
        fg = f.cpu().numpy().astype(np.float64)
        assert np.isfinite(fg).all()
        if ref.npairs == 0:
            assert np.all(fg == 0.0) and float(e.sum()) == 0.0
        else:
            assert rel_rms(fg, ref.f) <= TOL_F
            assert abs(float(e.sum()) - ref.energy) <= TOL_E * max(abs(ref.energy), abs(ref.e_lj) + abs(ref.e_coul))
            assert np.linalg.norm(v.cpu().numpy().reshape(3, 3) - ref.virial) <= TOL_E * np.linalg.norm(ref.virial)
        assert ctx.count_pairs()[0] == ref.npairs
        ctx.close()


def test_put_atoms_without_charges_and_types(cfg0):
    """q / type = NULL means "unchanged since the previous nb_put_atoms" (device and host entry points);
    NULL on the very first call is an argument error."""
    import torch
    from paper_2006_09167_b200 import nb
    w = cfg0
    d = Driver(w)
    with pytest.raises(nb.NbError):
        d.ctx.put_atoms(torch.from_numpy(w.x).to(d.dev), None, None, w.box)
    d.put()
    d.ctx.search(w.rlist_outer)
    x1 = w.positions_at(3)
    d.put(x1)
    f_full = d.forces()
    d.put()                                         # back to frame 0 with everything
    d.ctx.put_atoms(torch.from_numpy(x1).to(d.dev), None, None, w.box)
    assert rel_rms(d.forces(), f_full) < 1e-6      # same inputs up to atomic summation order
    d.put()
    d.ctx.put_atoms_host(x1, None, None, w.box)
    assert rel_rms(d.forces(), f_full) < 1e-6


def test_host_entry_points(cfg0):
    w = cfg0
    d = Driver(w)
    d.ctx.put_atoms_host(w.x, w.q, w.type, w.box)
    d.ctx.search(w.rlist_outer)
    f = np.zeros((w.natoms, 3), np.float32)
    e = np.zeros(2)
    v = np.zeros(9)
    d.ctx.forces_host(f, e, v)
    ref = oracle_forces(w)
    assert rel_rms(f.astype(np.float64), ref.f) <= TOL_F
    assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E


def test_error_codes(cfg0):
    from paper_2006_09167_b200 import nb
    w = cfg0
    d = Driver(w)
    with pytest.raises(nb.NbError) as ei:
        d.ctx.search(w.rlist_outer)
    assert ei.value.code == -2   # NB_ERR_STATE: no atoms yet
    d.put()
    with pytest.raises(nb.NbError) as ei:
        d.ctx.search(0.5)        # below rc
    assert ei.value.code == -3
    with pytest.raises(nb.NbError) as ei:
        d.ctx.search(1.0)        # above L/2
    assert ei.value.code == -3
    with pytest.raises(nb.NbError) as ei:
        d.ctx.forces(d.f)
    assert ei.value.code == -2
    d.ctx.search(w.rlist_outer)
    with pytest.raises(nb.NbError) as ei:
        d.ctx.prune(0.95)        # above rlist_outer
    assert ei.value.code == -3
    with pytest.raises(nb.NbError) as ei:
        d.ctx.prune(w.rlist_inner, 2, 2)
    assert ei.value.code == -1
    with pytest.raises(nb.NbError):
        nb.Context(10, np.zeros((1, 1, 2), np.float32), None, None, rc=-1.0)


def test_pair_count_and_stage_timing(cfg0):
    """nb_count_pairs equals the oracle's count of pairs within rc (a handful of pairs may sit within
    fp32 rounding of rc); nb_timing_* reports one interval per stage call."""
    w = cfg0
    d = Driver(w)
    d.ctx.timing_enable(True)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.put()
    d.ctx.prune(w.rlist_inner)
    ref = oracle_forces(w)
    n_int, n_exc = d.ctx.count_pairs()
    assert abs(n_int - ref.npairs) <= 2 and ref.npairs > 90000
    assert abs(n_exc - ref.npairs_excl) <= 0 and n_exc == 3 * (w.natoms // 3)
    d.forces()
    d.forces(energy=True, virial=True)
    t = d.ctx.timing_read()
    assert t["put"][1] == 2 and t["grid"][1] == 1 and t["search"][1] == 1 and t["masks"][1] == 1
    assert t["prune"][1] == 1 and t["force"][1] == 2 and t["reduce"][1] == 2
    assert all(v[0] > 0 for v in t.values())
    t2 = d.ctx.timing_read()
    assert all(v == (0.0, 0) for v in t2.values())
    d.ctx.timing_enable(False)
    d.forces()
    assert d.ctx.timing_read()["force"][1] == 0
