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


def spread_ranges(ncl, nranges, width):
    """nranges cluster ranges of `width` clusters spread evenly over [0, ncl), the first and last touching the ends."""
    starts = np.unique(np.linspace(0, max(ncl - width, 0), nranges).astype(int))
    return [(int(a), int(min(a + width, ncl))) for a in starts]


def check_half_list(d, w, c_ranges=None, part=None, before=None):
    """The compact inner list the force kernel streams (nb_inner_dump: single j atoms of the cluster pairs without a
    mask, whole cluster pairs with one) against oracle_atom_lists on the
    library's slot table at the CURRENT coordinates, bit-exact as sets (no guard band: both sides decide
    in fp32 with the A12 operation order); no duplicates, no dummy entries.
    c_ranges: compare only entries whose first or second cluster lies in one of the ranges (sampled check);
    part: compare only the entries of this rolling part (the one just pruned) -- the other parts must be
    what they were in `before` (a previous return value of this function: the keys of all entries)."""
    aos, xq = d.slots()
    ncl = aos.size // 8
    ci, ent, s, kind, prt = d.inner_dump()
    keys = LC.half_entry_keys(ci, ent, s, kind)
    assert np.unique(keys).size == keys.size, "duplicate entry in the compact inner list"
    cj = np.where(kind == 0, ent // 8, ent)
    assert ent.size == 0 or (cj.max() < ncl and cj.min() >= 0 and ci.max() < ncl), "dummy or out-of-range entry leaked"
    if part is not None:
        # the oracle's entries of that part: the part of an entry is the part of its outer triple in the library's list
        oci, ocj, os_, _, opart = d.dump(0)
        okeys = LC.triple_keys(oci, ocj, os_)
        order = np.argsort(okeys)
        okeys, opart = okeys[order], opart[order]
    for (c0, c1) in (c_ranges if c_ranges is not None else [(0, ncl)]):
        ref = O.atom_lists(aos, xq, w.box, w.rlist_outer, w.rlist_inner, w.excl_off, w.excl_idx, c_begin=c0, c_end=c1)
        rkeys = ref.keys()
        sel = ((ci >= c0) & (ci < c1)) | ((cj >= c0) & (cj < c1))
        if part is not None:
            rcj = np.where(ref.kind == 0, ref.entry // 8, ref.entry)
            tk = LC.triple_keys(ref.ci, rcj, ref.s)
            pos = np.searchsorted(okeys, tk)
            assert (pos < okeys.size).all() and np.array_equal(okeys[pos], tk), "oracle inner entry outside the library's outer list"
            rkeys = rkeys[opart[pos] == part]
            sel &= prt == part
        got, want = np.sort(keys[sel]), np.sort(rkeys)
        assert got.size == want.size and np.array_equal(got, want), (c0, c1, part, got.size, want.size)
    if part is not None and before is not None:
        # label the earlier entries with TODAY's parts (through their outer triple) and compare the other parts
        bci, bent, bsid, bkind = before >> 38, (before >> 9) & ((1 << 29) - 1), (before >> 1) & 0xFF, before & 1
        btk = (bci << 36) | (np.where(bkind == 0, bent // 8, bent) << 8) | bsid
        bpart = opart[np.searchsorted(okeys, btk)]
        assert np.array_equal(np.sort(before[bpart != part]), np.sort(keys[prt != part])), "a prune changed another part"
    return keys


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
    assert st["slots_last_forces"] == d.ctx.count_slots() < 64 * st["n_pairs_inner"]
    hci, hent, _, hkind, _ = d.inner_dump()
    assert st["slots_last_forces"] == 8 * int((hkind == 0).sum()) + 64 * int((hkind == 1).sum())   # 8 i atoms x 1 j atom; whole masked pairs
    check_half_list(d, w)
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


def test_many_atom_types():
    """NB_MAX_TYPES - 1 = 95 LJ types (the paired LJ table of a block is then 6 KB of shared memory, the per-cluster rows
    95 x 64 B): a charged LJ mixture without exclusions, every flavour's forces / energies against the all-pairs oracle."""
    import dataclasses
    base = W.lj_fluid(12, rc=0.9)
    rng = np.random.Generator(np.random.PCG64(95))
    nt = 95
    sigma, eps = rng.uniform(0.25, 0.38, nt), rng.uniform(0.2, 1.0, nt)
    q = rng.uniform(-0.5, 0.5, base.natoms).astype(np.float32)
    q -= np.float32(q.mean())
    w = dataclasses.replace(base, type=rng.integers(0, nt, base.natoms).astype(np.int32), q=q, ntypes=nt,
                            lj_c6c12=W.lj_table(sigma, eps), coulomb="ewald")
    for coulomb in ("ewald", "rf", "none"):
        ww = dataclasses.replace(w, coulomb=coulomb)
        d = Driver(ww)
        d.put()
        d.ctx.search(ww.rlist_outer)
        d.ctx.prune(ww.rlist_inner)
        ref = oracle_forces(ww)
        f, e, vir = d.forces(energy=True, virial=True)
        assert rel_rms(f, ref.f) <= TOL_F
        assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
        assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
        assert rel_rms(d.forces(), ref.f) <= TOL_F
        d.ctx.close()


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
    # full-size list parity over ALL clusters (outer, inner, pair masks; then the half-cluster list the force kernel streams)
    d.ctx.prune(w.rlist_inner)
    check_lists(d, w, w.rlist_outer, w.rlist_inner)
    check_half_list(d, w)
    aos, xq = d.slots()
    ci, cj, s, _, _ = d.dump(1)
    miss, n = LC.coverage_missing(aos, xq, w.box, w.rlist_inner - 1e-6, ci, cj, s)
    assert miss == 0 and n > 5_000_000
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
    # rolling over moving atoms (motion recipe): forces, energies and virial stay equal to the all-pairs oracle,
    # the pruned part of the compact inner list is bit-exact against the oracle at the coordinates of the prune
    hl = check_half_list(d, w)
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
        hl = check_half_list(d, w, part=part, before=hl)
        r = oracle_forces(w, x=x, method="cells")
        f, e, vir = d.forces(energy=True, virial=True)
        assert rel_rms(f, r.f) <= TOL_F
        assert abs(e.sum() - r.energy) / abs(r.energy) <= TOL_E
        assert np.linalg.norm(vir - r.virial) / np.linalg.norm(r.virial) <= TOL_E
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
    drives them (search, full prune, then rolling parts on the motion recipe).  Lists: config 2 Ewald over ALL
    clusters (outer, inner, pair masks, and the half-cluster list the force kernel streams); the others on
    >= 1 % of the clusters in >= 8 ranges (the list oracle is O(n^2)), config 4's ranges including the
    slab/vapour boundaries; k-d-tree completeness of the inner list (whole box, or slabs of config 3 that
    include the periodic face).  Forces / energy / virial against the fp64 linked-cell oracle (pinned equal to
    all-pairs) at t = 0 and on moved frames after rolling prunes; effective pair count against the oracle's."""
    w = {"cfg2_ewald": lambda: W.config2("ewald"), "cfg2_rf": lambda: W.config2("rf"), "cfg4": W.config4,
         "cfg3": W.config3}[which]()
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    aos, xq = check_layout(d, w)
    d.ctx.prune(w.rlist_inner)
    ncl = d.ctx.get_layout()["nclusters"]
    if which == "cfg2_ewald":
        ranges = None
        check_lists(d, w, w.rlist_outer, w.rlist_inner)
    else:
        width = {"cfg2_rf": 16, "cfg4": 24, "cfg3": 176}[which]
        ranges = spread_ranges(ncl, 8, width)
        if which == "cfg4":
            # clusters at the two slab/vapour interfaces (x ~ 0 = 36.2 and x ~ 18.1): where cluster occupancy and list lengths jump
            with np.errstate(all="ignore"):
                import warnings
                with warnings.catch_warnings():
                    warnings.simplefilter("ignore", RuntimeWarning)   # (clusters of padding only have no mean)
                    xc = np.nanmean(np.where((aos >= 0)[:, None], xq[:, :3], np.nan).reshape(-1, 8, 3)[:, :, 0], axis=1)
            for x0 in (18.1, 0.3):
                c = int(np.nanargmin(np.abs(xc - x0)))
                ranges.append((max(c - 12, 0), min(c + 12, ncl)))
        assert sum(b - a for a, b in ranges) >= 0.01 * ncl and len(ranges) >= 8
        for r in ranges:
            check_lists(d, w, w.rlist_outer, w.rlist_inner, c_range=r)
    hl = check_half_list(d, w, c_ranges=ranges)
    # layout-independent completeness of the inner list (k-d tree, fp64)
    ci, cj, s, _, _ = d.dump(1)
    if which == "cfg2_ewald":
        miss, n = LC.coverage_missing(aos, xq, w.box, w.rlist_inner - 1e-6, ci, cj, s)
        assert miss == 0 and n > 20_000_000
    else:
        for z0 in (3.0, float(w.box[2]) - 1.2):   # one slab inside the box, one across the periodic face
            sub = LC.z_slab_subset(xq, w.box, z0, 2.4)
            miss, n = LC.coverage_missing(aos, xq, w.box, w.rlist_inner - 1e-6, ci, cj, s, subset=sub)
            assert miss == 0 and n > 3_000_000
    ref = oracle_forces(w, method="cells")
    f, e, vir = d.forces(energy=True, virial=True)
    assert rel_rms(f, ref.f) <= TOL_F
    assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
    assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    npairs, _ = d.ctx.count_pairs()
    assert abs(npairs - ref.npairs) <= 2 + 1e-6 * ref.npairs     # fp32 vs fp64 at r = rc
    fsum = np.abs(f.sum(axis=0)).max() / (np.sqrt((f**2).mean()) * w.natoms)
    assert fsum < 1e-6                                           # T6 on the GPU
    sample = ranges if ranges is not None else spread_ranges(ncl, 8, 32)
    if which == "cfg3":
        sample = sample[::3]   # (the O(n^2) list oracle on 1.07 M atoms: the full sample once, above; three ranges per rolling check)
    for t in (1, 2, w.nparts + 1, 50, 99) if which != "cfg3" else (1, w.nparts + 1, 99):
        x = w.positions_at(t)
        d.put(x)
        part = t % w.nparts
        d.ctx.prune(w.rlist_inner, part, w.nparts)
        # the pruned part of the compact list against the oracle at THESE coordinates (config 2 Ewald: all clusters at t = 1)
        hl = check_half_list(d, w, c_ranges=None if (which == "cfg2_ewald" and t == 1) else sample, part=part,
                             before=hl if which != "cfg3" else None)
        r = oracle_forces(w, x=x, method="cells")
        if t in (1, 99):
            f, e, vir = d.forces(energy=True, virial=True)     # energies and virial on a moved frame after a rolling prune
            assert abs(e.sum() - r.energy) / abs(r.energy) <= TOL_E
            assert np.linalg.norm(vir - r.virial) / np.linalg.norm(r.virial) <= TOL_E
            assert rel_rms(f, r.f) <= TOL_F
        assert rel_rms(d.forces(), r.f) <= TOL_F
    # the inner steps as bench.py launches them: nb_step (each rolling part: plain path once, graph capture once, then
    # graph launches); forces of the graph-launched steps against the oracle, the part pruned by the last one against
    # the oracle's half-cluster list
    import torch
    k = w.nparts
    t0, t1 = 10, 10 + 3 * k
    for t in range(t0, t1):
        x = w.positions_at(t)
        xt = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(d.dev)
        ft = torch.full((w.natoms, 3), float("nan"), dtype=torch.float32, device=d.dev)
        d.ctx.step(xt, w.rlist_inner, t % k, k, ft)
        if t >= t1 - 2:
            torch.cuda.synchronize()
            assert rel_rms(ft.cpu().numpy().astype(np.float64), oracle_forces(w, x=x, method="cells").f) <= TOL_F
    check_half_list(d, w, c_ranges=sample, part=(t1 - 1) % k)
    # ... and the other order bench.py --prune auto may pick: the rolling prune on the second stream next to the force
    # kernel (nb_prune_overlapped; the part pruned on step t's coordinates is first used at step t + 1)
    for t in range(t1, t1 + 2 * k + 1):
        x = w.positions_at(t)
        d.put(x)                                          # joins the prune of step t - 1: its part flips here
        d.ctx.prune_overlapped(w.rlist_inner, t % k, k)
        f = d.forces()
    assert rel_rms(f, oracle_forces(w, x=x, method="cells").f) <= TOL_F   # (every part has been through the second buffer by now)
    d.put(x)                                              # same coordinates again: the last prune is joined, nothing moved
    if which != "cfg3":
        check_half_list(d, w, c_ranges=sample, part=(t1 + 2 * k) % k)


@pytest.mark.parametrize("which", ["cfg0", "rect_rf", "lj"])
def test_half_cluster_inner_list(which):
    """The compact inner list the force kernel streams is kept at single-j-atom granularity (DESIGN.md
    section 5, reading A22).  Bit-exact against oracle_atom_lists after a full prune and after rolling parts on moved
    coordinates; layout-independent fp64 check (k-d tree) that it is COMPLETE; the cluster pairs it spans
    are exactly the inner list of nb_list_dump (which is derived from it)."""
    w = {"cfg0": W.config0, "lj": lambda: W.lj_fluid(12, rc=0.9),
         "rect_rf": lambda: W.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84,
                                          box_scale=(1.0, 1.1, 1.25), coulomb="rf")}[which]()
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner, 0, 1)
    hl = check_half_list(d, w)
    for x, part, nparts in ((w.positions_at(40), 0, 2), (w.positions_at(41), 1, 2), (w.positions_at(42), 0, 2)):
        d.put(x)
        d.ctx.prune(w.rlist_inner, part, nparts)
        hl = check_half_list(d, w, part=part, before=hl)
    aos, xq = d.slots()
    box = np.asarray(w.box, dtype=np.float64)
    ci, ent, svec, kind, _ = d.inner_dump()
    half = kind == 0
    skey = LC.shift_id(svec)
    hkeys = set(zip(ci[half].tolist(), ent[half].tolist(), skey[half].tolist()))
    mkeys = set(zip(ci[~half].tolist(), ent[~half].tolist(), skey[~half].tolist()))
    # complete for the CURRENT coordinates at rc (parts pruned at earlier frames keep what was within rlist_inner then)
    si, sj, sp, _ = LC.close_atom_pairs(aos, xq, box, w.rc)
    ka, kb = LC.shift_id(sp), LC.shift_id(-sp)
    missing = 0
    for a, b, k1, k2 in zip(si.tolist(), sj.tolist(), ka.tolist(), kb.tolist()):
        if ((a // 8, b, k1) in hkeys or (b // 8, a, k2) in hkeys or (a // 8, b // 8, k1) in mkeys
                or (b // 8, a // 8, k2) in mkeys):
            continue
        missing += 1
    assert missing == 0 and si.size > 1000
    # same cluster pairs as the bit-plane inner list
    dci, dcj, dsv, _, _ = d.dump(1)
    planes = set(zip(dci.tolist(), dcj.tolist(), LC.shift_id(dsv).tolist()))
    spanned = {(a, e // 8, k) for a, e, k in hkeys} | mkeys
    assert spanned == planes


def test_overlapped_prune(cfg1):
    """nb_prune_overlapped: the prune of a rolling part runs on the library's second stream next to the force
    kernel and the part switches to the new list at the next nb_put_atoms.  Forces of the step that issued
    it still come from the previous list; after the switch the part is bit-exact against the oracle ON THE
    COORDINATES THE PRUNE SAW, the other parts are untouched; forces / energies stay equal to the oracle over
    a run that alternates parts; plain nb_prune and a change of nparts in between keep everything consistent."""
    w = cfg1
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner)
    hl = check_half_list(d, w)
    k = w.nparts
    for t in range(1, 8):
        x = w.positions_at(t)
        d.put(x)                                     # joins the prune of step t-1: its part flips here
        if t > 1:
            # the part pruned at t-1 must equal the oracle at x_{t-1}; check by putting x_{t-1} back for the comparison only
            d.put(w.positions_at(t - 1))
            hl = check_half_list(d, w, c_ranges=spread_ranges(d.ctx.get_layout()["nclusters"], 6, 24), part=(t - 1) % k, before=hl)
            d.put(x)
        d.ctx.prune_overlapped(w.rlist_inner, t % k, k)
        f, e, vir = d.forces(energy=True, virial=True)
        r = oracle_forces(w, x=x, method="cells")
        assert rel_rms(f, r.f) <= TOL_F
        assert abs(e.sum() - r.energy) / abs(r.energy) <= TOL_E
        assert np.linalg.norm(vir - r.virial) / np.linalg.norm(r.virial) <= TOL_E
    # a plain prune of the other part while one part lives in the second buffer, then a different nparts
    x = w.positions_at(8)
    d.put(x)
    cur = check_half_list(d, w, c_ranges=[(0, 0)])   # (nothing compared: just the current entries)
    d.ctx.prune(w.rlist_inner, 0, k)
    hl = check_half_list(d, w, part=0, before=cur)
    assert rel_rms(d.forces(), oracle_forces(w, x=x, method="cells").f) <= TOL_F
    d.ctx.prune_overlapped(w.rlist_inner, 2, 3)
    assert rel_rms(d.forces(), oracle_forces(w, x=x, method="cells").f) <= TOL_F
    d.put(x)
    hl = check_half_list(d, w, part=2)
    d.ctx.prune(w.rlist_inner)                       # full prune: everything back in one buffer
    check_half_list(d, w)
    assert rel_rms(d.forces(), oracle_forces(w, x=x, method="cells").f) <= TOL_F


def inner_keys(d):
    ci, ent, sv, kind, part = d.inner_dump()
    return set(zip(ci.tolist(), ent.tolist(), LC.shift_id(sv).tolist(), kind.tolist()))


@pytest.mark.parametrize("which", ["cfg1", "tiny"])
def test_step_graph(which):
    """nb_step = nb_put_atoms + nb_prune + nb_forces in one call; from the second use of a rolling part on a list
    it is one CUDA graph launch.  Two contexts on the same box, one driven by the three calls and one by nb_step,
    over two list lifetimes (the graphs are updated in place after the second search): identical inner lists at every
    step, forces equal up to the order of the atomic adds and within 1e-5 of the oracle; with stage timing on
    (plain path inside nb_step) still the same; errors before a search / after a box change."""
    import torch
    from paper_2006_09167_b200 import nb
    w = W.config1() if which == "cfg1" else W.small_water(150, 2.0, seed=23, rc=0.8, rlist_outer=0.9, rlist_inner=0.84)
    k = 2
    a, b = Driver(w), Driver(w)
    with pytest.raises(nb.NbError):
        b.put()
        b.ctx.step(b.x, w.rlist_inner, 0, k, b.f)          # no list yet
    for life in range(2):
        x0 = w.positions_at(10 * life)
        for d in (a, b):
            d.put(x0)
            d.ctx.search(w.rlist_outer)
            d.ctx.prune(w.rlist_inner)
            d.forces()
        for t in range(1, 9):
            x = w.positions_at(10 * life + t)
            a.put(x)
            a.ctx.prune(w.rlist_inner, t % k, k)
            fa = a.forces()
            xb = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(b.dev)
            fb_t = torch.full((w.natoms, 3), float("nan"), dtype=torch.float32, device=b.dev)   # new buffers every step: patched in
            if t == 6:
                b.ctx.timing_enable(True)                  # plain path inside nb_step
            b.ctx.step(xb, w.rlist_inner, t % k, k, fb_t)
            if t == 6:
                b.ctx.timing_enable(False)
            torch.cuda.synchronize()
            fb = fb_t.cpu().numpy().astype(np.float64)
            assert rel_rms(fb, fa) <= 2e-6
            if t in (1, 4, 8):
                assert rel_rms(fb, oracle_forces(w, x=x, method="cells" if which == "cfg1" else "allpairs").f) <= TOL_F
                assert inner_keys(a) == inner_keys(b)
    st = b.ctx.get_stats()
    assert st["force_count"] == a.ctx.get_stats()["force_count"] and st["prune_count"] == a.ctx.get_stats()["prune_count"]
    # more keys than the cache holds (8): ten inner radii, three uses each (plain, capture, graph launch), evicting as it goes
    x = w.positions_at(19)
    xb = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(b.dev)
    fb_t = torch.empty((w.natoms, 3), dtype=torch.float32, device=b.dev)
    ref = oracle_forces(w, x=x, method="cells" if which == "cfg1" else "allpairs").f
    for i in range(10):
        rl = w.rlist_inner + 1e-4 * i
        for _ in range(3):
            b.ctx.step(xb, rl, 1, k, fb_t)
        torch.cuda.synchronize()
        assert rel_rms(fb_t.cpu().numpy().astype(np.float64), ref) <= TOL_F
    bad_box = np.asarray(w.box, dtype=np.float32) * np.float32(1.01)
    b.ctx.put_atoms(b.x, b.q, b.t, bad_box)
    with pytest.raises(nb.NbError):
        b.ctx.step(b.x, w.rlist_inner, 0, k, b.f)


def test_step_host(cfg1):
    """nb_step_host: host positions in, host forces out, the prune of the next step's part started after the force
    kernel on the second stream (overlapping the copies).  Forces within 1e-5 of the oracle at every step of a run
    over two rolling parts; the part pruned by the last call equals the oracle's half-cluster list on the coordinates
    that call saw; pinned and pageable buffers both work."""
    import torch
    w = cfg1
    k = w.nparts
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner)
    d.forces()
    f_pin = torch.zeros((w.natoms, 3), dtype=torch.float32).pin_memory()
    x_pin = torch.zeros((w.natoms, 3), dtype=torch.float32).pin_memory()
    f_pag = np.zeros((w.natoms, 3), dtype=np.float32)
    for t in range(1, 9):
        x = np.ascontiguousarray(w.positions_at(t), dtype=np.float32)
        if t % 3:
            x_pin.numpy()[:] = x
            d.ctx.step_host(x_pin.numpy(), f_pin.numpy(), w.rlist_inner, (t + 1) % k, k)
            f = f_pin.numpy().astype(np.float64)
        else:
            d.ctx.step_host(x, f_pag, w.rlist_inner, (t + 1) % k, k)
            f = f_pag.astype(np.float64)
        assert rel_rms(f, oracle_forces(w, x=x, method="cells").f) <= TOL_F
    # the last call pruned part (8 + 1) % k on x_8: join it by putting x_8 again, then compare that part with the oracle
    d.put(w.positions_at(8))
    check_half_list(d, w, c_ranges=spread_ranges(d.ctx.get_layout()["nclusters"], 6, 24), part=9 % k)
    assert rel_rms(d.forces(), oracle_forces(w, x=w.positions_at(8), method="cells").f) <= TOL_F


@pytest.mark.parametrize("which", ["cfg0", "cfg1", "rect_rf", "lj"])
def test_fused_first_prune(which):
    """nb_forces_prune -- one kernel walks the OUTER list of a fresh search,
    computes forces (+ energies, virial) and writes the inner list.  The list it writes is bit-equal to
    nb_prune's and to the oracle's half-cluster list; forces / energies / virial within 1e-5 of the oracle,
    in every flavour {Ewald, RF, LJ-only} x {F, F+E+virial}; the steps after it run on its list."""
    w = {"cfg0": W.config0, "cfg1": W.config1, "lj": lambda: W.lj_fluid(12, rc=0.9),
         "rect_rf": lambda: W.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84,
                                          box_scale=(1.0, 1.1, 1.25), coulomb="rf")}[which]()
    method = "cells" if which == "cfg1" else "allpairs"
    ref = oracle_forces(w, method=method)
    d = Driver(w)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner)
    by_prune = np.sort(LC.half_entry_keys(*d.inner_dump()[:4]))
    for energy in (False, True):
        d.ctx.search(w.rlist_outer)
        d.f.fill_(float("nan"))
        d.ctx.forces_prune(w.rlist_inner, d.f, d.e if energy else None, d.v if energy else None)
        d.torch.cuda.synchronize()
        f = d.f.cpu().numpy().astype(np.float64)
        assert rel_rms(f, ref.f) <= TOL_F
        if energy:
            e, vir = d.e.cpu().numpy(), d.v.cpu().numpy().reshape(3, 3)
            assert abs(e.sum() - ref.energy) / abs(ref.energy) <= TOL_E
            assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
        fused = check_half_list(d, w)                                   # bit-exact against the oracle ...
        assert np.array_equal(np.sort(fused), by_prune)                 # ... and against the separate prune kernel
        assert rel_rms(d.forces(), ref.f) <= TOL_F                      # the next step runs on the list it wrote
    x = w.positions_at(3)
    d.put(x)
    d.ctx.prune(w.rlist_inner, 1 % w.nparts, w.nparts)
    assert rel_rms(d.forces(), oracle_forces(w, x=x, method=method).f) <= TOL_F
    st = d.ctx.get_stats()
    assert st["prune_count"] == 4 and st["search_count"] == 3


@pytest.mark.parametrize("coulomb", ["ewald", "rf"])
def test_twin_cutoffs(coulomb):
    """SURVEY 8.1 (f4), PAPER.md L205 / L215: rc_vdw < rc (electrostatics cut-off scaled up by PME load balancing).
    Forces, both energies and the virial against the oracle's twin cut-off reading, plain and fused-prune flavours."""
    w = W.small_water(150, 2.0, seed=21, rc=0.9, rlist_outer=0.98, rlist_inner=0.93, box_scale=(1.0, 1.1, 1.25), coulomb=coulomb)
    rcv = 0.7
    p = O.Params(rc=w.rc, ntypes=w.ntypes, coulomb=coulomb, beta=O.beta_from_rtol(w.rc, w.ewald_rtol) if coulomb == "ewald" else 0.0,
                 rc_vdw=rcv)
    ref = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p)
    single = oracle_forces(w)
    assert abs(ref.e_lj - single.e_lj) > 1e-3 * abs(single.e_lj)       # the second cut-off matters on this box
    d = Driver(w, rc_vdw=rcv)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.forces_prune(w.rlist_inner, d.f, d.e, d.v)
    d.torch.cuda.synchronize()
    for f, e, vir in ((d.f.cpu().numpy().astype(np.float64), d.e.cpu().numpy(), d.v.cpu().numpy().reshape(3, 3)),
                      d.forces(energy=True, virial=True)):
        assert rel_rms(f, ref.f) <= TOL_F
        assert abs(e[0] - ref.e_lj) <= TOL_E * abs(ref.energy) and abs(e[1] - ref.e_coul) <= TOL_E * abs(ref.energy)
        assert np.linalg.norm(vir - ref.virial) / np.linalg.norm(ref.virial) <= TOL_E
    assert rel_rms(d.forces(), ref.f) <= TOL_F
    from paper_2006_09167_b200 import nb
    with pytest.raises(nb.NbError):
        nb.context_for(w, rc_vdw=1.0)                                  # rc_vdw > rc


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
            assert r["eff_searched"] <= r["eff_pruned"] < r["eff_streamed"] < r["eff_1x1_ideal"] <= 1.0   # finer list, fewer slots
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
    assert t["prune"][1] == 1 and t["force"][1] == 1 and t["force_energy"][1] == 1 and t["reduce"][1] == 2
    assert all(v[0] > 0 for v in t.values())
    t2 = d.ctx.timing_read()
    assert all(v == (0.0, 0) for v in t2.values())
    d.ctx.timing_enable(False)
    d.forces()
    assert d.ctx.timing_read()["force"][1] == 0
