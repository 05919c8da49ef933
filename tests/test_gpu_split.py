"""Local / non-local split of the non-bonded work, through the C ABI on the B200:
nb_set_local / nb_forces_nonlocal / nb_sync_nonlocal / nb_forces_local against the oracle (oracle_forces_split and the
all-pairs definition), lists bit-exact as without the split, clusters pure, the force order partitioned by locality."""
import numpy as np
import pytest

from paper_2006_09167_b200 import workloads as W
from tests.gpu_util import Driver, oracle_forces, oracle_params, rel_rms
from tests.splitutil import local_first
from tests.test_gpu_parity import check_half_list, check_lists

pytestmark = pytest.mark.gpu
TOL_F = 1e-5


def split_oracle(w, nlocal, which):
    from oracle import oracle as O
    return O.forces_split(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, oracle_params(w), nlocal, which)


def halo_workload(w0, frac=0.5):
    """Local atoms = the molecules whose first atom has x < frac * Lx: a home slab with its periodic halo around it."""
    return local_first(w0, lambda x: x[:, 0] < frac * w0.box[0])


def split_forces(d, nlocal):
    """nb_forces_nonlocal -> sync -> check what is there -> nb_forces_local; returns (f after the first call, f at the end)."""
    d.f.fill_(float("nan"))
    d.ctx.forces_nonlocal(d.f)
    d.ctx.sync_nonlocal()
    f_nl = d.f.cpu().numpy().astype(np.float64)       # the halo rows are complete here, by contract
    d.ctx.forces_local(d.f)
    d.torch.cuda.synchronize()
    return f_nl, d.f.cpu().numpy().astype(np.float64)


def check_partition(d, nlocal):
    """Clusters are pure and local ones come first; the force order has every local-local entry before every other."""
    info = d.ctx.split_info()
    aos, _ = d.slots()
    ncl_loc = info["nclusters_local"]
    cl = aos.reshape(-1, 8)
    real = cl >= 0
    is_loc = np.where(real, cl < nlocal, True).all(axis=1)
    is_nl = np.where(real, cl >= nlocal, True).all(axis=1)
    nclusters = cl.shape[0]
    assert is_loc[:ncl_loc].all() and is_nl[ncl_loc:].all()
    assert info["nlocal"] == nlocal and 0 < ncl_loc < nclusters
    assert np.sort(aos[aos >= 0]).tolist() == list(range(d.w.natoms))
    ci, ent, _, kind, _ = d.inner_dump()               # walks the segments in the force kernel's order
    cj = np.where(kind == 0, ent // 8, ent)
    loc = (ci < ncl_loc) & (cj < ncl_loc)
    nloc = int(loc.sum())
    assert 0 < nloc < loc.size
    assert loc[:nloc].all() and not loc[nloc:].any(), "local and non-local segments interleave in the force order"
    assert 0 < info["nseg_local"] < info["nseg"]
    return info


@pytest.mark.parametrize("which", ["cfg0", "rect_rf", "lj"])
def test_split_small_systems(which):
    w0 = {"cfg0": W.config0,
          "rect_rf": lambda: W.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84,
                                           box_scale=(1.0, 1.1, 1.25), coulomb="rf"),
          "lj": lambda: W.lj_fluid(12, rc=0.9)}[which]()
    w, nlocal = halo_workload(w0, 0.45)
    d = Driver(w)
    d.ctx.set_local(nlocal)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner, 0, 1)
    check_lists(d, w, w.rlist_outer, w.rlist_inner)          # the lists are the same sets, bit for bit, on the split grid
    check_half_list(d, w)
    check_partition(d, nlocal)
    whole = oracle_forces(w)
    f_all, e, v = d.forces(energy=True, virial=True)           # the union path is unchanged by the split
    assert rel_rms(f_all, whole.f) <= TOL_F
    assert abs(e.sum() - whole.energy) <= 1e-5 * abs(whole.energy)
    assert np.linalg.norm(v - whole.virial) <= 1e-5 * np.linalg.norm(whole.virial)
    f_nl, f = split_forces(d, nlocal)
    nl = split_oracle(w, nlocal, 2)
    # after the non-local kernel: the halo atoms' forces are final (= their rows of the non-local part = of the whole),
    # the local atoms' rows have not been written
    assert rel_rms(f_nl[nlocal:], nl.f[nlocal:]) <= TOL_F and rel_rms(f_nl[nlocal:], whole.f[nlocal:]) <= TOL_F
    assert np.isnan(f_nl[:nlocal]).all()
    assert rel_rms(f, whole.f) <= TOL_F and rel_rms(f, f_all) <= 2e-6
    # twice in a row, and the plain call afterwards: the accumulator is left clean
    _, f2 = split_forces(d, nlocal)
    assert rel_rms(f2, whole.f) <= TOL_F
    assert rel_rms(d.forces(), whole.f) <= TOL_F
    # the F + E + virial flavour of the pair: both kernels add into the energies and the per-shift sums, both gathers into
    # sum x (x) f; complete after nb_forces_local
    d.f.fill_(float("nan"))
    d.e.fill_(float("nan"))
    d.v.fill_(float("nan"))
    d.ctx.forces_nonlocal(d.f, d.e, d.v)
    d.ctx.sync_nonlocal()
    d.ctx.forces_local(d.f)
    d.torch.cuda.synchronize()
    fe, ee, ve = d.f.cpu().numpy().astype(np.float64), d.e.cpu().numpy(), d.v.cpu().numpy().reshape(3, 3)
    assert rel_rms(fe, whole.f) <= TOL_F
    assert abs(ee[0] - whole.e_lj) <= 1e-5 * abs(whole.energy) and abs(ee[1] - whole.e_coul) <= 1e-5 * abs(whole.energy)
    assert np.linalg.norm(ve - whole.virial) <= 1e-5 * np.linalg.norm(whole.virial)
    assert np.allclose(ee, e, rtol=1e-9, atol=1e-9 * abs(whole.energy)) and np.linalg.norm(ve - v) <= 1e-5 * np.linalg.norm(v)
    with pytest.raises(Exception):
        d.ctx.forces_nonlocal(d.f, None, d.v)      # virial needs energies
    assert rel_rms(d.forces(), whole.f) <= TOL_F   # (the rejected call left no split step pending)
    # the local kernel alone = the local atoms alone (oracle part 1): non-local forces on the local atoms are the difference
    loc = split_oracle(w, nlocal, 1)
    assert rel_rms(f[:nlocal] - nl.f[:nlocal], loc.f[:nlocal]) <= 1e-4   # (difference of two fp32 results)


def test_split_config1_rolling_and_step(cfg1):
    w, nlocal = halo_workload(cfg1, 0.6)
    d = Driver(w)
    d.ctx.set_local(nlocal)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner, 0, 1)
    check_lists(d, w, w.rlist_outer, w.rlist_inner)
    keys = check_half_list(d, w)
    info = check_partition(d, nlocal)
    assert info["nseg_local"] > 1000 and info["nseg"] - info["nseg_local"] > 1000
    fx = d.torch.zeros_like(d.f)
    for t in (1, 2, 7):
        x = w.positions_at(t)
        part = t % w.nparts
        if t == 7:
            xt = d.torch.from_numpy(x).to(d.dev)
            d.ctx.step(xt, w.rlist_inner, part, w.nparts, fx)       # the one-call inner step on the split grid
            d.torch.cuda.synchronize()
            d.x = xt
        elif t == 2:
            d.put(x)
            d.ctx.prune_overlapped(w.rlist_inner, part, w.nparts)   # second stream; joined by the split calls / the dump
        else:
            d.put(x)
            d.ctx.prune(w.rlist_inner, part, w.nparts)
        keys = check_half_list(d, w, part=part, before=keys)
        check_partition(d, nlocal)
        ww = __import__("dataclasses").replace(w, x=x)
        whole = oracle_forces(ww, method="cells")
        f_nl, f = split_forces(d, nlocal)
        assert rel_rms(f_nl[nlocal:], whole.f[nlocal:]) <= TOL_F and np.isnan(f_nl[:nlocal]).all()
        assert rel_rms(f, whole.f) <= TOL_F
        if t == 7:
            assert rel_rms(fx.cpu().numpy().astype(np.float64), whole.f) <= TOL_F
    # switching the split off again needs a new search and gives the plain grid back
    d.ctx.set_local(w.natoms)
    from paper_2006_09167_b200 import nb
    with pytest.raises(nb.NbError) as ei:
        d.ctx.forces(d.f)
    assert ei.value.code == -2     # NB_ERR_STATE: the list was dropped
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner, 0, 1)
    info = d.ctx.split_info()
    assert info["nseg_local"] == info["nseg"] and info["nlocal"] == w.natoms
    assert rel_rms(d.forces(), oracle_forces(w, method="cells").f) <= TOL_F


def test_split_config4_heterogeneous_full_size():
    """The slab / vapour system with five atom types and random charges at full size (150k atoms): half of the dense slab
    is local, the other half and the vapour non-local; sampled list ranges on both sides of the class boundary."""
    import dataclasses
    from tests.test_gpu_parity import spread_ranges
    w0 = W.config4()
    w, nlocal = local_first(w0, lambda x: x[:, 0] < 9.0)
    assert 0.2 * w.natoms < nlocal < 0.6 * w.natoms
    d = Driver(w)
    d.ctx.set_local(nlocal)
    d.put()
    d.ctx.search(w.rlist_outer)
    d.ctx.prune(w.rlist_inner, 0, 1)
    info = check_partition(d, nlocal)
    ncl = d.ctx.get_layout()["nclusters"]
    ncl_loc = info["nclusters_local"]
    ranges = [(max(ncl_loc - 12, 0), min(ncl_loc + 12, ncl))] + spread_ranges(ncl, 4, 16)   # the first straddles the class boundary
    for r in ranges:
        check_lists(d, w, w.rlist_outer, w.rlist_inner, c_range=r)
    check_half_list(d, w, c_ranges=ranges)
    whole = oracle_forces(w, method="cells")
    f_nl, f = split_forces(d, nlocal)
    assert rel_rms(f_nl[nlocal:], whole.f[nlocal:]) <= TOL_F and np.isnan(f_nl[:nlocal]).all()
    assert rel_rms(f, whole.f) <= TOL_F
    # a moved frame after a rolling prune
    x = w.positions_at(3)
    d.put(x)
    d.ctx.prune(w.rlist_inner, 3 % w.nparts, w.nparts)
    whole = oracle_forces(dataclasses.replace(w, x=x), method="cells")
    f_nl, f = split_forces(d, nlocal)
    assert rel_rms(f_nl[nlocal:], whole.f[nlocal:]) <= TOL_F and rel_rms(f, whole.f) <= TOL_F


def test_split_call_order_and_arguments(cfg0):
    from paper_2006_09167_b200 import nb
    w, nlocal = halo_workload(cfg0, 0.5)
    d = Driver(w)
    for bad in (0, -3, w.natoms + 1):
        with pytest.raises(nb.NbError) as ei:
            d.ctx.set_local(bad)
        assert ei.value.code == -1
    d.ctx.set_local(nlocal)
    d.put()
    with pytest.raises(nb.NbError) as ei:
        d.ctx.forces_nonlocal(d.f)              # no list yet
    assert ei.value.code == -2
    d.ctx.search(w.rlist_outer)
    with pytest.raises(nb.NbError) as ei:
        d.ctx.forces_local(d.f)                 # local before non-local
    assert ei.value.code == -2
    d.ctx.forces_nonlocal(d.f)
    with pytest.raises(nb.NbError) as ei:
        d.ctx.forces_nonlocal(d.f)              # twice
    assert ei.value.code == -2
    with pytest.raises(nb.NbError) as ei:
        d.ctx.set_local(nlocal - 3)             # in the middle of a split step
    assert ei.value.code == -2
    for call in (lambda: d.put(), lambda: d.ctx.search(w.rlist_outer), lambda: d.ctx.prune(w.rlist_inner, 0, 1),
                 lambda: d.ctx.forces(d.f)):    # nothing may overtake the non-local kernel: these wait for nb_forces_local
        with pytest.raises(nb.NbError) as ei:
            call()
        assert ei.value.code == -2
    d.ctx.forces_local(d.f)
    d.torch.cuda.synchronize()
    assert rel_rms(d.f.cpu().numpy().astype(np.float64), oracle_forces(w).f) <= TOL_F
    # a context without a split: the two calls still work (everything is local, the non-local kernel is empty)
    d2 = Driver(cfg0)
    d2.put()
    d2.ctx.search(cfg0.rlist_outer)
    d2.f.fill_(float("nan"))
    d2.ctx.forces_nonlocal(d2.f)
    d2.ctx.sync_nonlocal()
    d2.ctx.forces_local(d2.f)
    d2.torch.cuda.synchronize()
    assert rel_rms(d2.f.cpu().numpy().astype(np.float64), oracle_forces(cfg0).f) <= TOL_F
