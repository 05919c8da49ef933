"""nb_forces_static (include/nb.h): nb_forces with the force kernel's scratch in a static device array of the library,
for callers that cannot call cudaMalloc.  Checked against the existing path (nb_forces) on the same context and the same
lists, two calls in a row and with contexts of different sizes sharing the array.  Collected last on purpose (zz): the
suite runs with -x.  Must pass alone in a fresh process and after the other GPU tests."""
import numpy as np
import pytest

from tests.gpu_util import Driver, oracle_forces, rel_rms

pytestmark = pytest.mark.gpu

# nb_forces_static runs the same kernels on the same list: the two paths differ by the order of the fp32 atomic adds only
# (the bound the suite uses for nb_step against the three calls); energies are fp64 sums of the same fp32 partials
F_TOL, E_TOL, V_TOL = 2e-6, 1e-9, 1e-5


def forces_static(d, energy=False, virial=False):
    d.f.fill_(float("nan"))
    if energy:
        d.e.fill_(float("nan"))
    if virial:
        d.v.fill_(float("nan"))
    d.ctx.forces_static(d.f, d.e if energy else None, d.v if virial else None)
    d.torch.cuda.synchronize()
    out = [d.f.cpu().numpy().astype(np.float64)]
    if energy:
        out.append(d.e.cpu().numpy().copy())
    if virial:
        out.append(d.v.cpu().numpy().reshape(3, 3).copy())
    return out[0] if len(out) == 1 else tuple(out)


def check_same(got, ref):
    f, e, v = got
    f0, e0, v0 = ref
    assert np.isfinite(f).all() and np.isfinite(e).all() and np.isfinite(v).all()
    assert rel_rms(f, f0) <= F_TOL
    assert np.all(np.abs(e - e0) <= E_TOL * np.abs(e0).sum())
    assert np.linalg.norm(v - v0) <= V_TOL * np.linalg.norm(v0)


def moved(w, t):
    return (w.x.astype(np.float64) + t * 2.5e-4 * w.unit_dir[w.mol_of_atom]).astype(np.float32)


def test_static_scratch_matches_nb_forces(cfg0, cfg1):
    d1 = Driver(cfg1)
    d1.put()
    d1.ctx.search(cfg1.rlist_outer)
    d1.ctx.prune(cfg1.rlist_inner, 0, 1)
    ref1 = d1.forces(energy=True, virial=True)
    # two calls in a row on the larger system: F+E+virial, then force-only; the second starts from what the first left
    check_same(forces_static(d1, True, True), ref1)
    f = forces_static(d1)
    assert np.isfinite(f).all() and rel_rms(f, ref1[0]) <= F_TOL
    check_same(forces_static(d1, True, True), ref1)

    # a smaller context on the same device shares the array (it holds the larger system's last state)
    d0 = Driver(cfg0)
    d0.put()
    d0.ctx.search(cfg0.rlist_outer)
    d0.ctx.prune(cfg0.rlist_inner, 0, 1)
    ref0 = d0.forces(energy=True, virial=True)
    check_same(forces_static(d0, True, True), ref0)
    check_same(forces_static(d0, True, True), ref0)
    ref = oracle_forces(cfg0)
    f, e, v = forces_static(d0, True, True)
    assert rel_rms(f, ref.f) <= 1e-5
    assert abs(e.sum() - ref.energy) <= 1e-5 * abs(ref.energy)
    assert np.linalg.norm(v - ref.virial) <= 1e-5 * np.linalg.norm(ref.virial)

    # back to the larger one, on a moved frame after a rolling prune, interleaved with the existing path
    x = moved(cfg1, 7)
    d1.put(x)
    d1.ctx.prune(cfg1.rlist_inner, 1, 2)
    got = forces_static(d1, True, True)
    ref = d1.forces(energy=True, virial=True)
    check_same(got, ref)
    check_same(forces_static(d1, True, True), ref)
    # the existing path's own accumulator is untouched by the static calls
    check_same(d1.forces(energy=True, virial=True), ref)


def test_static_scratch_flavours():
    from paper_2006_09167_b200 import workloads
    for coulomb in ("rf", "none"):
        w = workloads.small_water(150, 2.0, seed=21, rc=0.8, rlist_outer=0.9, rlist_inner=0.84, coulomb=coulomb) \
            if coulomb == "rf" else workloads.lj_fluid(12, rc=0.9)
        d = Driver(w)
        d.put()
        d.ctx.search(w.rlist_outer)
        d.ctx.prune(w.rlist_inner, 0, 1)
        ref = d.forces(energy=True, virial=True)
        check_same(forces_static(d, True, True), ref)
        check_same(forces_static(d, True, True), ref)


def test_static_scratch_rejects_large_systems_and_bad_calls(cfg0):
    from paper_2006_09167_b200 import nb, workloads
    d = Driver(cfg0)
    d.put()
    with pytest.raises(nb.NbError) as ei:       # no list yet
        d.ctx.forces_static(d.f)
    assert ei.value.code == -2     # NB_ERR_STATE
    d.ctx.search(cfg0.rlist_outer)
    with pytest.raises(nb.NbError) as ei:       # virial without energies
        d.ctx.forces_static(d.f, None, d.v)
    assert ei.value.code == -1     # NB_ERR_ARG

    w = workloads.lj_fluid(nside=64, rc=0.7, buffer_outer=0.05, buffer_inner=0.02)   # 262 144 atoms: beyond the limit
    big = Driver(w)
    big.put()
    big.ctx.search(w.rlist_outer)
    big.ctx.prune(w.rlist_inner, 0, 1)
    ref = big.forces()
    big.f.fill_(123.0)
    with pytest.raises(nb.NbError) as ei:
        big.ctx.forces_static(big.f)
    assert ei.value.code == -7     # NB_ERR_OVERFLOW
    assert "NB_STATIC_MAX_SLOTS" in str(ei.value)
    big.torch.cuda.synchronize()
    assert float(big.f.min()) == 123.0 and float(big.f.max()) == 123.0   # the rejected call did nothing
    assert rel_rms(big.forces(), ref) <= F_TOL                           # and the context still works
    # the small context still does, right after the rejection
    d.ctx.prune(cfg0.rlist_inner, 0, 1)
    refs = d.forces(energy=True, virial=True)
    check_same(forces_static(d, True, True), refs)
