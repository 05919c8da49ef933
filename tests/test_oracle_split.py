"""Pins of the local / non-local split oracle ("splitting non-bonded work into two
kernels: one for local-only interactions and one for interactions that involve non-local particles"; reading A25).
CPU only.  The split is pinned to things other than itself: the all-pairs definition (already pinned), the all-pairs
sum of the local atoms ALONE (a different system handed to a different function), and a numpy pair loop."""
import numpy as np

from oracle import oracle as O
from paper_2006_09167_b200 import workloads as W
from tests.splitutil import local_first


def params(w):
    beta = O.beta_from_rtol(w.rc, w.ewald_rtol) if w.coulomb == "ewald" else 0.0
    return O.Params(rc=w.rc, ntypes=w.ntypes, coulomb=w.coulomb, beta=beta)


def split(w, nlocal, which):
    return O.forces_split(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, params(w), nlocal, which)


def test_parts_sum_to_the_whole_and_local_part_is_the_local_system_alone():
    for coul in ("ewald", "rf"):
        w0 = W.small_water(120, 1.9, seed=5, rc=0.8, rlist_outer=0.9, rlist_inner=0.85, coulomb=coul)
        w, nlocal = local_first(w0, lambda x: x[:, 0] < 0.55 * w0.box[0])
        assert 0 < nlocal < w.natoms and nlocal % 3 == 0
        p = params(w)
        whole = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p)
        # reordering the atoms does not change the physics (the helper keeps molecules and exclusions together)
        ref0 = O.forces(w0.x, w0.q, w0.type, w0.box, w0.lj_c6c12, w0.excl_off, w0.excl_idx, p)
        assert abs(whole.energy - ref0.energy) < 1e-9 * abs(ref0.energy) and whole.npairs == ref0.npairs
        loc, nl, al = split(w, nlocal, 1), split(w, nlocal, 2), split(w, nlocal, 0)
        scale = np.abs(whole.f).max()
        assert np.abs(al.f - whole.f).max() < 1e-12 * scale and al.npairs == whole.npairs
        assert np.abs(loc.f + nl.f - whole.f).max() < 1e-11 * scale
        assert abs(loc.e_lj + nl.e_lj - whole.e_lj) < 1e-11 * abs(whole.e_lj)
        assert abs(loc.e_coul + nl.e_coul - whole.e_coul) < 1e-11 * abs(whole.e_coul)
        assert np.abs(loc.virial + nl.virial - whole.virial).max() < 1e-11 * np.abs(whole.virial).max()
        assert loc.npairs + nl.npairs == whole.npairs and loc.npairs_excl + nl.npairs_excl == whole.npairs_excl
        assert loc.npairs > 1000 and nl.npairs > 1000
        # the local part is the force field of the local atoms alone in the same periodic box
        eo = w.excl_off[: nlocal + 1]
        alone = O.forces(w.x[:nlocal], w.q[:nlocal], w.type[:nlocal], w.box, w.lj_c6c12, eo, w.excl_idx[: eo[-1]], p)
        assert np.abs(loc.f[:nlocal] - alone.f).max() < 1e-12 * scale and np.all(loc.f[nlocal:] == 0.0)
        assert abs(loc.energy - alone.energy) < 1e-12 * abs(alone.energy) and loc.npairs == alone.npairs
        assert np.abs(loc.virial - alone.virial).max() < 1e-12 * np.abs(alone.virial).max()
        # the non-local part obeys Newton's third law on its own, and touches local atoms only through halo partners
        assert np.abs(nl.f.sum(0)).max() < 1e-9 * scale


def test_nonlocal_part_against_a_numpy_pair_loop():
    """LJ only, tiny: the non-local part retyped as a plain loop over the pairs that involve a halo atom."""
    w = W.lj_fluid(6, rc=0.7)
    n = w.natoms
    nlocal = 130
    nl = split(w, nlocal, 2)
    c6, c12 = float(w.lj_c6c12[0, 0, 0]), float(w.lj_c6c12[0, 0, 1])
    x = w.x.astype(np.float64)
    L = w.box.astype(np.float64)
    f = np.zeros((n, 3))
    e = 0.0
    cnt = 0
    for i in range(n):
        for j in range(max(i + 1, nlocal), n):        # j >= nlocal or i >= nlocal  <=>  j >= nlocal (j > i)
            d = x[i] - x[j]
            d -= L * np.rint(d / L)
            r2 = float(d @ d)
            if r2 >= w.rc**2:
                continue
            r6 = r2**-3
            e += c12 * (r6 * r6 - w.rc**-12) - c6 * (r6 - w.rc**-6)
            fr = (12 * c12 * r6 * r6 - 6 * c6 * r6) / r2
            f[i] += fr * d
            f[j] -= fr * d
            cnt += 1
    assert cnt == nl.npairs and cnt > 500
    assert np.abs(nl.f - f).max() < 1e-10 * np.abs(f).max()
    assert abs(nl.e_lj - e) < 1e-10 * abs(e) and nl.e_coul == 0.0


def test_degenerate_splits():
    w = W.config0()
    p = params(w)
    whole = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p)
    n = w.natoms
    all_local, none_nl = split(w, n, 1), split(w, n, 2)
    assert np.abs(all_local.f - whole.f).max() < 1e-12 * np.abs(whole.f).max() and all_local.npairs == whole.npairs
    assert none_nl.npairs == 0 and np.all(none_nl.f == 0.0) and none_nl.energy == 0.0
    none_local, all_nl = split(w, 0, 1), split(w, 0, 2)
    assert none_local.npairs == 0 and np.all(none_local.f == 0.0)
    assert all_nl.npairs == whole.npairs and np.abs(all_nl.f - whole.f).max() < 1e-12 * np.abs(whole.f).max()
