"""Pins of the twin cut-off reading (PME load balancing raises only
the electrostatics cut-off, so rc_coulomb = rc >= rc_vdw): LJ interacts iff r < rc_vdw with its
potential shift taken at rc_vdw; Coulomb keeps rc.  CPU only."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2006_09167_b200 import workloads as W


def test_single_pair_closed_forms():
    rc, rcv = 1.2, 0.9
    beta = O.beta_from_rtol(rc, 1e-5)
    sig, eps = 0.3166, 0.650
    c6, c12 = 4 * eps * sig**6, 4 * eps * sig**12
    qq = -0.8476 * 0.4238
    for coul in ("ewald", "rf"):
        p2 = O.Params(rc=rc, ntypes=1, coulomb=coul, beta=beta, rc_vdw=rcv)
        p1 = O.Params(rc=rc, ntypes=1, coulomb=coul, beta=beta)
        # between the two radii: Coulomb only, identical to the single cut-off Coulomb part
        for r in (0.9, 0.95, 1.19999):
            vlj, vc, flj, fc = O.pair(p2, r, qq, c6, c12, False)
            _, vc1, _, fc1 = O.pair(p1, r, qq, c6, c12, False)
            assert vlj == 0.0 and flj == 0.0 and vc == vc1 and fc == fc1 and vc != 0.0
        # below rc_vdw: LJ with the shift constant taken at rc_vdw (closed form typed here)
        for r in (0.3, 0.5, 0.89999):
            vlj, vc, flj, fc = O.pair(p2, r, qq, c6, c12, False)
            want_v = c12 * (r**-12 - rcv**-12) - c6 * (r**-6 - rcv**-6)
            want_f = 12 * c12 * r**-13 - 6 * c6 * r**-7
            assert vlj == pytest.approx(want_v, rel=1e-13) and flj == pytest.approx(want_f, rel=1e-13)
            _, vc1, _, fc1 = O.pair(p1, r, qq, c6, c12, False)
            assert vc == vc1 and fc == fc1
        # V_lj -> 0 at rc_vdw from below (potential shift), and excluded pairs are untouched
        assert abs(O.pair(p2, rcv * (1 - 1e-12), qq, c6, c12, False)[0]) < 1e-12
        assert O.pair(p2, 0.5, qq, c6, c12, True) == O.pair(p1, 0.5, qq, c6, c12, True)
    # rc_vdw = rc (or <= 0) is the single cut-off, bit for bit
    pa = O.Params(rc=rc, ntypes=1, coulomb="ewald", beta=beta, rc_vdw=rc)
    pb = O.Params(rc=rc, ntypes=1, coulomb="ewald", beta=beta, rc_vdw=0.0)
    for r in (0.4, 0.9, 1.1):
        assert O.pair(pa, r, qq, c6, c12, False) == O.pair(pb, r, qq, c6, c12, False)


@pytest.fixture(scope="module")
def box():
    return W.small_water(60, 1.9, seed=5, rc=0.9, rlist_outer=0.94, rlist_inner=0.92, box_scale=(1.0, 1.05, 1.1))


def _run(w, p, x=None, method="allpairs"):
    return O.forces(w.x if x is None else x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p, method=method)


@pytest.mark.parametrize("coulomb", ["ewald", "rf"])
def test_sums_with_twin_cutoffs(box, coulomb):
    w = box
    rc, rcv = 0.9, 0.7
    beta = O.beta_from_rtol(rc, 1e-5)
    p2 = O.Params(rc=rc, ntypes=2, coulomb=coulomb, beta=beta, rc_vdw=rcv)
    p1 = O.Params(rc=rc, ntypes=2, coulomb=coulomb, beta=beta)
    pv = O.Params(rc=rcv, ntypes=2, coulomb="none")                      # LJ alone at the short cut-off
    a, b, c = _run(w, p2), _run(w, p1), _run(w, pv)
    # Coulomb energy is the single-cut-off one; LJ energy is that of an LJ-only run at rc_vdw
    assert a.e_coul == pytest.approx(b.e_coul, rel=1e-13)
    assert a.e_lj == pytest.approx(c.e_lj, rel=1e-13) and abs(a.e_lj - b.e_lj) > 1e-3 * abs(b.e_lj)
    assert a.npairs == b.npairs and a.npairs_excl == b.npairs_excl     # pair count: within rc (Coulomb range)
    # forces: F(twin) = F(single) - F_lj(rc) + F_lj(rc_vdw), all three from independent runs
    pl = O.Params(rc=rc, ntypes=2, coulomb="none")
    d = _run(w, pl)
    np.testing.assert_allclose(a.f, b.f - d.f + c.f, rtol=0, atol=1e-10 * np.abs(b.f).max())
    np.testing.assert_allclose(a.virial, b.virial - d.virial + c.virial, rtol=0, atol=1e-10 * np.abs(b.virial).max())
    # images brute force and linked cells agree with all-pairs
    for m in ("images",):
        r = _run(w, p2, method=m)
        np.testing.assert_allclose(r.f, a.f, rtol=0, atol=1e-9 * np.abs(a.f).max())
        assert r.energy == pytest.approx(a.energy, rel=1e-12)
    # f = -grad E with both potential shifts (E continuous at both radii)
    rng = np.random.default_rng(3)
    x = w.x.astype(np.float64)
    h = 1e-5
    frms = np.sqrt((a.f**2).mean())
    worst = 0.0
    for _ in range(40):
        i, k = int(rng.integers(w.natoms)), int(rng.integers(3))
        xp, xm = x.copy(), x.copy()
        xp[i, k] += h
        xm[i, k] -= h
        fd = -(_run(w, p2, x=xp).energy - _run(w, p2, x=xm).energy) / (2 * h)
        worst = max(worst, abs(fd - a.f[i, k]) / max(abs(a.f[i, k]), frms))
    assert worst < 1e-6, worst
    # Newton
    assert np.linalg.norm(a.f.sum(axis=0)) / (w.natoms * frms) < 1e-12
