"""Pins T5-T9, T14, T15 of the oracle's pair sums.  CPU only."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2006_09167_b200 import workloads as W


def _params(w, **kw):
    beta = O.beta_from_rtol(w.rc, w.ewald_rtol) if w.coulomb == "ewald" else 0.0
    return O.Params(rc=w.rc, ntypes=w.ntypes, coulomb=w.coulomb, beta=beta, **kw)


def _run(w, p, x=None, method="allpairs", box=None, excl=None):
    eo, ei = (w.excl_off, w.excl_idx) if excl is None else excl
    return O.forces(w.x if x is None else x, w.q, w.type, w.box if box is None else box, w.lj_c6c12,
                    eo, ei, p, method=method)


@pytest.fixture(scope="module", params=["ewald", "rf"])
def tiny(request):
    # 20 molecules = 60 atoms, rectangular box, rc <= L/2
    return W.small_water(20, 1.25, seed=11, rc=0.6, rlist_outer=0.62, rlist_inner=0.61,
                         box_scale=(1.0, 1.1, 1.2), coulomb=request.param)


def test_t5_image_brute_force_equals_minimum_image(tiny):
    p = _params(tiny)
    a = _run(tiny, p, method="allpairs")
    b = _run(tiny, p, method="images")
    assert a.npairs == b.npairs and a.npairs_excl == b.npairs_excl and a.npairs > 300
    np.testing.assert_allclose(a.f, b.f, rtol=0, atol=1e-9 * np.abs(a.f).max())
    assert a.energy == pytest.approx(b.energy, rel=1e-12)
    np.testing.assert_allclose(a.virial, b.virial, rtol=0, atol=1e-9 * np.abs(a.virial).max())


def test_t6_newton(cfg0):
    r = _run(cfg0, _params(cfg0))
    frms = np.sqrt((r.f**2).sum(axis=1).mean())
    assert np.linalg.norm(r.f.sum(axis=0)) / (cfg0.natoms * frms) < 1e-12


def test_t7_translation_and_box_vector_invariance(cfg0):
    w = cfg0
    p = _params(w)
    base = _run(w, p)
    rng = np.random.default_rng(5)
    box = w.box.astype(np.float64)
    x = w.x.astype(np.float64)
    # (a) translate everything by a random vector, re-wrap atom by atom
    xt = np.mod(x + rng.uniform(-3, 3, size=3), box)
    # (b) add integer box vectors to random individual atoms (breaks molecules across images)
    xb = x + rng.integers(-2, 3, size=x.shape) * box
    for xx in (xt, xb):
        r = _run(w, p, x=xx)
        assert r.npairs == base.npairs
        np.testing.assert_allclose(r.f, base.f, rtol=0, atol=1e-10 * np.abs(base.f).max())
        assert r.energy == pytest.approx(base.energy, rel=1e-10)
        np.testing.assert_allclose(r.virial, base.virial, rtol=0, atol=1e-9 * np.abs(base.virial).max())


@pytest.mark.parametrize("coulomb", ["ewald", "rf"])
def test_t8_finite_differences(cfg0, coulomb):
    """f = -grad E on random (i,k) of config 0; E is continuous at rc only with pot-shift."""
    w = cfg0
    p = O.Params(rc=w.rc, ntypes=2, coulomb=coulomb, beta=O.beta_from_rtol(w.rc, 1e-5))
    base = _run(w, p)
    rng = np.random.default_rng(7)
    x = w.x.astype(np.float64)
    h = 1e-5
    frms = np.sqrt((base.f**2).mean())
    worst = 0.0
    for _ in range(100):
        i, k = int(rng.integers(w.natoms)), int(rng.integers(3))
        xp, xm = x.copy(), x.copy()
        xp[i, k] += h
        xm[i, k] -= h
        fd = -(_run(w, p, x=xp).energy - _run(w, p, x=xm).energy) / (2 * h)
        worst = max(worst, abs(fd - base.f[i, k]) / max(abs(base.f[i, k]), frms))
    assert worst < 1e-6, worst


def test_t9_virial_identities(tiny):
    w = tiny
    p = _params(w)
    base = _run(w, p)
    # (a) pair-sum virial == shift-force identity (reading A8)
    vs = O.virial_shift_identity(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p)
    np.testing.assert_allclose(vs, base.virial, rtol=0, atol=1e-10 * np.abs(base.virial).max())
    # symmetric for central forces
    np.testing.assert_allclose(base.virial, base.virial.T, rtol=0, atol=1e-10 * np.abs(base.virial).max())
    # (b) scaling: dE/dln(lambda) at lambda = 1 (rc fixed) == 2 tr(Xi); needs E continuous at rc
    lam = 1e-6
    x, box = w.x.astype(np.float64), w.box.astype(np.float64)
    ep = _run(w, p, x=x * (1 + lam), box=box * (1 + lam)).energy
    em = _run(w, p, x=x * (1 - lam), box=box * (1 - lam)).energy
    assert (ep - em) / (2 * lam) == pytest.approx(2 * np.trace(base.virial), rel=2e-6)


def test_cells_equals_allpairs(cfg1):
    p = _params(cfg1)
    a = _run(cfg1, p, method="allpairs")
    c = _run(cfg1, p, method="cells")
    assert a.npairs == c.npairs and a.npairs_excl == c.npairs_excl
    np.testing.assert_allclose(a.f, c.f, rtol=0, atol=1e-12 * np.abs(a.f).max())
    assert a.energy == pytest.approx(c.energy, rel=1e-12)
    np.testing.assert_allclose(a.virial, c.virial, rtol=0, atol=1e-11 * np.abs(a.virial).max())
    # T14: non-excluded pairs within rc ~ N (2 pi/3) rc^3 rho for jittered-lattice water
    rho = cfg1.natoms / float(np.prod(cfg1.box.astype(np.float64)))
    ideal = cfg1.natoms * (2 * np.pi / 3) * cfg1.rc**3 * rho
    assert abs(a.npairs - ideal) / ideal < 0.02
    # independent count with a library k-d tree (all pairs within rc, minus the 3 per molecule)
    from scipy.spatial import cKDTree
    box = cfg1.box.astype(np.float64)
    t = cKDTree(np.mod(cfg1.x.astype(np.float64), box), boxsize=box)
    assert t.count_neighbors(t, cfg1.rc * (1 - 1e-9)) == 2 * (a.npairs + a.npairs_excl) + cfg1.natoms
    assert a.npairs_excl == cfg1.natoms  # 3 intramolecular pairs per molecule, all within rc


def test_t15_exclusion_extremes(tiny):
    w = tiny
    p = _params(w)
    n = w.natoms
    # no exclusions: plain pair sum -> equals sum over pairs of the interacting formula
    none = (np.zeros(n + 1, dtype=np.int32), np.zeros(0, dtype=np.int32))
    r0 = _run(w, p, excl=none)
    assert r0.npairs_excl == 0
    # all-excluded topology: E_lj = 0, only Coulomb corrections
    full_off = (np.arange(n + 1) * (n - 1)).astype(np.int32)
    full_idx = np.concatenate([np.delete(np.arange(n), i) for i in range(n)]).astype(np.int32)
    r1 = _run(w, p, excl=(full_off, full_idx))
    assert r1.npairs == 0 and r1.e_lj == 0.0 and r1.npairs_excl == r0.npairs
    # difference between the two = bare (unsplit) interaction: for Ewald, A/r - shift + LJ
    x = w.x.astype(np.float64)
    box = w.box.astype(np.float64)
    d = x[:, None, :] - x[None, :, :]
    d -= box * np.rint(d / box)
    r = np.sqrt((d**2).sum(-1))
    iu = np.triu_indices(n, 1)
    within = r[iu] < w.rc
    qq = (w.q.astype(np.float64)[:, None] * w.q.astype(np.float64)[None, :])[iu][within]
    rr = r[iu][within]
    if w.coulomb == "ewald":
        import math
        sh = math.erfc(p.beta * w.rc) / w.rc
        expect = (O.EPSFAC * qq * (1 / rr - sh)).sum()
    else:
        expect = (O.EPSFAC * qq / rr).sum()
    assert r0.e_coul - r1.e_coul == pytest.approx(expect, rel=1e-10)


def test_water_exclusions_change_only_intramolecular_terms(tiny):
    """Sanity on is_excluded/CSR handling: with water exclusions, E differs from the
    no-exclusion sum exactly by the intramolecular bare terms."""
    w = tiny
    p = _params(w)
    n = w.natoms
    none = (np.zeros(n + 1, dtype=np.int32), np.zeros(0, dtype=np.int32))
    r0, r1 = _run(w, p, excl=none), _run(w, p)
    assert r1.npairs_excl == n and r0.npairs - r1.npairs == n
