"""Pins of the oracle's LJ-only flavour (coulomb = "none", PAPER.md L167-L171:
the Lennard-Jones workload of Fig. 6).  Chosen so that a wrong reading of "charges are ignored"
(a leftover Coulomb term, a dropped LJ shift, a sign) fails one of them."""
import numpy as np

from oracle import oracle as O
from paper_2006_09167_b200 import workloads as W


def _run(w, p, x=None, q=None):
    return O.forces(w.x if x is None else x, w.q if q is None else q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p)


def test_none_equals_ewald_and_rf_with_zero_charges():
    """Water box: LJ-only == Ewald or RF evaluated with every charge set to zero; E_coul == 0 exactly."""
    w = W.config0()
    none = _run(w, O.Params(rc=w.rc, ntypes=2, coulomb="none"))
    q0 = np.zeros_like(w.q)
    for coul in ("ewald", "rf"):
        ref = _run(w, O.Params(rc=w.rc, ntypes=2, coulomb=coul, beta=O.beta_from_rtol(w.rc, 1e-5)), q=q0)
        assert np.abs(none.f - ref.f).max() <= 1e-12 * np.abs(ref.f).max()
        assert abs(none.e_lj - ref.e_lj) <= 1e-12 * abs(ref.e_lj)
        assert np.abs(none.virial - ref.virial).max() <= 1e-12 * np.abs(ref.virial).max()
    assert none.e_coul == 0.0
    # and the charges really are ignored: the charged water box gives the same LJ-only result
    assert none.npairs > 0 and np.isfinite(none.f).all()


def test_two_atom_closed_form():
    """Two LJ atoms at the minimum 2^(1/6) sigma: zero force, E = -eps - V_lj(rc) (potential shift)."""
    sig, eps, rc, L = W.LJ_SIGMA, W.LJ_EPS, 1.0, 4.0
    tab = W.lj_table(np.array([sig]), np.array([eps]))
    r = 2.0 ** (1.0 / 6.0) * sig
    x = np.array([[1.0, 1.0, 1.0], [1.0 + r, 1.0, 1.0]])
    res = O.forces(x, np.array([0.7, -0.7]), np.zeros(2, np.int32), np.full(3, L), tab, np.zeros(3, np.int32),
                   np.zeros(0, np.int32), O.Params(rc=rc, ntypes=1, coulomb="none"))
    c6, c12 = float(tab[0, 0, 0]), float(tab[0, 0, 1])
    shift = c12 / rc**12 - c6 / rc**6
    frms_scale = 24 * eps / sig
    assert np.abs(res.f).max() < 1e-6 * frms_scale          # table is fp32: c6, c12 carry 6e-8 relative error
    assert abs(res.e_lj - (-eps - shift)) < 1e-6 * eps
    assert res.e_coul == 0.0
    # a little closer the pair repels along x, equal and opposite
    x[1, 0] -= 0.02
    res = O.forces(x, np.zeros(2), np.zeros(2, np.int32), np.full(3, L), tab, np.zeros(3, np.int32),
                   np.zeros(0, np.int32), O.Params(rc=rc, ntypes=1, coulomb="none"))
    assert res.f[0, 0] < 0 < res.f[1, 0] and abs(res.f[0, 0] + res.f[1, 0]) < 1e-12 * abs(res.f[0, 0])


def test_lj_fluid_finite_differences_newton_and_pair_count():
    w = W.lj_fluid(8, rc=0.9)
    p = O.Params(rc=w.rc, ntypes=1, coulomb="none")
    base = _run(w, p)
    frms = np.sqrt((base.f**2).mean())
    assert np.abs(base.f.sum(axis=0)).max() < 1e-10 * frms * w.natoms
    # pairs within rc ~ N (2 pi / 3) rc^3 rho for a near-uniform fluid
    ideal = w.natoms * (2 * np.pi / 3) * w.rc**3 * W.LJ_RHO
    assert abs(base.npairs - ideal) / ideal < 0.03
    rng = np.random.default_rng(11)
    x = w.x.astype(np.float64)
    h, worst = 1e-5, 0.0
    for _ in range(40):
        i, k = int(rng.integers(w.natoms)), int(rng.integers(3))
        xp, xm = x.copy(), x.copy()
        xp[i, k] += h
        xm[i, k] -= h
        fd = -(_run(w, p, x=xp).energy - _run(w, p, x=xm).energy) / (2 * h)
        worst = max(worst, abs(fd - base.f[i, k]) / max(abs(base.f[i, k]), frms))
    assert worst < 1e-6, worst
