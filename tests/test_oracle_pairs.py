"""Pins T1-T4 of the oracle's per-pair formulas.  CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SIGMA, EPS = 0.3166, 0.650
C6 = 4 * EPS * SIGMA**6
C12 = 4 * EPS * SIGMA**12


def _constants():
    out = {}
    for line in open(os.path.join(GOLD, "constants.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = float(v)
    return out


def _params(coulomb, rc, **kw):
    beta = O.beta_from_rtol(rc, 1e-5) if coulomb == "ewald" else 0.0
    return O.Params(rc=rc, ntypes=2, coulomb=coulomb, beta=beta, **kw)


def test_t1_golden_single_pairs():
    n = 0
    for line in open(os.path.join(GOLD, "t1_single_pairs.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, coul, rc, r, qi, qj, ex, V, F = line.split()
        p = _params(coul, float(rc))
        vlj, vc, flj, fc = O.pair(p, float(r), float(qi) * float(qj), C6, C12, bool(int(ex)))
        got = (vlj, flj) if kind == "lj" else (vc, fc)
        assert got[0] == pytest.approx(float(V), rel=2e-9, abs=1e-9), line
        assert got[1] == pytest.approx(float(F), rel=2e-9, abs=1e-9), line
        n += 1
    assert n == 9


def test_t2_lj_closed_forms():
    c = _constants()
    assert C6 == pytest.approx(c["c6_OO"], rel=1e-9)
    assert C12 == pytest.approx(c["c12_OO"], rel=1e-9)
    p_ns = _params("ewald", 0.9, lj_shift=False)
    # unshifted V(sigma) = 0
    assert O.pair(p_ns, SIGMA, 0.0, C6, C12, False)[0] == pytest.approx(0.0, abs=1e-12)
    # minimum at 2^(1/6) sigma, depth -eps, zero force
    rmin = 2 ** (1 / 6) * SIGMA
    assert rmin == pytest.approx(c["lj_min_r"], abs=1e-6)
    v, _, f, _ = O.pair(p_ns, rmin, 0.0, C6, C12, False)
    assert v == pytest.approx(c["lj_min_depth"], rel=1e-12)
    assert f == pytest.approx(0.0, abs=1e-10)
    for rc, key in ((0.9, "lj_shift_rc0.9"), (1.0, "lj_shift_rc1.0"), (1.2, "lj_shift_rc1.2")):
        p = _params("ewald", rc)
        # shifted V(sigma) = -V_lj(rc);  V_shift(rc-) = 0
        assert O.pair(p, SIGMA, 0.0, C6, C12, False)[0] == pytest.approx(-c[key], rel=2e-8)
        assert O.pair(p, rc * (1 - 1e-12), 0.0, C6, C12, False)[0] == pytest.approx(0.0, abs=1e-12)
    # force is unaffected by the shift
    assert O.pair(_params("ewald", 0.9), 0.31, 0.0, C6, C12, False)[2] == \
        O.pair(p_ns, 0.31, 0.0, C6, C12, False)[2]
    # excluded pair: no LJ at all
    assert O.pair(_params("ewald", 0.9), 0.31, 0.0, C6, C12, True)[0::2] == (0.0, 0.0)


def test_t3_rf_and_ewald_limits():
    c = _constants()
    A = O.EPSFAC * 0.3
    # eps_rf = inf: V(rc) = 0, F(rc) = 0
    for rc, kk, ck in ((1.2, "krf_rc1.2", "crf_rc1.2"), (1.0, "krf_rc1.0", "crf_rc1.0")):
        p = _params("rf", rc)
        _, v, _, f = O.pair(p, rc, 0.3, 0, 0, False)
        assert v == pytest.approx(0.0, abs=1e-12) and f == pytest.approx(0.0, abs=1e-12)
        # V = A (1/r + k r^2 - c) at r = 0.5 from the golden constants
        _, v, _, f = O.pair(p, 0.5, 0.3, 0, 0, False)
        assert v == pytest.approx(A * (2.0 + c[kk] * 0.25 - c[ck]), rel=1e-9)
        assert f == pytest.approx(A * (4.0 - 2 * c[kk] * 0.5), rel=1e-9)
    # eps_rf = 1 -> k_rf = 0 -> shifted plain Coulomb
    p1 = _params("rf", 1.0, eps_rf=1.0)
    _, v, _, f = O.pair(p1, 0.4, 0.3, 0, 0, False)
    assert v == pytest.approx(A * (1 / 0.4 - 1 / 1.0), rel=1e-12)
    assert f == pytest.approx(A / 0.16, rel=1e-12)
    # Ewald beta -> 0: plain Coulomb A/r, excluded correction -> 0
    p0 = O.Params(rc=1.0, ntypes=2, coulomb="ewald", beta=1e-9, coul_shift=False)
    _, v, _, f = O.pair(p0, 0.4, 0.3, 0, 0, False)
    assert v == pytest.approx(A / 0.4, rel=1e-8) and f == pytest.approx(A / 0.16, rel=1e-8)
    _, v, _, f = O.pair(p0, 0.4, 0.3, 0, 0, True)
    assert abs(v) < 1e-6 and abs(f) < 1e-6
    # interacting minus excluded Ewald = full Coulomb (erfc + erf = 1), any beta
    p = _params("ewald", 1.0, coul_shift=False)
    _, v1, _, f1 = O.pair(p, 0.37, 0.3, 0, 0, False)
    _, v0, _, f0 = O.pair(p, 0.37, 0.3, 0, 0, True)
    assert v1 - v0 == pytest.approx(A / 0.37, rel=1e-12)
    assert f1 - f0 == pytest.approx(A / 0.37**2, rel=1e-12)
    # Ewald shift makes V vanish at rc
    ps = _params("ewald", 1.0)
    assert O.pair(ps, 1.0, 0.3, 0, 0, False)[1] == pytest.approx(0.0, abs=1e-12)


def test_t4_beta():
    c = _constants()
    for rc, key in ((0.9, "beta_rc0.9"), (1.0, "beta_rc1.0")):
        b = O.beta_from_rtol(rc, 1e-5)
        assert math.erfc(b * rc) == pytest.approx(1e-5, rel=1e-10)
        assert b == pytest.approx(c[key], rel=1e-10)
        assert b * rc == pytest.approx(c["erfcinv_1e-5"], rel=1e-12)


def test_pair_force_is_minus_derivative():
    """Radial force = -dV/dr for every row of the formula table (central difference)."""
    h = 1e-6
    for coul, rc in (("ewald", 0.9), ("rf", 1.2)):
        p = _params(coul, rc)
        for ex in (False, True):
            for r in (0.12, 0.3, 0.7, rc - 0.01):
                vp = O.pair(p, r + h, -0.36, C6, C12, ex)
                vm = O.pair(p, r - h, -0.36, C6, C12, ex)
                v0 = O.pair(p, r, -0.36, C6, C12, ex)
                assert v0[2] == pytest.approx(-(vp[0] - vm[0]) / (2 * h), rel=1e-6, abs=1e-7)
                assert v0[3] == pytest.approx(-(vp[1] - vm[1]) / (2 * h), rel=1e-6, abs=1e-7)
