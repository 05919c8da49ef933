"""Verlet-buffer estimate.  The paper prints no formula, only two numbers
for SPC/E water (rc 0.9 nm, 40-step list, default tolerance): 0.218 nm for the 1x1 list, 0.105 nm for 8x4.
Those pin the ORDER OF MAGNITUDE of this reading; the rest are properties any such estimate has.  CPU only."""
import numpy as np
import pytest

from paper_2006_09167_b200 import verlet_buffer as VB


@pytest.fixture(scope="module")
def water():
    return VB.spce_water()


def test_paper_numbers_order_of_magnitude(water):
    sp, tab = water
    b11 = VB.verlet_buffer(sp, tab, 0.9, 40, cluster=(1, 1))[0] - 0.9
    b84 = VB.verlet_buffer(sp, tab, 0.9, 40, cluster=(8, 4))[0] - 0.9
    assert 0.5 * 0.218 < b11 < 2.0 * 0.218          # 0.218 nm
    assert 0.5 * 0.105 < b84 < 2.0 * 0.105          # 0.105 nm
    assert b84 < 0.8 * b11                          # the implicit buffer of the cluster list (L153-L157)


def test_monotone_in_lifetime_tolerance_temperature(water):
    sp, tab = water
    b = lambda **kw: VB.verlet_buffer(sp, tab, 1.0, **{"nstlist": 40, **kw})[0]
    assert b(nstlist=10) < b(nstlist=20) < b(nstlist=40)
    assert b(tolerance=0.05) < b(tolerance=0.005) < b(tolerance=0.0005)
    assert b(temperature=200.0) < b(temperature=400.0)
    # the drift estimate at the returned radius meets the tolerance, and just inside it does not
    rl, d = VB.verlet_buffer(sp, tab, 1.0, 40)
    assert d <= 0.005
    from scipy.special import erfcinv
    beta = float(erfcinv(1e-5)) / 1.0
    assert VB.drift_estimate(sp, tab, rl - 0.01, 1.0, 40, 0.002, 298.15, "ewald", beta) > 0.005
    # a one-step list needs no buffer at all
    assert VB.verlet_buffer(sp, tab, 1.0, 1)[0] == pytest.approx(1.0, abs=0.02)


def test_rigid_effective_masses():
    # a free atom: its own mass.  A rigid dumbbell of two equal masses m at +-d/2: translation 1/(2m) plus
    # rotation about the two axes perpendicular to the bond, each I = m d^2 / 2: (1/3)(2 (d/2)^2 / I) = 1/(3m)
    assert VB.rigid_inverse_masses(np.zeros((1, 3)), np.array([12.0]))[0] == pytest.approx(1 / 12.0)
    inv = VB.rigid_inverse_masses(np.array([[0, 0, -0.05], [0, 0, 0.05]]), np.array([7.0, 7.0]))
    assert inv == pytest.approx([1 / 14.0 + 1 / 21.0] * 2)
    # water: H is light but rides on the molecule; between the free-H and the whole-molecule values
    sp, _ = VB.spce_water()
    assert 1 / 18.0152 < sp[0].inv_mass_eff < 1 / 15.9994 and 1 / 18.0152 < sp[1].inv_mass_eff < 1 / 1.008


def test_listed_probability_limits():
    r0 = np.array([0.5, 0.99, 1.01, 1.2, 2.5])
    assert VB.listed_probability(r0, 1.0, 1, 1, 100.0).tolist() == [1, 1, 0, 0, 0]
    p = VB.listed_probability(r0, 1.0, 8, 4, 100.0)
    assert p[0] == 1.0 and p[1] == 1.0 and 0.3 < p[2] <= 1.0 and p[2] >= p[3] >= p[4] and p[4] == 0.0
    p88 = VB.listed_probability(r0, 1.0, 8, 8, 100.0)
    assert (p88 >= p - 0.03).all()                  # larger clusters list more


def test_dual_list_radii(water):
    sp, tab = water
    outer, inner = VB.dual_list_radii(sp, tab, 1.0, nstlist=40, nstprune=4)
    assert 1.0 <= inner < outer < 1.3
