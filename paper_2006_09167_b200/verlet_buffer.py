"""Tolerance-based Verlet-buffer estimate (second half).

The paper: "our implementation estimates the Verlet buffer for a given upper bound for the error in the
energy.  The estimate is based on the particle masses, temperature, pair interaction functions and
constraints, also taking into account the cluster setup and its implicit buffering" -- with a default
bound of 0.005 kJ/mol/ps per atom (L161) and, for SPC/E water at rc = 0.9 nm with a 40-step list, a
buffer of 0.218 nm for a particle (1x1) list against 0.105 nm for the 8x4 cluster list (L157).
It prints NO formula (it cites its reference 9), so everything below is a READING, listed in DESIGN.md:

 R1  A pair that is not in the list when it is made (distance r0 >= rlist) contributes nothing until the
     next search.  Over the list lifetime t = (nstlist - 1) dt the two atoms move ballistically; the
     displacement of their separation along the line joining them is Gaussian with variance
     sigma^2 = t^2 kT (1/m_i + 1/m_j)  (free flight, the conservative choice: collisions only slow atoms down).
 R2  Constraints: an atom of a rigid molecule moves with the molecule.  Its thermal velocity variance per
     Cartesian component is kT/M + (kT/3) sum_k (|r|^2 - r_k^2)/I_k (centre-of-mass translation plus
     rigid rotation about the principal axes k), which defines the effective 1/m of R1.  (The paper's
     refinement -- constrained atoms ROTATE around their partner instead of moving linearly, L159 -- only
     tightens this for long lifetimes; linear motion is the upper bound.)
 R3  The energy error of one such pair at the end of the lifetime is |V(r)| (V potential-shifted: V(rc) = 0)
     if it has moved to r < rc.  Per atom of type a, with number densities rho_b and ideal-gas pair statistics:
        dE_a = sum_b rho_b  int_{r0 >= rlist} 4 pi r0^2 (1 - P_listed(r0))  int_{r < rc} |V_ab(r)| G(r - r0; sigma_ab) dr dr0
     and the drift estimate is  (1/2) <dE_a>_atoms / t  (each pair counted once), compared with the tolerance.
 R4  Cluster lists and their IMPLICIT buffer (L153-L157): a pair further apart than rlist is still listed when
     some other atom pair of the two clusters is within rlist.  P_listed(r0) is estimated by seeded Monte Carlo
     for clusters of n_i x n_j atoms filling cubes at the atom density (n_i = n_j = 1: P_listed = 0 beyond rlist,
     the particle list).  This build's inner list is 8 i-atoms x 4-atom half j-clusters, the paper's 8x4.

`verlet_buffer()` returns the smallest rlist (>= rc) whose drift estimate is below the tolerance.
CPU only (numpy); used to choose rlist_outer / rlist_inner, never on the GPU path.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

KB = 0.0083144626  # kJ/mol/K
EPSFAC = 138.935458  # kJ mol^-1 nm e^-2 (reading A2)


@dataclasses.dataclass
class Species:
    """One kind of atom: how many per nm^3, its charge, LJ row index and effective inverse mass (R2)."""
    name: str
    density: float       # atoms / nm^3
    charge: float        # e
    lj_type: int
    inv_mass_eff: float  # mol/g: variance of one velocity component = kT * inv_mass_eff


def rigid_inverse_masses(sites: np.ndarray, masses: np.ndarray) -> np.ndarray:
    """R2: effective 1/m of every site of a rigid molecule (sites [n,3] nm, masses [n] g/mol)."""
    sites = np.asarray(sites, dtype=np.float64)
    masses = np.asarray(masses, dtype=np.float64)
    M = masses.sum()
    r = sites - (masses[:, None] * sites).sum(axis=0) / M
    inertia = np.zeros((3, 3))
    for m, x in zip(masses, r):
        inertia += m * ((x @ x) * np.eye(3) - np.outer(x, x))
    evals, evecs = np.linalg.eigh(inertia)
    rp = r @ evecs                                   # coordinates along the principal axes
    out = np.full(len(masses), 1.0 / M)
    for k in range(3):
        if evals[k] > 1e-12 * max(evals.max(), 1e-300):   # (a linear molecule has one vanishing moment: no rotation about it)
            out += ((rp**2).sum(axis=1) - rp[:, k] ** 2) / (3.0 * evals[k])
    return out


def spce_water(density_molecules: float = 33.4):
    """The paper's workload (SPC/E water; the same numbers as workloads.py): species and the LJ table."""
    from . import workloads as W
    h = W.ANGLE_HOH / 2.0
    sites = np.array([[0.0, 0.0, 0.0], [W.R_OH * math.sin(h), 0.0, W.R_OH * math.cos(h)],
                      [-W.R_OH * math.sin(h), 0.0, W.R_OH * math.cos(h)]])
    inv = rigid_inverse_masses(sites, np.array([15.9994, 1.008, 1.008]))
    species = [Species("OW", density_molecules, W.Q_O, 0, float(inv[0])),
               Species("HW", 2 * density_molecules, W.Q_H, 1, float(inv[1]))]
    return species, W.lj_table(np.array([W.SIGMA_O, 0.0]), np.array([W.EPS_O, 0.0]))


def pair_potential(r, qq, c6, c12, rc, coulomb="ewald", beta=0.0, eps_rf=0.0):
    """|V(r)| of readings A1/A6 with both potential shifts (V(rc) = 0), r < rc."""
    from scipy.special import erfc
    v = c12 * (r**-12 - rc**-12) - c6 * (r**-6 - rc**-6)
    a = EPSFAC * qq
    if coulomb == "ewald":
        v = v + a * (erfc(beta * r) / r - math.erfc(beta * rc) / rc)
    elif coulomb == "rf":
        krf = 1.0 / (2 * rc**3) if (eps_rf <= 0 or math.isinf(eps_rf)) else (eps_rf - 1) / ((2 * eps_rf + 1) * rc**3)
        v = v + a * (1.0 / r + krf * r * r - (1.0 / rc + krf * rc * rc))
    return np.abs(v)


def listed_probability(r0, rlist, n_i, n_j, atom_density, nsample=4000, seed=2006_09167):
    """R4: probability that two atoms r0 apart belong to a listed cluster pair, i.e. that some atom of the
    n_i-cluster holding the first is within rlist of some atom of the n_j-cluster holding the second.
    Clusters are cubes of volume n/density with the atoms uniform inside; seeded Monte Carlo."""
    r0 = np.atleast_1d(np.asarray(r0, dtype=np.float64))
    if n_i == 1 and n_j == 1:
        return (r0 < rlist).astype(np.float64)
    rng = np.random.Generator(np.random.PCG64(seed))
    a_i, a_j = (n_i / atom_density) ** (1 / 3), (n_j / atom_density) ** (1 / 3)
    xi = rng.random((nsample, n_i, 3)) * a_i                       # atom 0 of each cluster is "the" atom of the pair
    xj = rng.random((nsample, n_j, 3)) * a_j
    u = rng.normal(size=(nsample, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    out = np.empty(r0.size)
    for k, r in enumerate(r0):
        shift = xi[:, 0, :] + r * u - xj[:, 0, :]                  # moves the j cluster so that |x_i0 - x_j0| = r
        d = xi[:, :, None, :] - (xj + shift[:, None, :])[:, None, :, :]
        out[k] = ((d**2).sum(-1).min(axis=(1, 2)) < rlist * rlist).mean()
    return out


def drift_estimate(species, lj_c6c12, rlist, rc, nstlist, dt, temperature, coulomb="ewald", beta=0.0, eps_rf=0.0,
                   cluster=(1, 1), ngrid=200, miss_of_delta=None):
    """R3: estimated energy drift, kJ/mol/ps per atom, of a list of radius rlist that lives nstlist steps.
    miss_of_delta = (delta grid, 1 - P_listed) tabulated against r0 - rlist (verlet_buffer tabulates it once:
    the dependence of P_listed on rlist itself at fixed r0 - rlist is second order)."""
    t = max(nstlist - 1, 1) * dt
    kT = KB * temperature
    rho_tot = sum(s.density for s in species)
    sig_max = t * math.sqrt(kT * 2 * max(s.inv_mass_eff for s in species))
    r0 = np.linspace(rlist, rlist + 7 * sig_max + 1e-6, ngrid)
    if miss_of_delta is not None:
        miss = np.interp(r0 - rlist, miss_of_delta[0], miss_of_delta[1], right=1.0)
    else:
        miss = 1.0 - listed_probability(r0, rlist, cluster[0], cluster[1], rho_tot)
    total = 0.0
    for a in species:
        for b in species:
            c6, c12 = (float(v) for v in lj_c6c12[a.lj_type, b.lj_type])
            sigma = t * math.sqrt(kT * (a.inv_mass_eff + b.inv_mass_eff))
            r = np.linspace(max(rc - 7 * sigma, 0.5 * rc), rc, ngrid)
            v = pair_potential(r, a.charge * b.charge, c6, c12, rc, coulomb, beta, eps_rf)
            g = np.exp(-0.5 * ((r[None, :] - r0[:, None]) / sigma) ** 2) / (sigma * math.sqrt(2 * math.pi))
            inner = np.trapezoid(v[None, :] * g, r, axis=1)                       # [r0]
            e_ab = np.trapezoid(4 * math.pi * r0**2 * miss * inner, r0)
            total += a.density * b.density * e_ab
    return 0.5 * total / rho_tot / t


def verlet_buffer(species, lj_c6c12, rc, nstlist, dt=0.002, temperature=298.15, tolerance=0.005, coulomb="ewald",
                  ewald_rtol=1e-5, eps_rf=0.0, cluster=(1, 1), rlist_max=None):
    """Smallest rlist >= rc whose drift estimate is <= tolerance (kJ/mol/ps per atom; PAPER.md L161 default 0.005);
    returns (rlist, drift at rlist).  cluster = (n_i, n_j): (1, 1) particle list, (8, 4) this build's inner list."""
    from scipy.special import erfcinv
    beta = float(erfcinv(ewald_rtol)) / rc if coulomb == "ewald" else 0.0
    tab = None
    if cluster != (1, 1):
        rho_tot = sum(s.density for s in species)
        rl_ref = rc + 0.12
        delta = np.linspace(0.0, 2.2 * (max(cluster) / rho_tot) ** (1 / 3) + 0.05, 48)
        tab = (delta, 1.0 - listed_probability(rl_ref + delta, rl_ref, cluster[0], cluster[1], rho_tot))
    f = lambda rl: drift_estimate(species, lj_c6c12, rl, rc, nstlist, dt, temperature, coulomb, beta, eps_rf, cluster,
                                  miss_of_delta=tab)
    lo, hi = rc, rlist_max if rlist_max is not None else rc + 0.6
    if f(lo) <= tolerance:
        return lo, f(lo)
    if f(hi) > tolerance:
        raise ValueError(f"drift estimate {f(hi):.3g} at rlist = {hi} is still above the tolerance {tolerance}")
    for _ in range(16):
        mid = 0.5 * (lo + hi)
        if f(mid) > tolerance:
            lo = mid
        else:
            hi = mid
    return hi, f(hi)


def dual_list_radii(species, lj_c6c12, rc, nstlist, nstprune, **kw):
    """rlist_outer (lives nstlist steps between searches, cluster criterion of the search: 8x8 bounding boxes are
    at least as inclusive as 8x8 atom distances) and rlist_inner (lives nstprune steps between the prunes of a
    rolling part, 8x4 half-cluster criterion) for the dual list of PAPER.md L193."""
    outer, _ = verlet_buffer(species, lj_c6c12, rc, nstlist, cluster=(8, 8), **kw)
    inner, _ = verlet_buffer(species, lj_c6c12, rc, nstprune, cluster=(8, 4), **kw)
    return outer, min(inner, outer)


if __name__ == "__main__":
    sp, tab = spce_water()
    for cl in ((1, 1), (8, 4)):
        rl, d = verlet_buffer(sp, tab, 0.9, 40, cluster=cl)
        print(f"SPC/E water, rc 0.9 nm, 40-step list, {cl[0]}x{cl[1]}: buffer {rl - 0.9:.3f} nm (drift estimate {d:.2e} kJ/mol/ps/atom)")
