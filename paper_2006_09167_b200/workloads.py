"""Seeded synthetic inputs for the cluster-pair non-bonded path.

This module serves BOTH the CUDA path and the CPU oracle (tests hand its arrays to
each side).  It holds none of the method's arithmetic: only positions, charges,
types, the LJ parameter table and the exclusion topology of water-like boxes.

The paper's water workloads are SPC/E boxes (Fig. 7 caption
L179); its benchmark inputs live on Zenodo and are not available
here, so these generators stand in for them with the same shape: rigid 3-site
water at liquid density, fp32 positions, intramolecular exclusions
(BASELINE.json configs[0..4]; recipe in DESIGN.md "Input recipe").
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SEED_BASE = 200609167  # arXiv number of the paper; seed = SEED_BASE + config index

# BASELINE.json configs[0]: SPC/E-like 3-site model
Q_O = -0.8476
Q_H = 0.4238
SIGMA_O = 0.3166  # nm
EPS_O = 0.650  # kJ/mol
R_OH = 0.1  # nm
ANGLE_HOH = math.radians(109.47)
MOLECULES_PER_NM3 = 33.4


@dataclasses.dataclass
class Workload:
    """One synthetic system plus the run parameters its config names."""

    name: str
    x: np.ndarray  # float32 [N,3], wrapped into [0,L) atom by atom
    q: np.ndarray  # float32 [N]
    type: np.ndarray  # int32 [N]
    box: np.ndarray  # float32 [3]
    ntypes: int
    lj_c6c12: np.ndarray  # float32 [ntypes, ntypes, 2]   c6 = 4 eps sigma^6, c12 = 4 eps sigma^12
    excl_off: np.ndarray  # int32 [N+1]  CSR, symmetric, no self entries
    excl_idx: np.ndarray  # int32 [nexcl]
    mol_of_atom: np.ndarray  # int32 [N]
    unit_dir: np.ndarray  # float32 [nmol,3] fixed random unit vector per molecule (motion recipe)
    rc: float
    rlist_outer: float
    rlist_inner: float
    nstlist: int
    nparts: int
    coulomb: str = "ewald"  # "ewald" | "rf" | "none" (LJ only)
    ewald_rtol: float = 1e-5
    delta_per_step: float = 2.5e-4  # nm/step drift along unit_dir

    @property
    def natoms(self) -> int:
        return int(self.x.shape[0])

    def positions_at(self, t: int) -> np.ndarray:
        """Continuous (not re-wrapped) coordinates after t steps of the motion recipe:
        x_t = x_0 + t * delta * u_m, u_m fixed per molecule (rigid translation of each
        molecule, so intramolecular geometry is unchanged)."""
        d = (np.float32(t * self.delta_per_step) * self.unit_dir)[self.mol_of_atom]
        return (self.x + d).astype(np.float32)


def _water_site_offsets() -> np.ndarray:
    """O at origin, two H at R_OH with the H-O-H angle; float64 [3,3]."""
    h = ANGLE_HOH / 2.0
    return np.array(
        [
            [0.0, 0.0, 0.0],
            [R_OH * math.sin(h), 0.0, R_OH * math.cos(h)],
            [-R_OH * math.sin(h), 0.0, R_OH * math.cos(h)],
        ]
    )


def _random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """Uniform random rotation matrices from normalised 4-Gaussian quaternions; [n,3,3]."""
    qn = rng.normal(size=(n, 4))
    qn /= np.linalg.norm(qn, axis=1, keepdims=True)
    w, x, y, z = qn[:, 0], qn[:, 1], qn[:, 2], qn[:, 3]
    r = np.empty((n, 3, 3))
    r[:, 0, 0] = 1 - 2 * (y * y + z * z)
    r[:, 0, 1] = 2 * (x * y - z * w)
    r[:, 0, 2] = 2 * (x * z + y * w)
    r[:, 1, 0] = 2 * (x * y + z * w)
    r[:, 1, 1] = 1 - 2 * (x * x + z * z)
    r[:, 1, 2] = 2 * (y * z - x * w)
    r[:, 2, 0] = 2 * (x * z - y * w)
    r[:, 2, 1] = 2 * (y * z + x * w)
    r[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return r


def _place_sites(o_pos: np.ndarray, rot: np.ndarray) -> np.ndarray:
    """Atom positions [nmol,3,3] (O,H,H) for molecule centres o_pos and rotations rot."""
    sites = _water_site_offsets()
    return o_pos[:, None, :] + np.einsum("mij,aj->mai", rot, sites)


def _orient_without_clashes(
    rng: np.random.Generator, o_pos: np.ndarray, box: np.ndarray, dmin: float, max_iter: int = 40
) -> np.ndarray:
    """Draw orientations; redraw those of molecules involved in an intermolecular atom
    pair closer than dmin (periodic), until none is left or max_iter is reached."""
    from scipy.spatial import cKDTree

    nmol = o_pos.shape[0]
    rot = _random_rotations(rng, nmol)
    for _ in range(max_iter):
        atoms = _place_sites(o_pos, rot).reshape(-1, 3)
        wrapped = np.mod(atoms, box)
        wrapped = np.where(wrapped >= box, 0.0, wrapped)
        tree = cKDTree(wrapped, boxsize=box)
        pairs = tree.query_pairs(dmin, output_type="ndarray")
        if pairs.size == 0:
            break
        mi, mj = pairs[:, 0] // 3, pairs[:, 1] // 3
        inter = mi != mj
        if not inter.any():
            break
        flip = rng.random(int(inter.sum())) < 0.5
        bad = np.unique(np.where(flip, mi[inter], mj[inter]))
        rot[bad] = _random_rotations(rng, bad.size)
    return rot


def _rsa_centres(
    rng: np.random.Generator, n: int, lo: np.ndarray, hi: np.ndarray, box: np.ndarray, dmin: float
) -> np.ndarray:
    """Random sequential insertion of n points in [lo,hi) with periodic minimum distance dmin."""
    pts = np.empty((n, 3))
    k = 0
    while k < n:
        cand = lo + rng.random(3) * (hi - lo)
        if k:
            d = pts[:k] - cand
            d -= box * np.rint(d / box)
            if (np.einsum("ij,ij->i", d, d) < dmin * dmin).any():
                continue
        pts[k] = cand
        k += 1
    return pts


def _water_topology(nmol: int):
    n = 3 * nmol
    q = np.tile(np.array([Q_O, Q_H, Q_H], dtype=np.float32), nmol)
    typ = np.tile(np.array([0, 1, 1], dtype=np.int32), nmol)
    mol = np.repeat(np.arange(nmol, dtype=np.int32), 3)
    excl_off = (2 * np.arange(n + 1)).astype(np.int32)
    base = 3 * mol
    a = np.arange(n) - base
    e0 = base + (a + 1) % 3
    e1 = base + (a + 2) % 3
    excl_idx = np.sort(np.stack([e0, e1], axis=1), axis=1).reshape(-1).astype(np.int32)
    return q, typ, mol, excl_off, excl_idx


def lj_table(sigma: np.ndarray, eps: np.ndarray) -> np.ndarray:
    """Lorentz-Berthelot pair table (the combination rule lives in the
    generator, the library only sees c6/c12).  A type with eps == 0 has no LJ with anything."""
    s = 0.5 * (sigma[:, None] + sigma[None, :])
    e = np.sqrt(eps[:, None] * eps[None, :])
    tab = np.empty((len(sigma), len(sigma), 2))
    tab[:, :, 0] = 4.0 * e * s**6
    tab[:, :, 1] = 4.0 * e * s**12
    return tab.astype(np.float32)


def _finish(name, rng, o_pos, rot, box, **run) -> Workload:
    nmol = o_pos.shape[0]
    atoms = _place_sites(o_pos, rot).reshape(-1, 3)
    box32 = box.astype(np.float32)
    x = np.mod(atoms, box).astype(np.float32)
    x = np.where(x >= box32, np.float32(0.0), x).astype(np.float32)  # individually wrapped into [0,L)
    q, typ, mol, excl_off, excl_idx = _water_topology(nmol)
    u = rng.normal(size=(nmol, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    tab = lj_table(np.array([SIGMA_O, 0.0]), np.array([EPS_O, 0.0]))
    return Workload(
        name=name, x=x, q=q, type=typ, box=box32, ntypes=2, lj_c6c12=tab,
        excl_off=excl_off, excl_idx=excl_idx, mol_of_atom=mol,
        unit_dir=u.astype(np.float32), **run,
    )


def _lattice_water(name, seed, nside, nvac, box_len, **run) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    spacing = box_len / nside
    g = np.arange(nside)
    sites = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    if nvac:
        keep = np.ones(sites.shape[0], dtype=bool)
        keep[rng.choice(sites.shape[0], size=nvac, replace=False)] = False
        sites = sites[keep]
    o_pos = (sites + 0.5) * spacing + rng.uniform(-0.2, 0.2, size=sites.shape) * spacing
    box = np.full(3, box_len)
    rot = _orient_without_clashes(rng, o_pos, box, 0.13)
    return _finish(name, rng, o_pos, rot, box, **run)


def config0(rlist_outer: float = 0.93, rlist_inner: float = 0.91) -> Workload:
    """BASELINE.json configs[0]: 216 molecules, L = 1.862 nm, random insertion."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 0))
    box = np.full(3, 1.862)
    o_pos = _rsa_centres(rng, 216, np.zeros(3), box, box, 0.25)
    rot = _orient_without_clashes(rng, o_pos, box, 0.13)
    return _finish("cfg0_water648", rng, o_pos, rot, box, rc=0.9, rlist_outer=rlist_outer,
                   rlist_inner=rlist_inner, nstlist=100, nparts=1)


def config1() -> Workload:
    """configs[1]: 8000 molecules on a jittered 20^3 lattice, L = (8000/33.4)^(1/3)."""
    L = (8000 / MOLECULES_PER_NM3) ** (1.0 / 3.0)
    return _lattice_water("cfg1_water24k", SEED_BASE + 1, 20, 0, L, rc=1.0, rlist_outer=1.1,
                          rlist_inner=1.03, nstlist=100, nparts=2)


def config2(coulomb: str = "ewald") -> Workload:
    """configs[2]: 32000 molecules (32^3 lattice, 768 vacancies); Ewald rc 1.0 or RF rc 1.2."""
    L = (32000 / MOLECULES_PER_NM3) ** (1.0 / 3.0)
    if coulomb == "ewald":
        run = dict(rc=1.0, rlist_outer=1.1, rlist_inner=1.03, coulomb="ewald")
    else:
        run = dict(rc=1.2, rlist_outer=1.3, rlist_inner=1.23, coulomb="rf")
    return _lattice_water(f"cfg2_water96k_{coulomb}", SEED_BASE + 2, 32, 768, L, nstlist=100,
                          nparts=2, **run)


def config3() -> Workload:
    """configs[3]: 357000 molecules (71^3 lattice, 911 vacancies)."""
    L = (357000 / MOLECULES_PER_NM3) ** (1.0 / 3.0)
    return _lattice_water("cfg3_water1M", SEED_BASE + 3, 71, 911, L, rc=1.0, rlist_outer=1.2,
                          rlist_inner=1.05, nstlist=100, nparts=4)


def config4() -> Workload:
    """configs[4]: 4:1:1 box, dense slab next to 1 % vapour, 10 % re-typed/re-charged atoms."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 4))
    box = np.array([36.2, 9.05, 9.05])
    nx, ny = 58, 29
    sp = box[1] / ny
    gx, gy = np.arange(nx), np.arange(ny)
    sites = np.stack(np.meshgrid(gx, gy, gy, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    slab = (sites + 0.5) * sp + rng.uniform(-0.2, 0.2, size=sites.shape) * sp
    nvap = int(round(0.01 * MOLECULES_PER_NM3 * 18.1 * box[1] * box[2]))
    lo = np.array([18.1 + 0.3, 0.0, 0.0])
    hi = np.array([36.2 - 0.3, box[1], box[2]])
    vap = _rsa_centres(rng, nvap, lo, hi, box, 0.35)
    o_pos = np.concatenate([slab, vap])
    rot = _orient_without_clashes(rng, o_pos, box, 0.13)
    w = _finish("cfg4_slab150k", rng, o_pos, rot, box, rc=1.0, rlist_outer=1.1, rlist_inner=1.03,
                nstlist=100, nparts=2)
    n = w.natoms
    pick = rng.choice(n, size=n // 10, replace=False)
    sig = np.concatenate([[SIGMA_O, 0.0], rng.uniform(0.25, 0.40, size=4)])
    eps = np.concatenate([[EPS_O, 0.0], rng.uniform(0.2, 1.0, size=4)])
    w.type = w.type.copy()
    w.q = w.q.copy()
    w.type[pick] = rng.integers(2, 6, size=pick.size).astype(np.int32)
    qn = rng.uniform(-0.5, 0.5, size=pick.size)
    w.q[pick] = qn.astype(np.float32)
    excess = float(w.q.astype(np.float64).sum())
    w.q[pick] = (w.q[pick].astype(np.float64) - excess / pick.size).astype(np.float32)
    w.ntypes = 6
    w.lj_c6c12 = lj_table(sig, eps)
    return w


def small_water(nmol: int, box_len: float, seed: int, rc: float, rlist_outer: float,
                rlist_inner: float, box_scale=(1.0, 1.0, 1.0), coulomb: str = "ewald") -> Workload:
    """Small random-insertion water box for unit tests (same recipe as config 0)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    box = box_len * np.asarray(box_scale, dtype=np.float64)
    o_pos = _rsa_centres(rng, nmol, np.zeros(3), box, box, 0.25)
    rot = _orient_without_clashes(rng, o_pos, box, 0.13)
    return _finish(f"water{3 * nmol}", rng, o_pos, rot, box, rc=rc, rlist_outer=rlist_outer,
                   rlist_inner=rlist_inner, nstlist=100, nparts=1, coulomb=coulomb)


# Second workload of the paper (Fig. 6): a Lennard-Jones fluid whose cut-off is
# swept to vary the number of pairs per atom ("157k-atom argon-like system"; the figure's values
# are an image, only the recipe is taken).  Stand-in: one LJ type, no charges, no exclusions,
# jittered simple-cubic lattice at 26 atoms/nm^3, sigma = 0.3345 nm, eps = 0.996 kJ/mol.
LJ_SIGMA, LJ_EPS, LJ_RHO = 0.3345, 0.996, 26.0


def lj_fluid(nside: int = 54, rc: float = 1.0, buffer_outer: float = 0.1, buffer_inner: float = 0.03,
             seed: int = SEED_BASE + 10) -> Workload:
    """nside^3 single-type LJ atoms (54^3 = 157 464), each its own 'molecule' in the motion recipe."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = nside**3
    box_len = (n / LJ_RHO) ** (1.0 / 3.0)
    spacing = box_len / nside
    g = np.arange(nside)
    sites = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    pos = (sites + 0.5) * spacing + rng.uniform(-0.15, 0.15, size=sites.shape) * spacing
    box = np.full(3, box_len)
    x = np.mod(pos, box).astype(np.float32)
    x = np.where(x >= box.astype(np.float32), np.float32(0.0), x).astype(np.float32)
    u = rng.normal(size=(n, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    return Workload(
        name=f"lj_fluid{n}_rc{rc:g}", x=x, q=np.zeros(n, np.float32), type=np.zeros(n, np.int32), box=box.astype(np.float32),
        ntypes=1, lj_c6c12=lj_table(np.array([LJ_SIGMA]), np.array([LJ_EPS])),
        excl_off=np.zeros(n + 1, np.int32), excl_idx=np.zeros(0, np.int32), mol_of_atom=np.arange(n, dtype=np.int32),
        unit_dir=u.astype(np.float32), rc=rc, rlist_outer=rc + buffer_outer, rlist_inner=rc + buffer_inner,
        nstlist=100, nparts=2, coulomb="none",
    )


def water_box(nside: int) -> Workload:
    """Size sweep of the water workload (Fig. 7: 3k to 3M atoms): nside^3 molecules on
    the jittered lattice of configs 1-3 at 33.4 molecules/nm^3, run parameters of config 1."""
    L = (nside**3 / MOLECULES_PER_NM3) ** (1.0 / 3.0)
    return _lattice_water(f"water{3 * nside**3}", SEED_BASE + 20 + nside, nside, 0, L, rc=1.0, rlist_outer=1.1,
                          rlist_inner=1.03, nstlist=100, nparts=2)


def local_first(w: Workload, is_local_atom):
    """Stand-in for the atom order of a decomposed run (local atoms and the non-local atoms received
    in the halo exchange): returns (the workload with the molecules whose FIRST atom satisfies is_local_atom(x) moved to
    the front, nlocal).  Pure index bookkeeping: molecules stay contiguous and whole, exclusions are remapped.
    is_local_atom maps the [N,3] coordinates to a boolean per atom."""
    n = w.natoms
    mol = w.mol_of_atom
    nmol = int(mol.max()) + 1
    first = np.full(nmol, n, dtype=np.int64)
    np.minimum.at(first, mol, np.arange(n))
    flag_mol = np.asarray(is_local_atom(w.x))[first]
    key = np.where(flag_mol[mol], 0, 1)
    perm = np.argsort(key, kind="stable")          # new position k holds old atom perm[k]
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n)
    nlocal = int((key == 0).sum())
    counts = (w.excl_off[1:] - w.excl_off[:-1])[perm]
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    idx = np.empty(int(off[-1]), dtype=np.int32)
    for k in range(n):                               # rows are short (intramolecular): a plain loop
        o = perm[k]
        idx[off[k]:off[k + 1]] = np.sort(inv[w.excl_idx[w.excl_off[o]:w.excl_off[o + 1]]])
    mol_old = mol[perm]
    _, first_pos, mol_new = np.unique(mol_old, return_index=True, return_inverse=True)
    order = np.argsort(first_pos, kind="stable")    # new molecule ids in order of first appearance
    rank = np.empty_like(order)
    rank[order] = np.arange(order.size)
    mol_new = rank[mol_new].astype(np.int32)
    old_of_new_mol = np.unique(mol_old)[order]
    w2 = dataclasses.replace(
        w, name=w.name + "_localfirst", x=np.ascontiguousarray(w.x[perm]), q=np.ascontiguousarray(w.q[perm]),
        type=np.ascontiguousarray(w.type[perm]), excl_off=off, excl_idx=idx, mol_of_atom=mol_new,
        unit_dir=np.ascontiguousarray(w.unit_dir[old_of_new_mol]))
    return w2, nlocal


def by_index(k: int, **kw) -> Workload:
    return [config0, config1, config2, config3, config4][k](**kw)
